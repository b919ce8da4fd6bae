"""The C-ABI library loads and exports every symbol include/tpcst.h declares (no GPU needed)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "tpcst.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tpcst_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for f in ("tpcst_create", "tpcst_track_event", "tpcst_destroy"):
        assert f in names


def test_library_exports_every_declared_symbol():
    import paper_1712_09407_b200 as t
    L = t.lib()
    for f in _declared():
        assert hasattr(L, f), f
    assert sorted(t.EXPORTS) == _declared()


def test_default_cuts_and_workspace_size_without_a_gpu():
    import paper_1712_09407_b200 as t
    from tpcsynth import Geometry
    c = t.tpcst_default_cuts()
    assert (c.min_clusters, c.alpha, c.chi2_cut) == (30, 6.0, 10.0)     # PAPER.md L116, L94; G20
    b1 = t.tpcst_workspace_bytes(Geometry(), c, 1_000_000, 100_000)
    b2 = t.tpcst_workspace_bytes(Geometry(), c, 4_000_000, 400_000)
    assert 0 < b1 < b2 < 4 << 30
    c.max_passes = 0                                  # the newest field: 0 means the default, 2 (include/tpcst.h)
    assert t.tpcst_workspace_bytes(Geometry(), c, 1_000_000, 100_000) == b1
    c.max_passes = 1
    assert t.tpcst_workspace_bytes(Geometry(), c, 1_000_000, 100_000) == 0
    c.max_passes = 2
    c.bin_y = -1.0
    assert t.tpcst_workspace_bytes(Geometry(), c, 1_000_000, 100_000) == 0
    assert t.lib().tpcst_error_string(t.TPCST_ERR_CAPACITY).decode().startswith("workspace capacity")
    assert ctypes.sizeof(t.tpcst_cuts) == 32 * 4 and t.tpcst_default_cuts().max_passes == 2


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1712_09407_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "tpc_oracle" not in txt, f
