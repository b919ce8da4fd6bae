"""ctypes front end of the CPU oracle (oracle/tpc_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, ``__graft_entry__.smoke()`` and bench.py's
``cpu_baseline`` / ``--impl reference`` legs.  The product package never imports this module and
this module never imports the product package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpc_oracle.cpp")
_LIB = os.path.join(_HERE, "libtpc_oracle.so")

# Defaults of every free parameter (G4, G6, G7, G12, G15-G21, G23, G26; the
# paper fixes only min_clusters = 30 (L116) and alpha = 6 (L94)).
DEFAULT_CUTS = dict(
    bin_y=1.0, bin_z=4.0, grid_pad=1e-3,
    nf_wy_slope=1.0, nf_wy_const=0.5, nf_wz_slope=0.5, nf_wz_const=0.5,
    nf_max_dev2=0.25,
    min_chain_clusters=3,
    err_y2=0.0144, err_z2=0.0144,
    q_sinphi=1e-6, q_dzds=1e-6,
    c0_sinphi=0.25, c0_dzds=1.0, c0_kappa=2.5e-3,
    max_sinphi=0.95,
    chi2_cut=10.0,
    max_row_gap=4,
    edge_margin=1.0,
    min_clusters=30,
    min_pt=0.05,
    select_mode=0,
    alpha=6.0,
    global_tracking=0, gt_max_rows=30, gt_edge=3.0,       # NEXT-2 (G33): off by default
    select_rounds=1,                                      # NEXT-4 (G26b): 2 = second selection round
    merge_tracks=0, merge_max_gap=10, merge_chi2_cut=30.0,    # NEXT-3 (G37-G40): off by default
    max_passes=2,                                         # NEXT-4 (G22d): > 2 = further passes until nothing is gained
)

MODE_GRID, MODE_ROWSCAN, MODE_TRIPLET = 0, 1, 2


class _Geometry(C.Structure):
    _fields_ = [("n_sectors", C.c_uint32), ("n_rows", C.c_uint32), ("row_x", C.POINTER(C.c_float)),
                ("tan_half_angle", C.c_float), ("z_max", C.c_float), ("bz_tesla", C.c_float)]


class _Cuts(C.Structure):
    _fields_ = [("bin_y", C.c_float), ("bin_z", C.c_float), ("grid_pad", C.c_float),
                ("nf_wy_slope", C.c_float), ("nf_wy_const", C.c_float), ("nf_wz_slope", C.c_float),
                ("nf_wz_const", C.c_float), ("nf_max_dev2", C.c_float),
                ("min_chain_clusters", C.c_uint32),
                ("err_y2", C.c_float), ("err_z2", C.c_float),
                ("q_sinphi", C.c_float), ("q_dzds", C.c_float),
                ("c0_sinphi", C.c_float), ("c0_dzds", C.c_float), ("c0_kappa", C.c_float),
                ("max_sinphi", C.c_float), ("chi2_cut", C.c_float),
                ("max_row_gap", C.c_uint32), ("edge_margin", C.c_float),
                ("min_clusters", C.c_uint32), ("min_pt", C.c_float),
                ("select_mode", C.c_uint32), ("alpha", C.c_float),
                ("global_tracking", C.c_uint32), ("gt_max_rows", C.c_uint32), ("gt_edge", C.c_float),
                ("select_rounds", C.c_uint32),
                ("merge_tracks", C.c_uint32), ("merge_max_gap", C.c_uint32), ("merge_chi2_cut", C.c_float),
                ("max_passes", C.c_uint32)]


TRACK_DTYPE = np.dtype([("sector", "<u4"), ("first_row", "<u4"), ("last_row", "<u4"), ("n_clusters", "<u4"),
                        ("first_cluster", "<u4"), ("seed_cluster", "<u4"),
                        ("x_ref", "<f4"), ("y", "<f4"), ("z", "<f4"), ("sinphi", "<f4"), ("dzds", "<f4"),
                        ("qpt", "<f4"), ("cov", "<f4", (15,)), ("chi2", "<f4")])

GLOBAL_DTYPE = np.dtype([("track", "<u4"), ("sector", "<u4"), ("end", "<u4"), ("n_clusters", "<u4"),
                         ("first_cluster", "<u4"), ("row", "<u4"),
                         ("x_ref", "<f4"), ("y", "<f4"), ("z", "<f4"), ("sinphi", "<f4"), ("dzds", "<f4"),
                         ("qpt", "<f4"), ("cov", "<f4", (15,)), ("chi2", "<f4")])

MERGE_DTYPE = np.dtype([("rank", "<u4"), ("next", "<i4"), ("prev", "<i4"), ("ok", "<u4"),
                        ("row_in", "<u4"), ("row_out", "<u4"), ("chi2", "<f4"),
                        ("match_chi2", "<f4"), ("in_par", "<f4", (5,)), ("in_cov", "<f4", (15,)),
                        ("out_par", "<f4", (5,)), ("out_cov", "<f4", (15,)),
                        ("chain_n_seg", "<u4"), ("chain_n_clusters", "<u4"), ("chain_chi2", "<f4"),
                        ("chain_par", "<f4", (5,)), ("chain_cov", "<f4", (15,))])
MERGE_CAND_DTYPE = np.dtype([("a", "<u4"), ("b", "<u4"), ("chi2", "<f4")])

_ARRAYS = {  # name -> (id, dtype)
    "bin_of": (0, np.uint32), "bin_row_offset": (1, np.uint32), "bin_count": (2, np.uint32),
    "bin_start": (3, np.uint32), "up_raw": (4, np.int32), "dn_raw": (5, np.int32), "up": (6, np.int32),
    "dn": (7, np.int32), "owner": (8, np.uint32), "start_cluster": (9, np.uint32), "chain_len": (10, np.uint32),
    "first_row": (11, np.uint32), "last_row": (12, np.uint32), "nhits": (13, np.uint32), "kept": (14, np.uint32),
    "accepted": (15, np.uint8), "params": (16, np.float32), "cov": (17, np.float32), "chi2": (18, np.float32),
    "hits": (19, np.int32), "tracks": (20, TRACK_DTYPE), "track_cluster_ids": (21, np.uint32),
    "counters": (22, np.uint64), "tracklet_sector": (23, np.uint32),
    "tab_ymax": (24, np.float32), "tab_ny": (25, np.uint32), "tab_ratio_up": (26, np.float32),
    "tab_ratio_dn": (27, np.float32), "tab_w_up": (28, np.float32), "tab_w_dn": (29, np.float32),
    "tab_wy_up": (30, np.float32), "tab_wy_dn": (31, np.float32), "tab_wz_up": (32, np.float32),
    "tab_wz_dn": (33, np.float32),
    "global_ext": (34, GLOBAL_DTYPE), "global_cluster_ids": (35, np.uint32),
    "merge": (36, MERGE_DTYPE), "merge_cand": (37, MERGE_CAND_DTYPE),
    "ref_row": (38, np.uint32), "n_passes": (39, np.uint32), "near": (40, np.uint32),
}
COUNTER_NAMES = ("nf_window_tests", "nf_pair_evals", "links_raw", "links_evolved", "starts", "kf_row_steps",
                 "kf_candidates", "kf_updates", "claimed_hits", "tracks", "track_clusters")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (fp32, one rounding per operation: no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-pthread",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.orc_create.restype = C.c_void_p
        lib.orc_create.argtypes = [C.POINTER(_Geometry), C.POINTER(_Cuts)]
        lib.orc_destroy.argtypes = [C.c_void_p]
        lib.orc_run.restype = C.c_int
        lib.orc_run.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_int, C.c_int, C.c_int]
        lib.orc_array.restype = C.c_void_p
        lib.orc_array.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_uint64)]
        lib.orc_nz.restype = C.c_uint32
        lib.orc_nz.argtypes = [C.c_void_p]
        lib.orc_transport.restype = C.c_int
        lib.orc_transport.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_void_p]
        lib.orc_update.restype = C.c_int
        lib.orc_update.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.POINTER(C.c_float)]
        lib.orc_third_pass_gain.restype = C.c_uint64
        lib.orc_third_pass_gain.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        lib.orc_rotate.restype = C.c_int
        lib.orc_rotate.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_void_p, C.POINTER(C.c_float)]
        _lib = lib
    return _lib


@dataclass
class OracleResult:
    arrays: dict

    def __getattr__(self, name):
        try:
            return self.arrays[name]
        except KeyError as e:
            raise AttributeError(name) from e


class Oracle:
    """One tracker instance: geometry + cuts; ``run`` tracks one event."""

    def __init__(self, n_sectors: int, row_x, tan_half_angle: float, z_max: float, bz_tesla: float, **cuts):
        lib = _load()
        self._row_x = np.ascontiguousarray(row_x, dtype=np.float32)
        g = _Geometry(n_sectors, self._row_x.size, self._row_x.ctypes.data_as(C.POINTER(C.c_float)),
                      tan_half_angle, z_max, bz_tesla)
        full = dict(DEFAULT_CUTS)
        unknown = set(cuts) - set(full)
        if unknown:
            raise KeyError(f"unknown cuts: {sorted(unknown)}")
        full.update(cuts)
        self.cuts = full
        c = _Cuts(**full)
        self.n_sectors, self.n_rows = n_sectors, int(self._row_x.size)
        self._h = C.c_void_p(lib.orc_create(C.byref(g), C.byref(c)))

    @classmethod
    def for_geometry(cls, geo, **cuts):
        return cls(geo.n_sectors, geo.row_x, geo.tan_half_angle, geo.z_max, geo.bz_tesla, **cuts)

    def __del__(self):
        if getattr(self, "_h", None):
            _load().orc_destroy(self._h)
            self._h = None

    def array(self, name: str) -> np.ndarray:
        idx, dt = _ARRAYS[name]
        cnt = C.c_uint64(0)
        p = _load().orc_array(self._h, idx, C.byref(cnt))
        n = int(cnt.value)
        dt = np.dtype(dt)
        if n == 0 or not p:
            return np.zeros(0, dt)
        buf = (C.c_char * (n * dt.itemsize)).from_address(p)
        return np.frombuffer(buf, dtype=dt, count=n).copy()

    @property
    def nz(self) -> int:
        return int(_load().orc_nz(self._h))

    def run(self, xyz, row_start, mode: int = MODE_GRID, stop_after: int = 0, n_threads: int = 1,
            fetch: bool = True) -> OracleResult | None:
        xyz = np.ascontiguousarray(xyz, dtype=np.float32)
        row_start = np.ascontiguousarray(row_start, dtype=np.uint32)
        assert row_start.size == self.n_sectors * self.n_rows + 1
        rc = _load().orc_run(self._h, xyz.ctypes.data, row_start.ctypes.data, xyz.shape[0], mode, stop_after, n_threads)
        if rc != 0:
            raise ValueError("oracle: bad row_start")
        if not fetch:
            return None
        skip = {"tab_ymax", "tab_ny", "tab_ratio_up", "tab_ratio_dn", "tab_w_up", "tab_w_dn", "tab_wy_up",
                "tab_wy_dn", "tab_wz_up", "tab_wz_dn"}
        arr = {k: self.array(k) for k in _ARRAYS if k not in skip}
        R = self.n_rows
        arr["params"] = arr["params"].reshape(-1, 5)
        arr["cov"] = arr["cov"].reshape(-1, 15)
        arr["hits"] = arr["hits"].reshape(-1, R)
        arr["near"] = arr["near"].reshape(-1, 2)          # G29 audit: (tracklet, row) of near-threshold pickup decisions
        arr["counters"] = dict(zip(COUNTER_NAMES, (int(v) for v in arr["counters"])))
        return OracleResult(arr)

    def third_pass_gain(self, xyz, n_tracklets: int) -> np.ndarray:
        """Diagnostic (NEXT-4, G22d): clusters a third construction pass would add to every tracklet of the last
        run, found by scanning whole rows (nothing is modified); bit 31 = the simulated pass ended on a failure."""
        xyz = np.ascontiguousarray(xyz, dtype=np.float32)
        out = np.zeros(n_tracklets, np.uint32)
        _load().orc_third_pass_gain(self._h, xyz.ctypes.data, out.ctypes.data)
        return out

    # single-step entry points for the closed-form pins
    def transport(self, state20, dx: float, nrows: float = 1.0):
        a = np.ascontiguousarray(state20, dtype=np.float32)
        b = np.zeros(20, np.float32)
        ok = _load().orc_transport(self._h, a.ctypes.data, dx, nrows, b.ctypes.data)
        return b if ok else None

    def update(self, state20, ym: float, zm: float):
        a = np.ascontiguousarray(state20, dtype=np.float32)
        b = np.zeros(20, np.float32)
        chi2 = C.c_float(0)
        ok = _load().orc_update(self._h, a.ctypes.data, ym, zm, b.ctypes.data, C.byref(chi2))
        return (b, float(chi2.value)) if ok else None

    def rotate(self, state20, x0: float, sg: float):
        """G34: the state at x0 seen from the neighbouring sector on the side sg = +-1 -> (state20, x')."""
        a = np.ascontiguousarray(state20, dtype=np.float32)
        b = np.zeros(20, np.float32)
        xr = C.c_float(0)
        ok = _load().orc_rotate(self._h, a.ctypes.data, x0, sg, b.ctypes.data, C.byref(xr))
        return (b, float(xr.value)) if ok else None
