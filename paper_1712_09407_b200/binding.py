"""ctypes binding of include/tpcst.h — argument marshalling only.

Every step of the sector tracker runs in the CUDA kernels of ``csrc/``; this
module only converts numpy / torch buffers to the plain pointers of the C ABI and wraps the results
as numpy views.  PyTorch is used for device memory (the workspace tensor) and CUDA streams, nothing
else.  There is no CPU fallback: if ``libtpcst.so`` cannot be loaded the import of the library
raises, and the oracle under ``oracle/`` is never imported from here.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

from . import build as _build

TPCST_OK, TPCST_ERR_ARG, TPCST_ERR_RANGE, TPCST_ERR_CAPACITY, TPCST_ERR_CUDA, TPCST_ERR_STATE = 0, -1, -2, -3, -4, -5
TPCST_ERR_STATIC_LIMIT = -6
TPCST_STATIC_MAX_CLUSTERS = 1 << 20
TPCST_HOST_PINNED, TPCST_HOST_PAGEABLE, TPCST_DEVICE = 0, 1, 2
TPCST_N_SLOTS = 4
(TPCST_DBG_BIN_OF, TPCST_DBG_BIN_START, TPCST_DBG_LINKS_RAW, TPCST_DBG_LINKS, TPCST_DBG_STARTS,
 TPCST_DBG_TRACKLETS, TPCST_DBG_ROW_HITS, TPCST_DBG_OWNERS, TPCST_DBG_COUNTERS, TPCST_DBG_KERNEL_MS,
 TPCST_DBG_WORK) = range(11)
WORK_NAMES = ("nf_window_tests", "nf_pair_evals", "kf_row_steps", "kf_searches", "kf_candidates", "kf_updates",
              "claimed_hits")

EXPORTS = ("tpcst_default_cuts", "tpcst_workspace_bytes", "tpcst_create", "tpcst_track_event",
           "tpcst_submit_event", "tpcst_wait_event", "tpcst_debug_fetch", "tpcst_kernels_per_event",
           "tpcst_kernel_name", "tpcst_set_profiling", "tpcst_set_graphs", "tpcst_selftest_math", "tpcst_error_string", "tpcst_destroy",
           "tpcst_select_owners_static", "tpcst_selftest_random_access")


class tpcst_geometry(C.Structure):
    _fields_ = [("n_sectors", C.c_uint32), ("n_rows", C.c_uint32), ("row_x", C.POINTER(C.c_float)),
                ("tan_half_angle", C.c_float), ("z_max", C.c_float), ("bz_tesla", C.c_float)]


class tpcst_cuts(C.Structure):
    _fields_ = [("bin_y", C.c_float), ("bin_z", C.c_float), ("grid_pad", C.c_float),
                ("nf_wy_slope", C.c_float), ("nf_wy_const", C.c_float), ("nf_wz_slope", C.c_float),
                ("nf_wz_const", C.c_float), ("nf_max_dev2", C.c_float),
                ("min_chain_clusters", C.c_uint32),
                ("err_y2", C.c_float), ("err_z2", C.c_float), ("q_sinphi", C.c_float), ("q_dzds", C.c_float),
                ("c0_sinphi", C.c_float), ("c0_dzds", C.c_float), ("c0_kappa", C.c_float),
                ("max_sinphi", C.c_float), ("chi2_cut", C.c_float), ("max_row_gap", C.c_uint32),
                ("edge_margin", C.c_float), ("min_clusters", C.c_uint32), ("min_pt", C.c_float),
                ("select_mode", C.c_uint32), ("alpha", C.c_float),
                ("global_tracking", C.c_uint32), ("gt_max_rows", C.c_uint32), ("gt_edge", C.c_float),
                ("select_rounds", C.c_uint32),
                ("merge_tracks", C.c_uint32), ("merge_max_gap", C.c_uint32), ("merge_chi2_cut", C.c_float),
                ("max_passes", C.c_uint32)]


class tpcst_clusters(C.Structure):
    _fields_ = [("xyz", C.c_void_p), ("row_start", C.c_void_p), ("n_clusters", C.c_uint32), ("location", C.c_int32)]


class tpcst_tracks(C.Structure):
    _fields_ = [("n_tracks", C.c_uint32), ("tracks", C.c_void_p), ("n_cluster_ids", C.c_uint32),
                ("cluster_ids", C.c_void_p), ("n_tracklets", C.c_uint32), ("gpu_ms", C.c_float),
                ("n_global", C.c_uint32), ("global_ext", C.c_void_p), ("n_global_cluster_ids", C.c_uint32),
                ("global_cluster_ids", C.c_void_p), ("n_merge", C.c_uint32), ("merge", C.c_void_p)]


# struct tpcst_track of include/tpcst.h (112 bytes)
TRACK_DTYPE = np.dtype([("sector", "<u4"), ("first_row", "<u4"), ("last_row", "<u4"), ("n_clusters", "<u4"),
                        ("first_cluster", "<u4"), ("seed_cluster", "<u4"), ("x_ref", "<f4"), ("y", "<f4"),
                        ("z", "<f4"), ("sinphi", "<f4"), ("dzds", "<f4"), ("qpt", "<f4"), ("cov", "<f4", (15,)),
                        ("chi2", "<f4")])
assert TRACK_DTYPE.itemsize == 112
# struct tpcst_global_ext of include/tpcst.h (112 bytes)
GLOBAL_DTYPE = np.dtype([("track", "<u4"), ("sector", "<u4"), ("end", "<u4"), ("n_clusters", "<u4"),
                         ("first_cluster", "<u4"), ("row", "<u4"), ("x_ref", "<f4"), ("y", "<f4"), ("z", "<f4"),
                         ("sinphi", "<f4"), ("dzds", "<f4"), ("qpt", "<f4"), ("cov", "<f4", (15,)), ("chi2", "<f4")])
assert GLOBAL_DTYPE.itemsize == 112
# struct tpcst_merge_seg of include/tpcst.h (284 bytes)
MERGE_DTYPE = np.dtype([("rank", "<u4"), ("next", "<i4"), ("prev", "<i4"), ("ok", "<u4"), ("row_in", "<u4"),
                        ("row_out", "<u4"), ("chi2", "<f4"), ("match_chi2", "<f4"), ("in_par", "<f4", (5,)),
                        ("in_cov", "<f4", (15,)), ("out_par", "<f4", (5,)), ("out_cov", "<f4", (15,)),
                        ("chain_n_seg", "<u4"), ("chain_n_clusters", "<u4"), ("chain_chi2", "<f4"),
                        ("chain_par", "<f4", (5,)), ("chain_cov", "<f4", (15,))])
assert MERGE_DTYPE.itemsize == 284

_lib = None


def lib() -> C.CDLL:
    """Load libtpcst.so (building it with nvcc if it is missing or stale).  Raises if impossible."""
    global _lib
    if _lib is not None:
        return _lib
    try:
        path = _build.build()
    except Exception as e:  # no nvcc / compile error: keep an existing library only if it is current
        if not os.path.exists(_build.LIB) or _build.stale():
            raise RuntimeError(f"libtpcst.so is missing or stale and cannot be built: {e}") from e
        path = _build.LIB
    L = C.CDLL(path)
    vp, u32, sz = C.c_void_p, C.c_uint32, C.c_size_t
    L.tpcst_default_cuts.argtypes = [C.POINTER(tpcst_cuts)]
    L.tpcst_workspace_bytes.restype = sz
    L.tpcst_workspace_bytes.argtypes = [C.POINTER(tpcst_geometry), C.POINTER(tpcst_cuts), u32, u32]
    L.tpcst_create.argtypes = [C.POINTER(tpcst_geometry), C.POINTER(tpcst_cuts), u32, u32, vp, sz, vp, vp, C.POINTER(vp)]
    L.tpcst_track_event.argtypes = [vp, C.POINTER(tpcst_clusters), C.POINTER(tpcst_tracks)]
    L.tpcst_submit_event.argtypes = [vp, C.POINTER(tpcst_clusters), C.c_int]
    L.tpcst_wait_event.argtypes = [vp, C.c_int, C.POINTER(tpcst_tracks)]
    L.tpcst_debug_fetch.argtypes = [vp, C.c_int, C.c_int, vp, sz, C.POINTER(sz)]
    L.tpcst_kernels_per_event.argtypes = [vp]
    L.tpcst_kernel_name.restype = C.c_char_p
    L.tpcst_kernel_name.argtypes = [C.c_int]
    L.tpcst_set_profiling.argtypes = [vp, C.c_int]
    L.tpcst_set_graphs.argtypes = [vp, C.c_int]
    L.tpcst_selftest_math.argtypes = [vp, C.c_uint64, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.tpcst_selftest_random_access.argtypes = [vp, u32, C.c_uint64, C.c_int, C.POINTER(C.c_float), C.POINTER(C.c_float)]
    L.tpcst_select_owners_static.argtypes = [vp, u32, u32, u32, u32, vp, vp, vp]
    L.tpcst_error_string.restype = C.c_char_p
    L.tpcst_error_string.argtypes = [C.c_int]
    L.tpcst_destroy.argtypes = [vp]
    for f in EXPORTS:                       # fail loudly on a library that lacks part of the ABI
        getattr(L, f)
    _lib = L
    return L


class TpcstError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {lib().tpcst_error_string(status).decode()} (status {status})")


def _check(status: int, where: str) -> None:
    if status != TPCST_OK:
        raise TpcstError(status, where)


def tpcst_default_cuts() -> tpcst_cuts:
    c = tpcst_cuts()
    _check(lib().tpcst_default_cuts(C.byref(c)), "tpcst_default_cuts")
    return c


def _geometry(geo) -> tuple[tpcst_geometry, np.ndarray]:
    row_x = np.ascontiguousarray(geo.row_x, dtype=np.float32)
    g = tpcst_geometry(int(geo.n_sectors), int(row_x.size), row_x.ctypes.data_as(C.POINTER(C.c_float)),
                       float(geo.tan_half_angle), float(geo.z_max), float(geo.bz_tesla))
    return g, row_x


def tpcst_workspace_bytes(geo, cuts: tpcst_cuts, max_clusters: int, max_tracklets: int) -> int:
    g, _keep = _geometry(geo)
    return int(lib().tpcst_workspace_bytes(C.byref(g), C.byref(cuts), max_clusters, max_tracklets))


@dataclass
class TrackResult:
    tracks: np.ndarray        # TRACK_DTYPE [K]   (view of library-owned pinned memory unless copied)
    cluster_ids: np.ndarray   # uint32 [sum n_clusters]
    n_tracklets: int
    gpu_ms: float
    global_ext: np.ndarray = None          # GLOBAL_DTYPE [n_global] (global tracking; empty unless enabled)
    global_cluster_ids: np.ndarray = None  # uint32
    merge: np.ndarray = None               # MERGE_DTYPE [K] (track sort / refit / links; empty unless enabled)

    def cluster_list(self, i: int) -> np.ndarray:
        t = self.tracks[i]
        return self.cluster_ids[int(t["first_cluster"]): int(t["first_cluster"]) + int(t["n_clusters"])]


def _marshal(xyz, row_start):
    """(pointer, pointer, n_clusters, location, keep-alive) of numpy / torch cluster arrays."""
    import torch
    if isinstance(xyz, torch.Tensor):
        if not isinstance(row_start, torch.Tensor) or row_start.device != xyz.device:
            raise ValueError("xyz and row_start must live in the same place")
        if xyz.dtype != torch.float32 or row_start.dtype not in (torch.int32, torch.uint32):
            raise ValueError("xyz must be float32 and row_start (u)int32")
        if not xyz.is_contiguous() or not row_start.is_contiguous():
            raise ValueError("cluster arrays must be contiguous")
        if xyz.is_cuda:
            loc = TPCST_DEVICE
        else:
            loc = TPCST_HOST_PINNED if (xyz.is_pinned() and row_start.is_pinned()) else TPCST_HOST_PAGEABLE
        n = xyz.numel() // 3
        return xyz.data_ptr(), row_start.data_ptr(), n, loc, (xyz, row_start)
    xyz = np.ascontiguousarray(xyz, dtype=np.float32)
    row_start = np.ascontiguousarray(row_start, dtype=np.uint32)
    return xyz.ctypes.data, row_start.ctypes.data, xyz.size // 3, TPCST_HOST_PAGEABLE, (xyz, row_start)


def selftest_math(n_div_pairs: int = 1 << 28, device="cuda:0"):
    """tpcst_selftest_math on `device`'s current stream -> (comparisons made, bit-level disagreements)."""
    import torch
    with torch.cuda.device(torch.device(device)):
        n, bad = C.c_uint64(0), C.c_uint64(0)
        _check(lib().tpcst_selftest_math(torch.cuda.current_stream().cuda_stream, int(n_div_pairs), C.byref(n), C.byref(bad)),
               "tpcst_selftest_math")
    return int(n.value), int(bad.value)


def selftest_random_access(n_words: int, n_access: int, reps: int = 20, device="cuda:0"):
    """tpcst_selftest_random_access on `device`'s current stream -> (ms of n_access random gathers, ms of n_access random atomic maxima)
    over an array of n_words 32-bit words: the device's own rate for the pattern that bounds the selection kernels."""
    import torch
    with torch.cuda.device(torch.device(device)):
        g, r = C.c_float(0), C.c_float(0)
        _check(lib().tpcst_selftest_random_access(torch.cuda.current_stream().cuda_stream, int(n_words), int(n_access), int(reps),
                                       C.byref(g), C.byref(r)), "tpcst_selftest_random_access")
    return float(g.value), float(r.value)


def select_owners_static(row_hits, n_clusters: int, min_clusters: int = 30, owner=None, kept=None):
    """tpcst_select_owners_static on the current stream of `row_hits`' device -> (owner, kept), both CUDA tensors.

    The one call of the library that allocates nothing: its per-cluster claim keys sit in a fixed 4 MiB array inside
    libtpcst.so's device image instead of a cudaMalloc'ed workspace.  It exists for callers that must not allocate
    where they select: real-time loops (cudaMalloc synchronises the whole device), plug-ins of a framework that
    owns all device memory, processes with a frozen memory budget.  At most TPCST_STATIC_MAX_CLUSTERS (1 Mi)
    clusters, else TpcstError(TPCST_ERR_STATIC_LIMIT).  Calls on one device share the array: do not overlap them.

    row_hits: int32 CUDA tensor [n_tracklets, n_rows], cluster index per row or -1 (the TPCST_DBG_ROW_HITS layout).
    owner / kept: optional preallocated int32 CUDA tensors [n_clusters] / [n_tracklets] to write into (a caller
    that really cannot allocate passes them; if omitted this wrapper, not the library, allocates them with torch).
    owner[c] = index of the tracklet that keeps cluster c, -1 (0xffffffff) if none; kept[t] = hits tracklet t keeps.
    The call is asynchronous on the stream; PyTorch's stream ordering makes later torch reads see the result.
    """
    import torch
    if not (isinstance(row_hits, torch.Tensor) and row_hits.is_cuda and row_hits.dtype == torch.int32
            and row_hits.dim() == 2 and row_hits.is_contiguous()):
        raise ValueError("row_hits must be a contiguous int32 CUDA tensor [n_tracklets, n_rows]")
    T, R = int(row_hits.shape[0]), int(row_hits.shape[1])
    n_clusters = int(n_clusters)
    if owner is None:
        owner = torch.empty(n_clusters, dtype=torch.int32, device=row_hits.device)
    if kept is None:
        kept = torch.empty(T, dtype=torch.int32, device=row_hits.device)
    for name, buf, n in (("owner", owner, n_clusters), ("kept", kept, T)):
        if not (buf.is_cuda and buf.device == row_hits.device and buf.dtype == torch.int32 and buf.is_contiguous()
                and buf.numel() == n):
            raise ValueError(f"{name} must be a contiguous int32 CUDA tensor of {n} elements on {row_hits.device}")
    with torch.cuda.device(row_hits.device):
        st = torch.cuda.current_stream().cuda_stream
    _check(lib().tpcst_select_owners_static(row_hits.data_ptr() if T else None, T, R, n_clusters, int(min_clusters),
                                            owner.data_ptr() if n_clusters else None, kept.data_ptr() if T else None, st),
           "tpcst_select_owners_static")
    return owner, kept


class SectorTracker:
    """tpcst_create / tpcst_track_event / tpcst_destroy with torch-owned device memory and streams.

    geometry: any object with n_sectors, row_x, tan_half_angle, z_max, bz_tesla (e.g. tpcsynth.Geometry).
    cuts: keyword overrides of tpcst_default_cuts.
    """

    def __init__(self, geometry, max_clusters: int, max_tracklets: int, device="cuda:0", **cuts):
        import torch
        L = lib()
        if not torch.cuda.is_available():
            raise RuntimeError("the TPC sector tracker needs a CUDA device (no CPU fallback)")
        self.device = torch.device(device)
        self.cuts = tpcst_default_cuts()
        for k, v in cuts.items():
            if not hasattr(self.cuts, k):
                raise KeyError(f"unknown cut: {k}")
            setattr(self.cuts, k, v)
        self.n_sectors, self.n_rows = int(geometry.n_sectors), int(len(geometry.row_x))
        self.max_clusters, self.max_tracklets = int(max_clusters), int(max_tracklets)
        g, self._row_x = _geometry(geometry)
        nbytes = int(L.tpcst_workspace_bytes(C.byref(g), C.byref(self.cuts), self.max_clusters, self.max_tracklets))
        if nbytes == 0:
            raise TpcstError(TPCST_ERR_ARG, "tpcst_workspace_bytes")
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self.stream_compute = torch.cuda.Stream(device=self.device)
            self.stream_copy = torch.cuda.Stream(device=self.device)
        base = (self._ws.data_ptr() + 255) & ~255
        h = C.c_void_p()
        _check(L.tpcst_create(C.byref(g), C.byref(self.cuts), self.max_clusters, self.max_tracklets, base, nbytes,
                              self.stream_compute.cuda_stream, self.stream_copy.cuda_stream, C.byref(h)),
               "tpcst_create")
        self._h = h
        self._keep = [None] * TPCST_N_SLOTS
        self.kernels_per_event = int(L.tpcst_kernels_per_event(self._h))
        self.kernel_names = [L.tpcst_kernel_name(i).decode() for i in range(self.kernels_per_event)]

    # -- lifetime ------------------------------------------------------------------------------
    def close(self) -> None:
        if getattr(self, "_h", None):
            lib().tpcst_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- the calls of the C ABI ----------------------------------------------------------------
    def _clusters(self, xyz, row_start):
        px, pr, n, loc, keep = _marshal(xyz, row_start)
        nrs = keep[1].size if isinstance(keep[1], np.ndarray) else keep[1].numel()
        if nrs != self.n_sectors * self.n_rows + 1:
            raise ValueError("row_start must have n_sectors * n_rows + 1 entries")
        return tpcst_clusters(px, pr, n, loc), keep

    @staticmethod
    def _result(out: tpcst_tracks, copy: bool) -> TrackResult:
        K, M = int(out.n_tracks), int(out.n_cluster_ids)
        if K:
            buf = (C.c_char * (K * TRACK_DTYPE.itemsize)).from_address(out.tracks)
            tracks = np.frombuffer(buf, dtype=TRACK_DTYPE, count=K)
        else:
            tracks = np.zeros(0, TRACK_DTYPE)
        if M:
            buf = (C.c_char * (M * 4)).from_address(out.cluster_ids)
            ids = np.frombuffer(buf, dtype=np.uint32, count=M)
        else:
            ids = np.zeros(0, np.uint32)
        if copy:
            tracks, ids = tracks.copy(), ids.copy()
        G, GM = int(out.n_global), int(out.n_global_cluster_ids)
        if G:
            buf = (C.c_char * (G * GLOBAL_DTYPE.itemsize)).from_address(out.global_ext)
            gext = np.frombuffer(buf, dtype=GLOBAL_DTYPE, count=G)
            buf = (C.c_char * (GM * 4)).from_address(out.global_cluster_ids)
            gids = np.frombuffer(buf, dtype=np.uint32, count=GM)
        else:
            gext, gids = np.zeros(0, GLOBAL_DTYPE), np.zeros(0, np.uint32)
        if int(out.n_merge):
            buf = (C.c_char * (int(out.n_merge) * MERGE_DTYPE.itemsize)).from_address(out.merge)
            merge = np.frombuffer(buf, dtype=MERGE_DTYPE, count=int(out.n_merge))
        else:
            merge = np.zeros(0, MERGE_DTYPE)
        if copy:                                         # else: views of the slot's pinned buffers, valid until its next submit
            gext, gids, merge = gext.copy(), gids.copy(), merge.copy()
        return TrackResult(tracks, ids, int(out.n_tracklets), float(out.gpu_ms), gext, gids, merge)

    def track_event(self, xyz, row_start, copy: bool = True) -> TrackResult:
        cl, keep = self._clusters(xyz, row_start)
        out = tpcst_tracks()
        _check(lib().tpcst_track_event(self._h, C.byref(cl), C.byref(out)), "tpcst_track_event")
        return self._result(out, copy)

    def submit_event(self, xyz, row_start, slot: int) -> None:
        cl, keep = self._clusters(xyz, row_start)
        _check(lib().tpcst_submit_event(self._h, C.byref(cl), slot), "tpcst_submit_event")
        self._keep[slot] = keep

    def wait_event(self, slot: int, copy: bool = True) -> TrackResult:
        out = tpcst_tracks()
        st = lib().tpcst_wait_event(self._h, slot, C.byref(out))
        self._keep[slot] = None
        _check(st, "tpcst_wait_event")
        return self._result(out, copy)

    def set_profiling(self, level) -> None:
        """0 off, 1 per-kernel CUDA events, 2 events + work counters (include/tpcst.h)."""
        _check(lib().tpcst_set_profiling(self._h, int(level)), "tpcst_set_profiling")

    def set_graphs(self, on: bool) -> None:
        """Replay of the launch set as a CUDA graph (include/tpcst.h), on by default."""
        _check(lib().tpcst_set_graphs(self._h, 1 if on else 0), "tpcst_set_graphs")

    def kernel_ms(self, slot: int = 0) -> np.ndarray:
        return self.debug_fetch(TPCST_DBG_KERNEL_MS, slot)

    def work_counters(self, slot: int = 0) -> dict:
        return dict(zip(WORK_NAMES, (int(v) for v in self.debug_fetch(TPCST_DBG_WORK, slot))))

    _DBG_DTYPE = {TPCST_DBG_BIN_OF: np.uint32, TPCST_DBG_BIN_START: np.uint32, TPCST_DBG_LINKS_RAW: np.int32,
                  TPCST_DBG_LINKS: np.int32, TPCST_DBG_STARTS: np.uint32, TPCST_DBG_TRACKLETS: TRACK_DTYPE,
                  TPCST_DBG_ROW_HITS: np.int32, TPCST_DBG_OWNERS: np.uint32, TPCST_DBG_COUNTERS: np.uint32,
                  TPCST_DBG_KERNEL_MS: np.float32, TPCST_DBG_WORK: np.uint64}

    def debug_fetch(self, what: int, slot: int = 0) -> np.ndarray:
        L = lib()
        need = C.c_size_t(0)
        st = L.tpcst_debug_fetch(self._h, slot, what, None, 0, C.byref(need))
        if st not in (TPCST_OK, TPCST_ERR_ARG) or (st == TPCST_ERR_ARG and need.value == 0):
            _check(st, "tpcst_debug_fetch")
        dt = np.dtype(self._DBG_DTYPE[what])
        buf = np.zeros(max(1, (need.value + dt.itemsize - 1) // dt.itemsize), dt)
        if need.value:
            _check(L.tpcst_debug_fetch(self._h, slot, what, buf.ctypes.data, buf.nbytes, C.byref(need)),
                   "tpcst_debug_fetch")
        return buf[: need.value // dt.itemsize]
