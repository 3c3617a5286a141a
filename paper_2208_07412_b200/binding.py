"""ctypes binding of libtpcca.so (include/tpcca.h).  Argument marshalling only.

Names follow the C-ABI: Tracker.load_clusters / run / get_tracks wrap tpcca_load_clusters /
tpcca_run / tpcca_get_tracks; the constructor wraps tpcca_workspace_bytes + tpcca_create and
close() wraps tpcca_destroy.  PyTorch provides the device workspace and the stream.
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os

import numpy as np

from . import build as _build

STAGE_GRID, STAGE_NEIGHBOURS, STAGE_CLEAN, STAGE_START, STAGE_TRACKLETS, STAGE_ALL = 1, 2, 4, 8, 16, 31
STAGE_SELECT, STAGE_RESIDUALS, STAGE_MERGE = 32, 64, 128
MEM_HOST, MEM_DEVICE, MEM_DEVICE_BORROW = 0, 1, 2

_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int32)
_up = C.POINTER(C.c_uint32)

#: every symbol include/tpcca.h declares
ABI_SYMBOLS = ("tpcca_workspace_bytes", "tpcca_create", "tpcca_load_clusters", "tpcca_reset", "tpcca_run",
               "tpcca_sync", "tpcca_get_tracks", "tpcca_get_counts", "tpcca_get_timings", "tpcca_get_work_counters",
               "tpcca_get_launch_count", "tpcca_get_info", "tpcca_get_tracks_all", "tpcca_pipeline_workspace_bytes",
               "tpcca_pipeline_create", "tpcca_pipeline_run", "tpcca_pipeline_get_groups", "tpcca_pipeline_last_error",
               "tpcca_pipeline_destroy", "tpcca_last_error", "tpcca_destroy", "tpcca_version", "tpcca_start_hits_noalloc")
OUT_ORDER, OUT_GRID, OUT_LINKS_RAW, OUT_LINKS, OUT_START, OUT_TRACKS, OUT_ALL = 1, 2, 4, 8, 16, 32, 63
OUT_SELECTION, OUT_TRACKS_SEL, OUT_RESIDUALS, OUT_MERGE = 64, 128, 256, 512


class TpccaError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"tpcca error {code}: {msg}")
        self.code = code


class _Params(C.Structure):
    _fields_ = [
        ("n_sectors", C.c_int32), ("n_rows", C.c_int32),
        ("row_x", _fp), ("grid_y_lo", _fp), ("grid_inv_bin_y", _fp), ("grid_ny", _ip),
        ("grid_z_lo", C.c_float), ("grid_inv_bin_z", _fp), ("grid_nz", _ip),
        ("nf_hy_up", _fp), ("nf_hz_up", _fp), ("nf_hy_dn", _fp), ("nf_hz_dn", _fp), ("nf_cut", _fp),
        ("kappa_per_qpt", C.c_float), ("err2_y", C.c_float), ("err2_z", C.c_float),
        ("init_cov", C.c_float * 5),
        ("tc_win_y", C.c_float), ("tc_win_z", C.c_float), ("tc_gate", C.c_float),
        ("max_sinphi", C.c_float), ("grid_margin", C.c_float),
        ("tc_max_gap", C.c_int32), ("tc_min_hits", C.c_int32), ("sel_max_shared_permille", C.c_int32),
        ("res_inv_quantum", C.c_float),
        ("sectors_per_side", C.c_int32), ("sector_cos", C.c_float), ("sector_sin", C.c_float),
        ("mg_max_row_gap", C.c_int32), ("mg_dy", C.c_float), ("mg_dz", C.c_float), ("mg_dsin", C.c_float),
        ("mg_zpre", C.c_float),
    ]


class _View(C.Structure):
    _fields_ = [
        ("n_clusters", C.c_int64), ("n_bins", C.c_int64), ("n_start", C.c_int64), ("n_tracks", C.c_int64),
        ("n_hits", C.c_int64), ("trk_stride", C.c_int64),
        ("order", _ip), ("syz", _fp), ("bin_start", _up), ("row_start", _ip),
        ("link_up_raw", _ip), ("link_dn_raw", _ip), ("link_up", _ip), ("link_dn", _ip),
        ("start_hit", _ip),
        ("x_ref", _fp), ("z_ref", _fp), ("par", _fp), ("cov", _fp), ("chi2", _fp),
        ("n_hits_trk", _ip), ("n_fit", _ip), ("first_row", _ip), ("last_row", _ip), ("trk_start_hit", _ip),
        ("hit_offset", _ip), ("hit_idx", _ip),
        ("n_selected", C.c_int64), ("n_sel_hits", C.c_int64), ("owner", _ip), ("n_own", _ip), ("sel_track", _ip),
        ("res", C.c_void_p),
        ("mg_stride", C.c_int64),
        ("mg_next_sec", _ip), ("mg_next_trk", _ip), ("mg_prev_sec", _ip), ("mg_prev_trk", _ip),
        ("mg_n_seg", _ip), ("mg_n_hits", _ip), ("mg_n_fit", _ip), ("mg_first_row", _ip), ("mg_last_row", _ip), ("mg_frame_seg", _ip),
        ("mg_x_ref", _fp), ("mg_z_ref", _fp), ("mg_chi2", _fp), ("mg_par", _fp), ("mg_cov", _fp),
    ]


#: numpy view of tpcca_residual (include/tpcca.h)
RESIDUAL_DTYPE = np.dtype([("trk", np.int32), ("res_y", np.float32), ("res_z", np.float32), ("q_y", np.int16), ("q_z", np.int16)])

_lib = None


def library_path() -> str:
    return _build.LIB


def load_library():
    """Load libtpcca.so (building it first if the sources are newer).  Fails loudly: no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build it with `python -m paper_2208_07412_b200.build`")
    lib = C.CDLL(path)
    lib.tpcca_workspace_bytes.argtypes = [C.POINTER(_Params), C.c_int64, C.c_int64, C.POINTER(C.c_size_t)]
    lib.tpcca_create.argtypes = [C.POINTER(_Params), C.c_int, C.c_void_p, C.c_void_p, C.c_size_t, C.c_int64,
                                 C.c_int64, C.POINTER(C.c_void_p)]
    lib.tpcca_load_clusters.argtypes = [C.c_void_p, C.c_int, C.c_int64] + [C.c_void_p] * 5 + [C.c_int]
    lib.tpcca_reset.argtypes = [C.c_void_p]
    lib.tpcca_run.argtypes = [C.c_void_p, C.c_uint32]
    lib.tpcca_sync.argtypes = [C.c_void_p]
    lib.tpcca_get_tracks.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_uint32, C.POINTER(_View)]
    lib.tpcca_get_counts.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
    lib.tpcca_get_timings.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_float)]
    lib.tpcca_get_work_counters.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
    lib.tpcca_get_launch_count.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
    lib.tpcca_get_info.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
    lib.tpcca_get_tracks_all.argtypes = [C.c_void_p, C.c_int, C.c_uint32, C.POINTER(_View)]
    lib.tpcca_pipeline_workspace_bytes.argtypes = [C.POINTER(_Params), C.c_int, C.c_int64, C.c_int64, C.POINTER(C.c_size_t)]
    lib.tpcca_pipeline_create.argtypes = [C.POINTER(_Params), C.c_int, C.c_int, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                          C.c_size_t, C.c_int64, C.c_int64, C.POINTER(C.c_void_p)]
    lib.tpcca_pipeline_run.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                       C.POINTER(C.c_void_p), C.c_int, C.c_uint32, C.c_uint32, C.POINTER(_View)]
    lib.tpcca_pipeline_get_groups.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_float)]
    lib.tpcca_pipeline_last_error.argtypes = [C.c_void_p]
    lib.tpcca_pipeline_last_error.restype = C.c_char_p
    lib.tpcca_pipeline_destroy.argtypes = [C.c_void_p]
    lib.tpcca_pipeline_destroy.restype = None
    lib.tpcca_last_error.argtypes = [C.c_void_p]
    lib.tpcca_last_error.restype = C.c_char_p
    lib.tpcca_destroy.argtypes = [C.c_void_p]
    lib.tpcca_destroy.restype = None
    lib.tpcca_version.restype = C.c_char_p
    lib.tpcca_start_hits_noalloc.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_int64,
                                             C.c_void_p, C.c_char_p, C.c_size_t]
    _lib = lib
    return lib


def abi_symbols():
    return ABI_SYMBOLS


def _f32(a):
    return np.ascontiguousarray(np.asarray(a), dtype=np.float32)


def _make_params(P):
    """tpcsynth.TrackerParams (or anything with the same attributes) -> (_Params, keep-alive)."""
    keep = {k: _f32(getattr(P, k)) for k in ("row_x", "grid_y_lo", "grid_inv_bin_y", "grid_inv_bin_z", "nf_hy_up",
                                             "nf_hz_up", "nf_hy_dn", "nf_hz_dn", "nf_cut")}
    keep["grid_ny"] = np.ascontiguousarray(P.grid_ny, dtype=np.int32)
    keep["grid_nz"] = np.ascontiguousarray(P.grid_nz, dtype=np.int32)
    p = _Params()
    p.n_sectors = int(P.n_sectors)
    p.n_rows = int(P.n_rows)
    for k in ("row_x", "grid_y_lo", "grid_inv_bin_y", "grid_inv_bin_z", "nf_hy_up", "nf_hz_up", "nf_hy_dn", "nf_hz_dn",
              "nf_cut"):
        setattr(p, k, keep[k].ctypes.data_as(_fp))
    p.grid_ny = keep["grid_ny"].ctypes.data_as(_ip)
    p.grid_nz = keep["grid_nz"].ctypes.data_as(_ip)
    p.grid_z_lo = float(P.grid_z_lo)
    p.kappa_per_qpt = float(P.kappa_per_qpt)
    p.err2_y = float(P.err2_y)
    p.err2_z = float(P.err2_z)
    for i in range(5):
        p.init_cov[i] = float(P.init_cov[i])
    p.tc_win_y = float(P.tc_win_y); p.tc_win_z = float(P.tc_win_z); p.tc_gate = float(P.tc_gate)
    p.max_sinphi = float(P.max_sinphi); p.grid_margin = float(P.grid_margin)
    p.tc_max_gap = int(P.tc_max_gap); p.tc_min_hits = int(P.tc_min_hits)
    p.sel_max_shared_permille = int(getattr(P, "sel_max_shared_permille", 500))
    p.res_inv_quantum = float(getattr(P, "res_inv_quantum", 128.0))
    p.sectors_per_side = int(getattr(P, "sectors_per_side", 18))
    p.sector_cos = float(getattr(P, "sector_cos", np.float32(np.cos(np.pi / 9))))
    p.sector_sin = float(getattr(P, "sector_sin", np.float32(np.sin(np.pi / 9))))
    p.mg_max_row_gap = int(getattr(P, "mg_max_row_gap", 8))
    p.mg_dy = float(getattr(P, "mg_dy", 1.0)); p.mg_dz = float(getattr(P, "mg_dz", 1.0))
    p.mg_dsin = float(getattr(P, "mg_dsin", 0.05)); p.mg_zpre = float(getattr(P, "mg_zpre", 32.0))
    return p, keep


def workspace_bytes(params, max_clusters: int, max_start_hits: int = 0) -> int:
    """tpcca_workspace_bytes (host-only call; needs no GPU)."""
    lib = load_library()
    p, _keep = _make_params(params)
    out = C.c_size_t(0)
    rc = lib.tpcca_workspace_bytes(C.byref(p), int(max_clusters), int(max_start_hits), C.byref(out))
    if rc:
        raise TpccaError(rc, lib.tpcca_last_error(None).decode())
    return int(out.value)


#: size limit of start_hits_noalloc (TPCCA_NOALLOC_MAX_CLUSTERS in include/tpcca.h)
NOALLOC_MAX_CLUSTERS = 1 << 24


def start_hits_noalloc(link_up, link_dn, start_hit, n_start, stream=None):
    """tpcca_start_hits_noalloc: S4 start-hit selection on the cleaned links of one sector, for callers that may
    not allocate device memory (a step inside a framework that owns all of the GPU's memory, a plug-in under a
    caching allocator, a hook without a tpcca context) -- include/tpcca.h says who they are and why.

    Every buffer is the caller's: `link_up`, `link_dn` int32 CUDA tensors of equal length (inputs), `start_hit` an
    int32 CUDA tensor whose length is the capacity, `n_start` an int32 CUDA tensor of one element.  Neither this
    wrapper nor the C call allocates; the call queues three kernels on `stream` (default: torch's current stream)
    and returns.  Afterwards n_start[0] holds the number of start hits found and start_hit[:n_start[0]] the hits in
    ascending position (only the first len(start_hit) are stored if more were found).  At most
    NOALLOC_MAX_CLUSTERS links per call (TpccaError beyond); calls that overlap on one GPU share the library's
    fixed scratch and race -- keep them on one stream.  Argument marshalling only."""
    import torch
    lib = load_library()
    for name, t in (("link_up", link_up), ("link_dn", link_dn), ("start_hit", start_hit), ("n_start", n_start)):
        if not (t.is_cuda and t.dtype == torch.int32 and t.is_contiguous()):
            raise TypeError(f"{name} must be a contiguous int32 CUDA tensor")
    if link_up.numel() != link_dn.numel() or n_start.numel() != 1:
        raise ValueError("link_up and link_dn must have the same length, n_start exactly one element")
    dev = link_up.device
    if any(t.device != dev for t in (link_dn, start_hit, n_start)):
        raise ValueError("all tensors must be on the same device")
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    msg = C.create_string_buffer(512)
    rc = lib.tpcca_start_hits_noalloc(dev.index, C.c_void_p(st.cuda_stream), C.c_void_p(link_up.data_ptr()),
                                      C.c_void_p(link_dn.data_ptr()), link_up.numel(), C.c_void_p(start_hit.data_ptr()),
                                      start_hit.numel(), C.c_void_p(n_start.data_ptr()), msg, len(msg))
    if rc:
        raise TpccaError(rc, msg.value.decode())


@dataclasses.dataclass
class SectorOutput:
    """Host copies of one sector's outputs (same field names as the C view; index space: sorted positions)."""
    n: int
    n_bins: int = 0
    order: np.ndarray = None
    sy: np.ndarray = None
    sz: np.ndarray = None
    bin_start: np.ndarray = None
    row_start: np.ndarray = None
    link_up_raw: np.ndarray = None
    link_dn_raw: np.ndarray = None
    link_up: np.ndarray = None
    link_dn: np.ndarray = None
    start_hit: np.ndarray = None
    x_ref: np.ndarray = None
    z_ref: np.ndarray = None
    par: np.ndarray = None      # [n_tracks, 5]
    cov: np.ndarray = None      # [n_tracks, 15]
    chi2: np.ndarray = None
    n_hits: np.ndarray = None
    n_fit: np.ndarray = None
    first_row: np.ndarray = None
    last_row: np.ndarray = None
    trk_start_hit: np.ndarray = None
    hit_offset: np.ndarray = None
    hit_idx: np.ndarray = None
    owner: np.ndarray = None       # S6
    n_own: np.ndarray = None
    selected: np.ndarray = None
    res_trk: np.ndarray = None     # S7
    res_y: np.ndarray = None
    res_z: np.ndarray = None
    q_y: np.ndarray = None
    q_z: np.ndarray = None
    merge: dict = None             # S8: per selected track: next_sec, next_trk, prev_sec, prev_trk, n_seg, ..., par, cov

    @property
    def n_tracks(self) -> int:
        return 0 if self.x_ref is None else int(self.x_ref.shape[0])


def _np(ptr, n, dtype):
    if not ptr or n == 0:
        return np.empty(0, dtype) if ptr else None
    return np.ctypeslib.as_array(ptr, shape=(n,)).astype(dtype, copy=True)


def output_from_view(v, what: int, n_rows: int) -> SectorOutput:
    """HOST tpcca_tracks_view -> numpy copies (argument marshalling only)."""
    n, nt = int(v.n_clusters), int(v.n_tracks)
    o = SectorOutput(n=n, n_bins=int(v.n_bins))
    o.order = _np(v.order, n, np.int32)
    if v.syz:
        syz = _np(v.syz, 2 * n, np.float32).reshape(n, 2)
        o.sy, o.sz = np.ascontiguousarray(syz[:, 0]), np.ascontiguousarray(syz[:, 1])
    o.bin_start = _np(v.bin_start, int(v.n_bins) + 1, np.uint32) if v.bin_start else None
    o.row_start = _np(v.row_start, n_rows + 1, np.int32) if v.row_start else None
    o.link_up_raw = _np(v.link_up_raw, n, np.int32); o.link_dn_raw = _np(v.link_dn_raw, n, np.int32)
    o.link_up = _np(v.link_up, n, np.int32); o.link_dn = _np(v.link_dn, n, np.int32)
    o.start_hit = _np(v.start_hit, int(v.n_start), np.int32)
    if what & OUT_TRACKS_SEL:          # the S5 fields hold the selected tracks only
        nt = int(v.n_selected)
    n_hits_total = int(v.n_sel_hits) if what & OUT_TRACKS_SEL else int(v.n_hits)
    if v.owner:
        o.owner = _np(v.owner, n, np.int32); o.n_own = _np(v.n_own, int(v.n_tracks), np.int32)
        o.selected = _np(v.sel_track, int(v.n_selected), np.int32)
    if v.res:
        rec = np.frombuffer((C.c_char * (16 * n)).from_address(v.res), dtype=RESIDUAL_DTYPE, count=n) if n else np.empty(0, RESIDUAL_DTYPE)
        o.res_trk, o.res_y, o.res_z, o.q_y, o.q_z = (np.ascontiguousarray(rec[f]) for f in ("trk", "res_y", "res_z", "q_y", "q_z"))
    if v.mg_next_sec:
        nk = int(v.n_selected)
        o.merge = {f: _np(getattr(v, "mg_" + f), nk, np.int32) for f in ("next_sec", "next_trk", "prev_sec", "prev_trk", "n_seg",
                                                                          "n_hits", "n_fit", "first_row", "last_row", "frame_seg")}
        for f in ("x_ref", "z_ref", "chi2"):
            o.merge[f] = _np(getattr(v, "mg_" + f), nk, np.float32)
        ms = int(v.mg_stride)
        o.merge["par"] = _np(v.mg_par, 5 * ms, np.float32).reshape(5, ms)[:, :nk].T.copy() if nk else np.empty((0, 5), np.float32)
        o.merge["cov"] = _np(v.mg_cov, 15 * ms, np.float32).reshape(15, ms)[:, :nk].T.copy() if nk else np.empty((0, 15), np.float32)
    if v.x_ref:
        o.x_ref = _np(v.x_ref, nt, np.float32); o.z_ref = _np(v.z_ref, nt, np.float32)
        o.chi2 = _np(v.chi2, nt, np.float32)
        stride = int(v.trk_stride)
        o.par = (_np(v.par, 5 * stride, np.float32).reshape(5, stride)[:, :nt].T.copy() if nt
                 else np.empty((0, 5), np.float32))
        o.cov = (_np(v.cov, 15 * stride, np.float32).reshape(15, stride)[:, :nt].T.copy() if nt
                 else np.empty((0, 15), np.float32))
        o.n_hits = _np(v.n_hits_trk, nt, np.int32); o.n_fit = _np(v.n_fit, nt, np.int32)
        o.first_row = _np(v.first_row, nt, np.int32); o.last_row = _np(v.last_row, nt, np.int32)
        o.trk_start_hit = _np(v.trk_start_hit, nt, np.int32)
        o.hit_offset = _np(v.hit_offset, nt + 1, np.int32)
        o.hit_idx = _np(v.hit_idx, n_hits_total, np.int32)
    return o


class Tracker:
    """One tpcca context: tables + a torch-owned device workspace + the current torch stream."""

    def __init__(self, params, max_clusters: int, max_start_hits: int = 0, device: int = 0, stream=None,
                 workspace_fill: int | None = None):
        import torch  # device memory and streams only
        self._lib = load_library()
        if not torch.cuda.is_available():
            raise TpccaError(-3, "no CUDA device: tpcca has no CPU path")
        self._torch = torch
        self.device = int(device)
        self.n_sectors = int(params.n_sectors)
        self.n_rows = int(params.n_rows)
        p, self._keep = _make_params(params)
        nbytes = C.c_size_t(0)
        rc = self._lib.tpcca_workspace_bytes(C.byref(p), int(max_clusters), int(max_start_hits), C.byref(nbytes))
        if rc:
            raise TpccaError(rc, self._lib.tpcca_last_error(None).decode())
        self.workspace_bytes = int(nbytes.value)
        with torch.cuda.device(self.device):
            self._ws = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=f"cuda:{self.device}")
            if workspace_fill is not None:      # tests: the library must not depend on what the workspace held
                self._ws.fill_(int(workspace_fill))
                torch.cuda.synchronize(self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        base = self._ws.data_ptr()
        aligned = (base + 255) // 256 * 256
        h = C.c_void_p()
        rc = self._lib.tpcca_create(C.byref(p), self.device, C.c_void_p(self._stream.cuda_stream), C.c_void_p(aligned),
                                    self.workspace_bytes, int(max_clusters), int(max_start_hits), C.byref(h))
        if rc:
            raise TpccaError(rc, self._lib.tpcca_last_error(None).decode())
        self._h = h
        self._inputs = []   # keep host / borrowed arrays alive until the next reset

    # ------------------------------------------------------------------------------------------
    def _check(self, rc):
        if rc:
            raise TpccaError(rc, self._lib.tpcca_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.tpcca_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # ------------------------------------------------------------------------------------------
    def reset(self):
        self._check(self._lib.tpcca_reset(self._h))
        self._inputs.clear()

    def load_clusters(self, sector: int, y, z, row, x=None, charge=None, borrow: bool = False):
        """tpcca_load_clusters.  numpy arrays / pinned torch CPU tensors -> HOST copy; torch CUDA tensors ->
        DEVICE copy (or in-place use with borrow=True)."""
        torch = self._torch
        if isinstance(y, torch.Tensor):
            assert y.dtype == torch.float32 and z.dtype == torch.float32 and row.dtype in (torch.uint16, torch.int16)
            assert y.is_contiguous() and z.is_contiguous() and row.is_contiguous()
            n = int(y.shape[0])
            if y.is_cuda:
                space = MEM_DEVICE_BORROW if borrow else MEM_DEVICE
            else:
                space = MEM_HOST
            ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None and t.numel() else None
            self._inputs.append((y, z, row))
            self._check(self._lib.tpcca_load_clusters(self._h, int(sector), n, ptr(x), ptr(y), ptr(z), ptr(charge),
                                                      ptr(row), space))
            return
        y = _f32(y); z = _f32(z)
        row = np.ascontiguousarray(row, dtype=np.uint16)
        n = int(y.shape[0])
        self._inputs.append((y, z, row))
        ptr = lambda a: C.c_void_p(a.ctypes.data) if a is not None and a.size else None
        xx = _f32(x) if x is not None else None
        qq = _f32(charge) if charge is not None else None
        self._check(self._lib.tpcca_load_clusters(self._h, int(sector), n, ptr(xx), ptr(y), ptr(z), ptr(qq), ptr(row),
                                                  MEM_HOST))

    def load_timeframe(self, tf):
        """Load every sector of a tpcsynth.Timeframe (host arrays)."""
        self.reset()
        for s in range(tf.n_sectors):
            self.load_clusters(s, tf.y[s], tf.z[s], tf.row[s], x=tf.x[s], charge=tf.q[s])

    def run(self, stage_mask: int = STAGE_ALL):
        self._check(self._lib.tpcca_run(self._h, int(stage_mask)))

    def sync(self):
        self._check(self._lib.tpcca_sync(self._h))

    def counts(self) -> dict:
        out = (C.c_int64 * 7)()
        self._check(self._lib.tpcca_get_counts(self._h, out))
        return dict(n_clusters=int(out[0]), n_start=int(out[1]), n_tracks=int(out[2]), n_hits=int(out[3]),
                    n_bins=int(out[4]), n_selected=int(out[5]), n_sel_hits=int(out[6]))

    def timings(self, runs_back: int = 0):
        """Per-stage device ms of a recent run (0 = last): [S1, S2, S3, S4, S5, S1..S5, S6, S7, S8]."""
        out = (C.c_float * 9)()
        self._check(self._lib.tpcca_get_timings(self._h, int(runs_back), out))
        return [float(v) for v in out]

    def work_counters(self) -> dict:
        """S5 work counters of the last run (tpcca_get_work_counters)."""
        out = (C.c_int64 * 5)()
        self._check(self._lib.tpcca_get_work_counters(self._h, out))
        return dict(zip(("propagations", "updates", "gates", "searches", "candidates"), (int(v) for v in out)))

    def info(self) -> dict:
        """tpcca_get_info: how tpcca_create configured the context."""
        out = (C.c_int64 * 8)()
        self._check(self._lib.tpcca_get_info(self._h, out))
        return dict(zip(("slab_shift", "n_coarse_buckets", "s2_variant", "sm_count", "s2_blocks_per_sm", "max_clusters",
                         "max_start_hits", "workspace_bytes"), (int(v) for v in out)))

    def launch_count(self) -> int:
        out = C.c_int64(0)
        self._check(self._lib.tpcca_get_launch_count(self._h, C.byref(out)))
        return int(out.value)

    def get_tracks_view(self, sector: int, mem_space: int = MEM_DEVICE, what: int = OUT_ALL) -> _View:
        """Raw tpcca_tracks_view (device pointers by default; HOST pointers live in the context's pinned
        arena until the next call)."""
        v = _View()
        self._check(self._lib.tpcca_get_tracks(self._h, int(sector), int(mem_space), int(what), C.byref(v)))
        return v

    def get_tracks(self, sector: int, what: int = OUT_ALL) -> SectorOutput:
        """tpcca_get_tracks(HOST) -> numpy copies."""
        return output_from_view(self.get_tracks_view(sector, MEM_HOST, what), what, self.n_rows)

    def get_tracks_all_views(self, mem_space: int = MEM_HOST, what: int = OUT_ALL):
        """Raw tpcca_get_tracks_all: the views of every sector (HOST: one arena, one synchronise; valid until the next
        HOST fetch)."""
        views = (_View * self.n_sectors)()
        self._check(self._lib.tpcca_get_tracks_all(self._h, int(mem_space), int(what), views))
        return views

    def get_tracks_all(self, what: int = OUT_ALL):
        """tpcca_get_tracks_all(HOST): every sector behind one synchronise -> list of SectorOutput."""
        views = (_View * self.n_sectors)()
        self._check(self._lib.tpcca_get_tracks_all(self._h, MEM_HOST, int(what), views))
        return [output_from_view(views[s], what, self.n_rows) for s in range(self.n_sectors)]


class Pipeline:
    """tpcca_pipeline: a time frame streamed through n_groups sector groups (one context, stream, host thread and
    workspace each).  PyTorch lends the streams and the workspaces."""

    def __init__(self, params, n_groups: int, max_clusters_group: int, max_start_hits_group: int = 0, device: int = 0):
        import torch
        self._lib = load_library()
        if not torch.cuda.is_available():
            raise TpccaError(-3, "no CUDA device: tpcca has no CPU path")
        self.n_sectors, self.n_rows, self.n_groups = int(params.n_sectors), int(params.n_rows), int(n_groups)
        self._torch, self.device = torch, int(device)
        p, self._keep = _make_params(params)
        nbytes = C.c_size_t(0)
        rc = self._lib.tpcca_pipeline_workspace_bytes(C.byref(p), self.n_groups, int(max_clusters_group), int(max_start_hits_group),
                                                      C.byref(nbytes))
        if rc:
            raise TpccaError(rc, self._lib.tpcca_pipeline_last_error(None).decode())
        self.workspace_bytes_each = int(nbytes.value)
        with torch.cuda.device(device):
            self._streams = [torch.cuda.Stream(device=device) for _ in range(self.n_groups)]
            self._ws = [torch.empty(self.workspace_bytes_each + 256, dtype=torch.uint8, device=f"cuda:{device}")
                        for _ in range(self.n_groups)]
        st = (C.c_void_p * self.n_groups)(*[s.cuda_stream for s in self._streams])
        ws = (C.c_void_p * self.n_groups)(*[(w.data_ptr() + 255) // 256 * 256 for w in self._ws])
        h = C.c_void_p()
        rc = self._lib.tpcca_pipeline_create(C.byref(p), int(device), self.n_groups, st, ws, self.workspace_bytes_each,
                                             int(max_clusters_group), int(max_start_hits_group), C.byref(h))
        if rc:
            raise TpccaError(rc, self._lib.tpcca_pipeline_last_error(None).decode())
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self._lib.tpcca_pipeline_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def run_views(self, y, z, row, stage_mask: int = STAGE_ALL, what: int = OUT_ALL):
        """tpcca_pipeline_run on per-sector arrays (numpy / pinned torch CPU tensors: HOST; torch CUDA tensors: DEVICE).
        Returns the raw views (HOST pointers, valid until the next run)."""
        ns = self.n_sectors
        assert len(y) == ns and len(z) == ns and len(row) == ns
        is_t = hasattr(y[0], "data_ptr")
        dev = is_t and y[0].is_cuda
        ptr = (lambda a: a.data_ptr() if a.numel() else None) if is_t else (lambda a: a.ctypes.data if a.size else None)
        if not is_t:
            y = [_f32(a) for a in y]; z = [_f32(a) for a in z]
            row = [np.ascontiguousarray(a, dtype=np.uint16) for a in row]
        self._inputs = (y, z, row)
        n = (C.c_int64 * ns)(*[int(a.shape[0]) for a in y])
        py = (C.c_void_p * ns)(*[ptr(a) for a in y]); pz = (C.c_void_p * ns)(*[ptr(a) for a in z])
        pr = (C.c_void_p * ns)(*[ptr(a) for a in row])
        views = (_View * ns)()
        if dev:
            # the groups copy the inputs on their own streams: order those copies after whatever the caller's current
            # stream still has queued on the tensors (a kernel writing them, an asynchronous upload)
            cur = self._torch.cuda.current_stream(self.device)
            for s in self._streams:
                s.wait_stream(cur)
        rc = self._lib.tpcca_pipeline_run(self._h, n, py, pz, pr, MEM_DEVICE if dev else MEM_HOST, int(stage_mask), int(what), views)
        if rc:
            raise TpccaError(rc, self._lib.tpcca_pipeline_last_error(self._h).decode())
        return views

    def run(self, y, z, row, stage_mask: int = STAGE_ALL, what: int = OUT_ALL):
        views = self.run_views(y, z, row, stage_mask, what)
        return [output_from_view(views[s], what, self.n_rows) for s in range(self.n_sectors)]

    def groups(self):
        first = (C.c_int32 * (self.n_groups + 1))()
        ms = (C.c_float * self.n_groups)()
        self._lib.tpcca_pipeline_get_groups(self._h, first, ms)
        return list(first), [float(v) for v in ms]
