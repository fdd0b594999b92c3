"""Thin Python binding of libtpc_b200.so (include/tpc_b200.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; PyTorch is used for device memory and
streams.  There is no CPU fallback: loading fails loudly when the library is missing or cannot be built,
and every compute entry point refuses non-CUDA tensors.

    lib = binding.load()
    trk = binding.Tracker(params, n_clusters)          # allocates workspace + outputs once
    res = trk.run(y, z, sector_row)                     # tpc_grid_build -> tpc_find_tracks -> tpc_fit_tracks
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

TPC_MAX_ROWS = 152
TPC_N_COUNTERS = 16
TPC_MAX_TRACKLETS = 1 << 25
CNT_TRACKS, CNT_TRACKLETS, CNT_HITS, CNT_STATUS, CNT_STARTS_FOUND, CNT_TRACKS_FOUND = 0, 1, 2, 3, 4, 5
CNT_FOLLOWED_DOWN = 6
CNT_PROP_LO, CNT_UPD_LO, CNT_CAND_LO, CNT_CLAIMS_LO = 8, 10, 12, 14
ST_TRACKLET_OVERFLOW, ST_TRACK_OVERFLOW, ST_Z_CLAMPED, ST_BAD_ROW = 1, 2, 4, 8

#: every symbol include/tpc_b200.h declares (checked by tests/test_abi.py against the header text)
SYMBOLS = ("tpc_strerror", "tpc_last_cuda_error", "tpc_version", "tpc_grid_bins", "tpc_workspace_bytes",
           "tpc_grid_build", "tpc_grid_export", "tpc_find_tracks", "tpc_find_export", "tpc_fit_tracks",
           "tpc_track_time", "tpc_collisions_workspace_bytes", "tpc_find_collisions", "tpc_merge_workspace_bytes",
           "tpc_merge_tracks", "tpc_clusterize_workspace_bytes", "tpc_clusterize", "tpc_fit_tracks_physics",
           "tpc_tag_clusters", "tpc_pair_sides_workspace_bytes", "tpc_pair_sides", "tpc_pair_sides_static", "tpc_track_host", "tpc_track_host_async", "tpc_track_host_fetch", "tpc_profile_enable", "tpc_profile_kernels", "tpc_profile_name", "tpc_profile_collect", "tpc_fp32_peak")


class tpc_params_t(C.Structure):
    """Mirror of the host POD in include/tpc_b200.h."""
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", C.c_float * TPC_MAX_ROWS),
                ("tan_half", C.c_float), ("kB", C.c_float), ("sigma_y", C.c_float), ("sigma_z", C.c_float),
                ("z_lo", C.c_float), ("z_hi", C.c_float), ("cell_y", C.c_float), ("cell_z", C.c_float),
                ("ca_max_dydx", C.c_float), ("ca_max_dzdx", C.c_float), ("ca_cut", C.c_float),
                ("chi2_cut", C.c_float), ("chi2_chain_cut", C.c_float), ("win_max", C.c_float),
                ("max_sinphi", C.c_float), ("edge_margin", C.c_float),
                ("max_gap", C.c_int32), ("min_hits", C.c_int32), ("n_fit_passes", C.c_int32),
                ("cov0", C.c_float * 5)]


class tpc_result_t(C.Structure):
    """Mirror of tpc_result_t: the outputs of find + fit, as device buffers or as pinned host buffers."""
    _fields_ = [(nm, C.c_void_p) for nm in ("cluster_track", "trk_seed", "trk_sector", "trk_nhits", "trk_first_hit", "trk_hits",
                                            "counters", "par", "cov", "xref", "zref", "chi2", "ndf")]


RESULT_FIELDS = tuple(f[0] for f in tpc_result_t._fields_)


class tpc_merge_params_t(C.Structure):
    _fields_ = [("chi2_cut", C.c_float), ("dz_max", C.c_float), ("ce_tol", C.c_float), ("max_rows", C.c_int32)]


class tpc_fit_options_t(C.Structure):
    """Mirror of tpc_fit_options_t (R28a, b, d, e)."""
    _fields_ = [(nm, C.c_float) for nm in ("x0inv", "outlier_cut", "dedx", "eloss_sigma", "err_ang_y", "err_ang_z", "err_drift_y",
                                           "err_drift_z", "v_drift", "z_len")]


class tpc_merged_t(C.Structure):
    """Mirror of tpc_merged_t: device outputs of tpc_merge_tracks (R26)."""
    _fields_ = [(nm, C.c_void_p) for nm in ("trk_succ", "trk_pred", "trk_succ_chi2", "trk_global", "n_global", "g_head", "g_nseg",
                                            "g_nhits", "gpar", "gcov", "gxref", "gzref", "gchi2", "gndf")]


MERGE_DEFAULTS = dict(chi2_cut=50.0, dz_max=64.0, ce_tol=1.0, max_rows=12)


class TpcError(RuntimeError):
    pass


_lib = None


def load(rebuild: bool = False):
    """Load (building in-tree first if needed) libtpc_b200.so.  Raises if it cannot be had."""
    global _lib
    if _lib is not None and not rebuild:
        return _lib
    path = _build.LIB
    if rebuild or not _build.up_to_date():
        try:
            path = _build.build_library(force=rebuild)
        except Exception as e:  # no nvcc on this machine: use the shipped binary if there is one
            if not os.path.exists(path):
                raise TpcError(f"libtpc_b200.so is missing and cannot be built ({e}); there is no CPU fallback") from e
    L = C.CDLL(path)
    for name in SYMBOLS:
        if not hasattr(L, name):
            raise TpcError(f"libtpc_b200.so does not export {name}")
    for name in ("tpc_strerror", "tpc_last_cuda_error", "tpc_version"):
        getattr(L, name).restype = C.c_char_p
    for name in SYMBOLS[3:]:
        getattr(L, name).restype = C.c_int
    L.tpc_profile_name.restype = C.c_char_p
    _lib = L
    return L


def make_params(p) -> tpc_params_t:
    """Marshal a TpcParams-like object (attribute names of tpc_params_t) into the C struct."""
    P = tpc_params_t()
    P.n_sectors, P.n_rows = int(p.n_sectors), int(p.n_rows)
    rx = np.asarray(p.row_x, dtype=np.float32)
    if not (0 < P.n_rows <= TPC_MAX_ROWS) or rx.size < P.n_rows:
        raise TpcError(f"n_rows = {P.n_rows} outside 1..{TPC_MAX_ROWS} or row_x too short")
    for i in range(P.n_rows):
        P.row_x[i] = float(rx[i])
    for name in ("tan_half", "kB", "sigma_y", "sigma_z", "z_lo", "z_hi", "cell_y", "cell_z", "ca_max_dydx",
                 "ca_max_dzdx", "ca_cut", "chi2_cut", "chi2_chain_cut", "win_max", "max_sinphi", "edge_margin"):
        setattr(P, name, float(getattr(p, name)))
    P.max_gap, P.min_hits, P.n_fit_passes = int(p.max_gap), int(p.min_hits), int(p.n_fit_passes)
    for i in range(5):
        P.cov0[i] = float(p.cov0[i])
    return P


def _check(rc: int, what: str):
    if rc != 0:
        L = load()
        msg = L.tpc_strerror(rc).decode()
        if rc == -3:
            msg += " (" + L.tpc_last_cuda_error().decode() + ")"
        raise TpcError(f"{what}: {msg}")


def _dp(t):
    """Device pointer of a CUDA tensor (None -> NULL)."""
    if t is None:
        return C.c_void_p(0)
    if not t.is_cuda:
        raise TpcError("expected a CUDA tensor: the hot path has no CPU implementation")
    if not t.is_contiguous():
        raise TpcError("expected a contiguous tensor")
    return C.c_void_p(t.data_ptr())


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def profile_enable(on: bool):
    """tpc_profile_enable: per-kernel CUDA-event timing on the launching stream."""
    _check(load().tpc_profile_enable(C.c_int(int(on))), "tpc_profile_enable")


def profile_collect(reset: bool = True) -> dict:
    """tpc_profile_collect: {kernel name: (summed ms, launches)} since the last reset (synchronises)."""
    L = load()
    k = L.tpc_profile_kernels()
    ms = (C.c_double * k)()
    cnt = (C.c_int64 * k)()
    _check(L.tpc_profile_collect(C.c_int(k), ms, cnt, C.c_int(int(reset))), "tpc_profile_collect")
    out = {}
    for i in range(k):      # kernel ids that share a name (the two phases of k_follow) are summed
        name = L.tpc_profile_name(i).decode()
        a, b = out.get(name, (0.0, 0))
        out[name] = (a + float(ms[i]), b + int(cnt[i]))
    return out


def fp32_peak(device="cuda:0") -> float:
    """tpc_fp32_peak: measured FFMA-chain rate of the device in TFLOP/s (synchronises)."""
    import torch
    scratch = torch.zeros(64, dtype=torch.float32, device=device)
    out = C.c_double(0.0)
    with torch.cuda.device(scratch.device):
        _check(load().tpc_fp32_peak(_dp(scratch), C.byref(out), _stream()), "tpc_fp32_peak")
    return float(out.value)


def clusterize(params, sector_row, pad, time, adc, pad_width, time_width, peak_min=6, max_clusters=None, want_numpy=True):
    """tpc_clusterize (R27) on CUDA int32 tensors of digits.  Returns dict(y, z, q, sector_row, pad, time, n_found) --
    numpy arrays of the clusters written (order unspecified) -- or, with want_numpy=False, the device tensors and the
    device counter (asynchronous)."""
    import torch
    L = load()
    n = int(sector_row.numel())
    dev = sector_row.device
    cap = int(max_clusters if max_clusters is not None else max(n, 1))
    wsb = C.c_size_t(0)
    _check(L.tpc_clusterize_workspace_bytes(C.c_int64(n), C.byref(wsb)), "tpc_clusterize_workspace_bytes")
    ws = torch.empty(int(wsb.value), dtype=torch.uint8, device=dev)
    f32, i32 = torch.float32, torch.int32
    out = dict(y=torch.empty(cap, dtype=f32, device=dev), z=torch.empty(cap, dtype=f32, device=dev),
               q=torch.empty(cap, dtype=f32, device=dev), sector_row=torch.empty(cap, dtype=i32, device=dev),
               pad=torch.empty(cap, dtype=i32, device=dev), time=torch.empty(cap, dtype=i32, device=dev))
    cnt = torch.zeros(2, dtype=i32, device=dev)
    with torch.cuda.device(dev):
        _check(L.tpc_clusterize(C.byref(make_params(params)), C.c_int64(n), _dp(sector_row), _dp(pad), _dp(time), _dp(adc),
                                C.c_float(pad_width), C.c_float(time_width), C.c_int32(int(peak_min)), _dp(ws),
                                C.c_size_t(int(wsb.value)), C.c_int64(cap), _dp(out["y"]), _dp(out["z"]), _dp(out["q"]),
                                _dp(out["sector_row"]), _dp(out["pad"]), _dp(out["time"]), _dp(cnt), _stream()), "tpc_clusterize")
    if not want_numpy:
        return dict(out, n_clusters=cnt, workspace=ws)
    found, written = (int(v) for v in cnt.cpu().numpy())
    res = {k: v[:written].cpu().numpy() for k, v in out.items()}
    res["n_found"] = found
    return res


PAIR_SIDES_STATIC_MAX = 16384   # TPC_PAIR_SIDES_STATIC_MAX


def pair_sides_static(n_a, t_a, c_a, n_c, t_c, c_c, max_collisions: int, dt_max: float = 15.5, sigma_t: float = 3.88,
                      v_drift: float = 2.58, out=None):
    """tpc_pair_sides_static: the R29 pairing for callers that cannot allocate device memory -- code running inside a
    framework that owns all GPU memory, or anywhere a cudaMalloc (device-wide lock, implicit synchronisation) is not
    acceptable.  The library keeps the two small arg-min tables the pairing needs in an array of its own device image
    (128.5 KiB per GPU, up to PAIR_SIDES_STATIC_MAX = 16384 collisions per side; more raises TpcError "size beyond the
    fixed scratch array").  The result is that of Tracker.pair_sides bit for bit.
    Inputs: the device tensors two find_collisions calls left (n_collisions [2] int32, coll_time float32, coll_ntracks
    int32, side A then side C).  out: optional dict of preallocated device tensors pair_of_a, pair_of_c (int32
    [max_collisions]), t, z_vertex (float32 [max_collisions]), n_pairs (int32 [1]); with it this wrapper allocates
    nothing on the device either and only enqueues (returns `out`).  Without it the outputs are torch tensors made here
    and the numpy dict of Tracker.pair_sides comes back (synchronises).
    The first call on a GPU looks up the array's address: make it before any stream capture.  All calls on a GPU share
    the array: keep them on one stream (calls that overlap on the GPU race)."""
    import torch as t
    cap = int(max_collisions)
    o = out
    if o is None:
        dev = t_a.device
        o = dict(pair_of_a=t.empty(max(cap, 1), dtype=t.int32, device=dev), pair_of_c=t.empty(max(cap, 1), dtype=t.int32, device=dev),
                 t=t.empty(max(cap, 1), dtype=t.float32, device=dev), z_vertex=t.empty(max(cap, 1), dtype=t.float32, device=dev),
                 n_pairs=t.zeros(1, dtype=t.int32, device=dev))
    _check(load().tpc_pair_sides_static(_dp(n_a), _dp(t_a), _dp(c_a), _dp(n_c), _dp(t_c), _dp(c_c), C.c_int64(cap),
                                        C.c_double(dt_max), C.c_double(sigma_t), C.c_double(v_drift), _dp(o["pair_of_a"]),
                                        _dp(o["pair_of_c"]), _dp(o["t"]), _dp(o["z_vertex"]), _dp(o["n_pairs"]), _stream()),
           "tpc_pair_sides_static")
    if out is not None:
        return out
    k = int(o["n_pairs"].item())
    na, nc_ = int(n_a[1].item()), int(n_c[1].item())
    return dict(pair_of_a=o["pair_of_a"][:na].cpu().numpy(), pair_of_c=o["pair_of_c"][:nc_].cpu().numpy(), t=o["t"][:k].cpu().numpy(),
                z_vertex=o["z_vertex"][:k].cpu().numpy())


def work_counts(counters) -> dict:
    """Follower work from the counters array: transports (R12), updates (R13), candidates tested (R16), and the hits
    recorded by the tracklets that went through phase B (the claims the selection works on, R18/R20)."""
    c = np.asarray(counters).astype(np.int64) & 0xFFFFFFFF
    return {"propagations": int(c[CNT_PROP_LO] | (c[CNT_PROP_LO + 1] << 32)),
            "updates": int(c[CNT_UPD_LO] | (c[CNT_UPD_LO + 1] << 32)),
            "candidates": int(c[CNT_CAND_LO] | (c[CNT_CAND_LO + 1] << 32)),
            "claims": int(c[CNT_CLAIMS_LO] | (c[CNT_CLAIMS_LO + 1] << 32))}


def grid_bins(params) -> int:
    out = C.c_int64(0)
    _check(load().tpc_grid_bins(C.byref(make_params(params)), C.byref(out)), "tpc_grid_bins")
    return int(out.value)


def workspace_bytes(params, n_clusters: int, max_tracklets: int) -> int:
    out = C.c_size_t(0)
    _check(load().tpc_workspace_bytes(C.byref(make_params(params)), C.c_int64(n_clusters), C.c_int64(max_tracklets),
                                      C.byref(out)), "tpc_workspace_bytes")
    return int(out.value)


def default_max_tracklets(n_clusters: int) -> int:
    """Start hits are ~4-7 % of the clusters on the BASELINE.json configs; n/8 + 1024 leaves headroom."""
    return min(int(n_clusters) // 8 + 1024, TPC_MAX_TRACKLETS)


def default_max_tracks(n_clusters: int) -> int:
    """Accepted tracks need >= min_hits (10) exclusive clusters each; n/16 + 1024 is never reached in practice."""
    return int(n_clusters) // 16 + 1024


class Tracker:
    """Owns the device buffers for events of up to `n_clusters` clusters and calls the three C entry points."""

    def __init__(self, params, n_clusters: int, max_tracklets: int | None = None, max_tracks: int | None = None,
                 device="cuda:0"):
        import torch
        self.torch = torch
        self.lib = load()
        self.params = params
        self.P = make_params(params)
        self.n = int(n_clusters)
        self.max_tracklets = int(max_tracklets) if max_tracklets is not None else default_max_tracklets(self.n)
        self.max_tracks = int(max_tracks) if max_tracks is not None else default_max_tracks(self.n)
        self.device = torch.device(device)
        self.ws_bytes = workspace_bytes(params, self.n, self.max_tracklets)
        i32, i64, f32 = torch.int32, torch.int64, torch.float32
        dev = self.device
        # torch allocations are >= 512-byte aligned, which satisfies the 256-byte requirement of the workspace
        self.workspace = torch.empty(self.ws_bytes, dtype=torch.uint8, device=dev)
        n1, K = max(self.n, 1), self.max_tracks
        self.cluster_track = torch.empty(n1, dtype=i32, device=dev)
        self.trk_seed = torch.empty(K, dtype=i32, device=dev)
        self.trk_sector = torch.empty(K, dtype=i32, device=dev)
        self.trk_nhits = torch.empty(K, dtype=i32, device=dev)
        self.trk_first_hit = torch.empty(K, dtype=i64, device=dev)
        self.trk_hits = torch.empty(n1, dtype=i32, device=dev)
        self.counters = torch.zeros(TPC_N_COUNTERS, dtype=i32, device=dev)
        self.par = torch.empty((5, K), dtype=f32, device=dev)
        self.cov = torch.empty((15, K), dtype=f32, device=dev)
        self.xref = torch.empty(K, dtype=f32, device=dev)
        self.zref = torch.empty(K, dtype=f32, device=dev)
        self.chi2 = torch.empty(K, dtype=f32, device=dev)
        self.ndf = torch.empty(K, dtype=i32, device=dev)
        self._inputs = None

    # ---- the three calls of the boundary -----------------------------------------------------
    def grid_build(self, y, z, sector_row, x=None, q=None):
        assert y.numel() == self.n and z.numel() == self.n and sector_row.numel() == self.n
        assert y.dtype == self.torch.float32 and z.dtype == self.torch.float32 and sector_row.dtype == self.torch.int32
        self._inputs = (y, z, sector_row)   # keep alive: the fit reads them
        _check(self.lib.tpc_grid_build(C.byref(self.P), C.c_int64(self.n), C.c_int64(self.max_tracklets), _dp(x), _dp(y),
                                       _dp(z), _dp(q), _dp(sector_row), _dp(self.workspace), C.c_size_t(self.ws_bytes),
                                       _stream()), "tpc_grid_build")

    def find_tracks(self):
        _check(self.lib.tpc_find_tracks(C.byref(self.P), C.c_int64(self.n), C.c_int64(self.max_tracklets),
                                        _dp(self.workspace), C.c_size_t(self.ws_bytes), _dp(self.cluster_track),
                                        C.c_int64(self.max_tracks), _dp(self.trk_seed), _dp(self.trk_sector),
                                        _dp(self.trk_nhits), _dp(self.trk_first_hit), _dp(self.trk_hits),
                                        _dp(self.counters), _stream()), "tpc_find_tracks")

    def fit_tracks(self, gather: bool = False):
        """tpc_fit_tracks; gather=True passes workspace = NULL (self-contained gather through y/z/sector_row)."""
        y, z, sr = self._inputs
        ws = C.c_void_p(0) if gather else _dp(self.workspace)
        _check(self.lib.tpc_fit_tracks(C.byref(self.P), C.c_int64(self.n), C.c_int64(self.max_tracklets), ws,
                                       C.c_size_t(self.ws_bytes), _dp(y), _dp(z), _dp(sr), _dp(self.counters),
                                       C.c_int64(self.max_tracks), _dp(self.trk_nhits), _dp(self.trk_first_hit),
                                       _dp(self.trk_hits), _dp(self.par), _dp(self.cov), _dp(self.xref), _dp(self.zref),
                                       _dp(self.chi2), _dp(self.ndf), _stream()), "tpc_fit_tracks")

    def track_time(self, v_drift: float = 2.58):
        """tpc_track_time (R24) on the last fit: dict(phi0, z0, dca, t0) as numpy fp32 [K]; synchronises."""
        t = self.torch
        K = self.max_tracks
        out = {k: t.empty(K, dtype=t.float32, device=self.device) for k in ("phi0", "z0", "dca", "t0")}
        _check(self.lib.tpc_track_time(C.byref(self.P), _dp(self.counters), C.c_int64(K), _dp(self.trk_sector), _dp(self.par),
                                       _dp(self.xref), _dp(self.zref), C.c_float(v_drift), _dp(out["phi0"]), _dp(out["z0"]),
                                       _dp(out["dca"]), _dp(out["t0"]), _stream()), "tpc_track_time")
        self.trk_t0 = out["t0"]                           # device [max_tracks]: what fit_tracks_physics(trk_t0=...) takes
        k = int(self.counters[CNT_TRACKS].item())
        return {n: v[:k].cpu().numpy() for n, v in out.items()}

    def find_collisions(self, t_lo: float, t_hi: float, v_drift: float = 2.58, bin_width: float = 1.0, dca_max: float = 3.0,
                        n_min: int = 5, max_collisions: int = 1 << 16, side: int = 0):
        """tpc_track_time + tpc_find_collisions (R24, R25) on the last fit; numpy results; synchronises."""
        import math
        t = self.torch
        K = self.max_tracks
        dev = self.device
        tt = {k: t.empty(K, dtype=t.float32, device=dev) for k in ("phi0", "z0", "dca", "t0")}
        _check(self.lib.tpc_track_time(C.byref(self.P), _dp(self.counters), C.c_int64(K), _dp(self.trk_sector), _dp(self.par),
                                       _dp(self.xref), _dp(self.zref), C.c_float(v_drift), _dp(tt["phi0"]), _dp(tt["z0"]),
                                       _dp(tt["dca"]), _dp(tt["t0"]), _stream()), "tpc_track_time")
        self.trk_t0 = tt["t0"]
        nb = int(math.ceil((t_hi - t_lo) / bin_width))
        wsb = C.c_size_t(0)
        _check(self.lib.tpc_collisions_workspace_bytes(C.c_int64(nb), C.c_int64(K), C.byref(wsb)), "tpc_collisions_workspace_bytes")
        ws = t.empty(int(wsb.value), dtype=t.uint8, device=dev)
        ct = t.empty(max_collisions, dtype=t.float32, device=dev)
        cn = t.empty(max_collisions, dtype=t.int32, device=dev)
        cb = t.empty(max_collisions, dtype=t.int32, device=dev)
        tc = t.empty(K, dtype=t.int32, device=dev)
        nc = t.zeros(2, dtype=t.int32, device=dev)
        _check(self.lib.tpc_find_collisions(_dp(self.counters), C.c_int64(K), _dp(tt["t0"]), _dp(tt["dca"]), _dp(self.trk_sector),
                                            C.c_int32(side), C.c_double(t_lo),
                                            C.c_double(bin_width), C.c_int64(nb), C.c_double(dca_max), C.c_int32(n_min), _dp(ws),
                                            C.c_size_t(int(wsb.value)), C.c_int64(max_collisions), _dp(ct), _dp(cn), _dp(cb),
                                            _dp(tc), _dp(nc), _stream()), "tpc_find_collisions")
        k = int(self.counters[CNT_TRACKS].item())
        found, n = (int(v) for v in nc.cpu().numpy())
        self._coll = getattr(self, "_coll", {})
        self._coll[side] = dict(n=nc, time=ct, ntracks=cn, cap=max_collisions)      # device views for pair_sides
        return dict(n_found=found, coll_time=ct[:n].cpu().numpy(), coll_ntracks=cn[:n].cpu().numpy(), coll_bin=cb[:n].cpu().numpy(),
                    trk_collision=tc[:k].cpu().numpy(), t0=tt["t0"][:k].cpu().numpy(), dca=tt["dca"][:k].cpu().numpy())

    def fit_tracks_physics(self, x0inv: float = 0.0, outlier_cut: float = 0.0, dedx: float = 0.0, eloss_sigma: float = 0.0,
                           err_ang_y: float = 0.0, err_ang_z: float = 0.0, err_drift_y: float = 0.0, err_drift_z: float = 0.0,
                           v_drift: float = 0.0, z_len: float = 250.0, trk_t0=None, want_numpy: bool = True,
                           use_workspace: bool = True):
        """tpc_fit_tracks_physics (R28a/b/d/e) on the hit lists of the last find: numpy dict(par, cov, xref, zref, chi2,
        ndf, hit_flag); the Tracker's own fit outputs are left untouched.  trk_t0: device float32 [max_tracks] (the t0 of
        track_time) or None.  use_workspace=False takes the self-contained gather path.  Synchronises unless want_numpy is False (then: the device tensors, enqueue only)."""
        t = self.torch
        K, dev = self.max_tracks, self.device
        y, z, sr = self._inputs
        o = getattr(self, "_physics", None)
        opt = tpc_fit_options_t(x0inv, outlier_cut, dedx, eloss_sigma, err_ang_y, err_ang_z, err_drift_y, err_drift_z, v_drift,
                                z_len)
        if trk_t0 is not None and (trk_t0.dtype != t.float32 or trk_t0.numel() < K or not trk_t0.is_cuda):
            raise ValueError("trk_t0: device float32 [max_tracks]")
        if o is None:
            o = dict(par=t.empty((5, K), dtype=t.float32, device=dev), cov=t.empty((15, K), dtype=t.float32, device=dev),
                     xref=t.empty(K, dtype=t.float32, device=dev), zref=t.empty(K, dtype=t.float32, device=dev),
                     chi2=t.empty(K, dtype=t.float32, device=dev), ndf=t.empty(K, dtype=t.int32, device=dev),
                     hit_flag=t.zeros(max(self.n, 1), dtype=t.uint8, device=dev))
        _check(self.lib.tpc_fit_tracks_physics(C.byref(self.P), C.c_int64(self.n), C.c_int64(self.max_tracklets),
                                               _dp(self.workspace) if use_workspace else C.c_void_p(0), C.c_size_t(self.ws_bytes),
                                               _dp(y), _dp(z), _dp(sr), _dp(self.counters),
                                               C.c_int64(K), _dp(self.trk_nhits), _dp(self.trk_first_hit), _dp(self.trk_hits),
                                               C.byref(opt), _dp(trk_t0), _dp(o["par"]), _dp(o["cov"]),
                                               _dp(o["xref"]), _dp(o["zref"]), _dp(o["chi2"]), _dp(o["ndf"]), _dp(o["hit_flag"]),
                                               _stream()), "tpc_fit_tracks_physics")
        self._physics = o
        if not want_numpy:
            return o
        cnt = self.counters.cpu().numpy()
        k, h = int(cnt[CNT_TRACKS]), int(cnt[CNT_HITS])
        return dict(par=o["par"][:, :k].cpu().numpy(), cov=o["cov"][:, :k].cpu().numpy(), xref=o["xref"][:k].cpu().numpy(),
                    zref=o["zref"][:k].cpu().numpy(), chi2=o["chi2"][:k].cpu().numpy(), ndf=o["ndf"][:k].cpu().numpy(),
                    hit_flag=o["hit_flag"][:h].cpu().numpy())

    def tag_clusters(self, qpt_max: float = 10.0, use_physics_fit: bool = False, want_numpy: bool = True):
        """tpc_tag_clusters (R28c): uint8 tag per cluster, from the Tracker's fit or from the last fit_tracks_physics."""
        t = self.torch
        tag = getattr(self, "_tag", None)
        if tag is None:
            tag = self._tag = t.empty(max(self.n, 1), dtype=t.uint8, device=self.device)
        src = self._physics if use_physics_fit else dict(par=self.par, ndf=self.ndf, hit_flag=None)
        _check(self.lib.tpc_tag_clusters(C.c_int64(self.n), _dp(self.cluster_track), _dp(self.counters), C.c_int64(self.max_tracks),
                                         _dp(src["par"]), _dp(src["ndf"]), _dp(self.trk_hits), _dp(src["hit_flag"]),
                                         C.c_double(qpt_max), _dp(tag), _stream()), "tpc_tag_clusters")
        return tag[:self.n].cpu().numpy() if want_numpy else tag

    def merge_alloc(self):
        """Workspace and device outputs of tpc_merge_tracks (allocated once per Tracker)."""
        if getattr(self, "_merge", None) is not None:
            return self._merge
        t = self.torch
        K, dev = self.max_tracks, self.device
        wsb = C.c_size_t(0)
        _check(self.lib.tpc_merge_workspace_bytes(C.byref(self.P), C.c_int64(K), C.byref(wsb)), "tpc_merge_workspace_bytes")
        i32, f32 = t.int32, t.float32
        o = dict(trk_succ=t.empty(K, dtype=i32, device=dev), trk_pred=t.empty(K, dtype=i32, device=dev),
                 trk_succ_chi2=t.empty(K, dtype=f32, device=dev), trk_global=t.empty(K, dtype=i32, device=dev),
                 n_global=t.zeros(4, dtype=i32, device=dev), g_head=t.empty(K, dtype=i32, device=dev),
                 g_nseg=t.empty(K, dtype=i32, device=dev), g_nhits=t.empty(K, dtype=i32, device=dev),
                 gpar=t.empty((5, K), dtype=f32, device=dev), gcov=t.empty((15, K), dtype=f32, device=dev),
                 gxref=t.empty(K, dtype=f32, device=dev), gzref=t.empty(K, dtype=f32, device=dev),
                 gchi2=t.empty(K, dtype=f32, device=dev), gndf=t.empty(K, dtype=i32, device=dev))
        self._merge = dict(ws=t.empty(int(wsb.value), dtype=t.uint8, device=dev), ws_bytes=int(wsb.value), out=o,
                           out_c=tpc_merged_t(*[C.c_void_p(o[nm].data_ptr()) for nm, _ in tpc_merged_t._fields_]),
                           dev_c=tpc_result_t(*[C.c_void_p(getattr(self, nm).data_ptr()) for nm in RESULT_FIELDS]))
        return self._merge

    def merge_enqueue(self, **mp):
        """tpc_merge_tracks (R26) on the last find + fit; asynchronous."""
        m = self.merge_alloc()
        d = dict(MERGE_DEFAULTS, **mp)
        M = tpc_merge_params_t(float(d["chi2_cut"]), float(d["dz_max"]), float(d["ce_tol"]), int(d["max_rows"]))
        _check(self.lib.tpc_merge_tracks(C.byref(self.P), C.byref(M), C.c_int64(self.n), C.c_int64(self.max_tracklets),
                                         _dp(self.workspace), C.c_size_t(self.ws_bytes), _dp(self.counters),
                                         C.c_int64(self.max_tracks), C.byref(m["dev_c"]), _dp(m["ws"]), C.c_size_t(m["ws_bytes"]),
                                         C.byref(m["out_c"]), _stream()), "tpc_merge_tracks")

    def merge_tracks(self, **mp):
        """merge_enqueue + numpy results (links, global tracks, merged fits); synchronises."""
        self.merge_enqueue(**mp)
        o = self._merge["out"]
        k = int(self.counters[CNT_TRACKS].item())
        m, links, pairs, dropped = (int(v) for v in o["n_global"].cpu().numpy())
        if dropped:
            raise TpcError(f"tpc_merge_tracks: {dropped} of {pairs} candidate pairs did not fit the pair list (4 x max_tracks "
                           f"entries) and were not tested: links are incomplete and depend on arrival order; raise max_tracks")
        per_trk = ("trk_succ", "trk_pred", "trk_succ_chi2", "trk_global")
        res = {nm: o[nm][:k].cpu().numpy() for nm in per_trk}
        res.update({nm: (o[nm][:, :m] if o[nm].dim() == 2 else o[nm][:m]).cpu().numpy()
                    for nm in o if nm not in per_trk and nm != "n_global"})
        res.update(n_global=m, n_links=links, n_pairs=pairs, n_pairs_dropped=dropped)
        return res

    def pair_sides(self, dt_max: float = 15.5, sigma_t: float = 3.88, v_drift: float = 2.58):
        """tpc_pair_sides (R29) on the last find_collisions(side=+1) and find_collisions(side=-1): numpy dict(pair_of_a,
        pair_of_c, t, z_vertex); synchronises."""
        t = self.torch
        a, c = self._coll[1], self._coll[-1]
        cap = min(a["cap"], c["cap"])
        wsb = C.c_size_t(0)
        _check(self.lib.tpc_pair_sides_workspace_bytes(C.c_int64(cap), C.byref(wsb)), "tpc_pair_sides_workspace_bytes")
        ws = t.empty(int(wsb.value), dtype=t.uint8, device=self.device)
        pa = t.empty(cap, dtype=t.int32, device=self.device); pc = t.empty(cap, dtype=t.int32, device=self.device)
        tt = t.empty(cap, dtype=t.float32, device=self.device); zv = t.empty(cap, dtype=t.float32, device=self.device)
        npairs = t.zeros(1, dtype=t.int32, device=self.device)
        _check(self.lib.tpc_pair_sides(_dp(a["n"]), _dp(a["time"]), _dp(a["ntracks"]), _dp(c["n"]), _dp(c["time"]), _dp(c["ntracks"]),
                                       C.c_int64(cap), C.c_double(dt_max), C.c_double(sigma_t), C.c_double(v_drift), _dp(ws),
                                       C.c_size_t(int(wsb.value)), _dp(pa), _dp(pc), _dp(tt), _dp(zv), _dp(npairs), _stream()),
               "tpc_pair_sides")
        k = int(npairs.item())
        na, nc_ = int(a["n"][1].item()), int(c["n"][1].item())
        return dict(pair_of_a=pa[:na].cpu().numpy(), pair_of_c=pc[:nc_].cpu().numpy(), t=tt[:k].cpu().numpy(),
                    z_vertex=zv[:k].cpu().numpy())

    def pair_sides_static(self, dt_max: float = 15.5, sigma_t: float = 3.88, v_drift: float = 2.58):
        """pair_sides through tpc_pair_sides_static: same result, no workspace (see pair_sides_static below)."""
        a, c = self._coll[1], self._coll[-1]
        return pair_sides_static(a["n"], a["time"], a["ntracks"], c["n"], c["time"], c["ntracks"], min(a["cap"], c["cap"]),
                                 dt_max, sigma_t, v_drift)

    def step(self, y, z, sector_row):
        """One pass of the whole hot path (a1..a6) on device-resident inputs; asynchronous."""
        self.grid_build(y, z, sector_row)
        self.find_tracks()
        self.fit_tracks()

    # ---- parity / debug views -----------------------------------------------------------------
    def grid_export(self):
        t = self.torch
        nb = grid_bins(self.params)
        sorted_idx = t.empty(max(self.n, 1), dtype=t.int32, device=self.device)
        bin_first = t.empty(nb + 1, dtype=t.int32, device=self.device)
        _check(self.lib.tpc_grid_export(C.byref(self.P), C.c_int64(self.n), C.c_int64(self.max_tracklets),
                                        _dp(self.workspace), C.c_size_t(self.ws_bytes), _dp(sorted_idx), _dp(bin_first),
                                        _stream()), "tpc_grid_export")
        return sorted_idx[:self.n].cpu().numpy(), bin_first.cpu().numpy()

    def find_export(self, want_row_hit=True):
        t = self.torch
        n1 = max(self.n, 1)
        S = int(self.counters[CNT_TRACKLETS].item())
        mk = lambda m: t.full((max(m, 1),), -1, dtype=t.int32, device=self.device)
        up, dn, upc, dnc = mk(n1), mk(n1), mk(n1), mk(n1)
        starts, nh = mk(self.max_tracklets), mk(self.max_tracklets)
        nrows = int(self.params.n_rows)
        rh = t.full((max(S, 1) * nrows,), -1, dtype=t.int32, device=self.device) if want_row_hit else None
        _check(self.lib.tpc_find_export(C.byref(self.P), C.c_int64(self.n), C.c_int64(self.max_tracklets),
                                        _dp(self.workspace), C.c_size_t(self.ws_bytes), _dp(up), _dp(dn), _dp(upc),
                                        _dp(dnc), _dp(starts), _dp(nh), _dp(rh), _stream()), "tpc_find_export")
        out = dict(link_up=up[:self.n].cpu().numpy(), link_dn=dn[:self.n].cpu().numpy(), up_c=upc[:self.n].cpu().numpy(),
                   dn_c=dnc[:self.n].cpu().numpy(), starts=starts[:S].cpu().numpy(), n_hits=nh[:S].cpu().numpy())
        if want_row_hit:
            out["row_hit"] = rh[:S * nrows].cpu().numpy().reshape(S, nrows)
        return out

    def results(self):
        """Synchronise and copy the outputs of the last step to numpy (original cluster indices)."""
        cnt = self.counters.cpu().numpy()
        K, H = int(cnt[CNT_TRACKS]), int(cnt[CNT_HITS])
        return dict(counters=cnt, status=int(cnt[CNT_STATUS]),
                    cluster_track=self.cluster_track[:self.n].cpu().numpy(),
                    trk_seed=self.trk_seed[:K].cpu().numpy(), trk_sector=self.trk_sector[:K].cpu().numpy(),
                    trk_nhits=self.trk_nhits[:K].cpu().numpy(), trk_first_hit=self.trk_first_hit[:K].cpu().numpy(),
                    trk_hits=self.trk_hits[:H].cpu().numpy(), par=self.par[:, :K].cpu().numpy(),
                    cov=self.cov[:, :K].cpu().numpy(), xref=self.xref[:K].cpu().numpy(), zref=self.zref[:K].cpu().numpy(),
                    chi2=self.chi2[:K].cpu().numpy(), ndf=self.ndf[:K].cpu().numpy())

    def run(self, y, z, sector_row):
        self.step(y, z, sector_row)
        return self.results()

    # ---- host-buffer path (bench.py e2e) ------------------------------------------------------
    def make_host_staging(self):
        """Device staging buffers for the inputs + pinned host buffers for every output (`track_host`)."""
        t = self.torch
        n1 = max(self.n, 1)
        self._y_dev = t.empty(n1, dtype=t.float32, device=self.device)
        self._z_dev = t.empty(n1, dtype=t.float32, device=self.device)
        self._sr_dev = t.empty(n1, dtype=t.int32, device=self.device)
        self.host = {nm: t.empty_like(getattr(self, nm), device="cpu").pin_memory() for nm in RESULT_FIELDS}
        self.host["counters"].zero_()
        self.counters_host = self.host["counters"]
        self._res_dev = tpc_result_t(*[C.c_void_p(getattr(self, nm).data_ptr()) for nm in RESULT_FIELDS])
        self._res_host = tpc_result_t(*[C.c_void_p(self.host[nm].data_ptr()) for nm in RESULT_FIELDS])

    def _host_args(self, y_host, z_host, sr_host):
        for a in (y_host, z_host, sr_host):
            assert not a.is_cuda and a.is_contiguous() and a.numel() == self.n
        hp = lambda a: C.c_void_p(a.data_ptr())
        self._inputs = (self._y_dev, self._z_dev, self._sr_dev)
        return (C.byref(self.P), C.c_int64(self.n), C.c_int64(self.max_tracklets), C.c_int64(self.max_tracks),
                hp(y_host), hp(z_host), hp(sr_host), _dp(self._y_dev), _dp(self._z_dev), _dp(self._sr_dev),
                _dp(self.workspace), C.c_size_t(self.ws_bytes), C.byref(self._res_dev), C.byref(self._res_host), _stream())

    def track_host(self, y_host, z_host, sr_host):
        """tpc_track_host: H2D of the inputs, a1..a6, D2H of every output; synchronous.  Returns (h2d, d2h) bytes."""
        _check(self.lib.tpc_track_host(*self._host_args(y_host, z_host, sr_host)), "tpc_track_host")
        return 12 * self.n, self.d2h_bytes()

    def track_host_async(self, y_host, z_host, sr_host):
        """tpc_track_host_async on the current stream: H2D, a1..a6, D2H of counters + cluster_track; enqueue only."""
        _check(self.lib.tpc_track_host_async(*self._host_args(y_host, z_host, sr_host)), "tpc_track_host_async")

    def track_host_fetch(self) -> int:
        """tpc_track_host_fetch on the current stream (the counters must have arrived): D2H of exactly K tracks and H
        hits of every other output.  Returns the bytes enqueued."""
        nb = C.c_int64(0)
        _check(self.lib.tpc_track_host_fetch(C.c_int64(self.max_tracks), C.byref(self._res_dev), C.byref(self._res_host),
                                             C.byref(nb), _stream()), "tpc_track_host_fetch")
        return int(nb.value)

    def d2h_bytes(self) -> int:
        """Bytes one host-buffer step copies device->host, from the counters of the last completed step."""
        K, H = int(self.counters_host[CNT_TRACKS]), int(self.counters_host[CNT_HITS])
        return 4 * TPC_N_COUNTERS + 4 * self.n + K * (4 * 3 + 8 + 4 * (5 + 15) + 4 * 4) + 4 * H

    def host_results(self):
        """numpy views of the pinned host buffers after a completed host-buffer step (same keys as results())."""
        cnt = self.host["counters"].numpy()
        K, H = int(cnt[CNT_TRACKS]), int(cnt[CNT_HITS])
        h = {k: v.numpy() for k, v in self.host.items()}
        return dict(counters=cnt, status=int(cnt[CNT_STATUS]), cluster_track=h["cluster_track"][:self.n],
                    trk_seed=h["trk_seed"][:K], trk_sector=h["trk_sector"][:K], trk_nhits=h["trk_nhits"][:K],
                    trk_first_hit=h["trk_first_hit"][:K], trk_hits=h["trk_hits"][:H], par=h["par"][:, :K], cov=h["cov"][:, :K],
                    xref=h["xref"][:K], zref=h["zref"][:K], chi2=h["chi2"][:K], ndf=h["ndf"][:K])
