"""ctypes front end of the CPU ORACLE (oracle/tpc_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Nothing under paper_2106_03636_b200/ imports it and it
imports nothing from there (parameters arrive as any object with the TpcParams attribute names;
clusters as numpy arrays).

`build()` compiles the oracle with g++ (-O2 -ffp-contract=off: one IEEE operation per written
operation -- the fused multiply-adds of the arithmetic contract are explicit std::fma calls -- which is
what makes float mode comparable with the GPU; -mfma only turns those calls into the instruction).  `run()` chains the stages
R7 -> R9 -> R10 -> R14-R18 -> R20 -> R21-R22 and returns every intermediate
so the parity tests can compare stage by stage.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
import time

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpc_oracle.cpp")
_LIB = os.path.join(_HERE, "libtpc_oracle.so")
_lib = None

N_ROWS_MAX = 152


class OrcParams(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("row_x", C.c_double * N_ROWS_MAX),
                ("tan_half", C.c_double), ("kB", C.c_double), ("sigma_y", C.c_double), ("sigma_z", C.c_double),
                ("z_lo", C.c_double), ("z_hi", C.c_double), ("cell_y", C.c_double), ("cell_z", C.c_double),
                ("ca_max_dydx", C.c_double), ("ca_max_dzdx", C.c_double), ("ca_cut", C.c_double),
                ("chi2_cut", C.c_double), ("chi2_chain_cut", C.c_double), ("win_max", C.c_double),
                ("max_sinphi", C.c_double), ("edge_margin", C.c_double),
                ("max_gap", C.c_int32), ("min_hits", C.c_int32), ("n_fit_passes", C.c_int32), ("reserved", C.c_int32),
                ("cov0", C.c_double * 5)]


class TraceRec(C.Structure):
    _fields_ = [("tracklet", C.c_int32), ("row", C.c_int32), ("chosen", C.c_int32), ("pad", C.c_int32),
                ("y_pred", C.c_double), ("dz_pred", C.c_double), ("zref", C.c_double),
                ("S00", C.c_double), ("S01", C.c_double), ("S11", C.c_double), ("chi2", C.c_double)]


DECISION_DTYPE = np.dtype([("tracklet", "i4"), ("row", "i4"), ("kind", "i4"), ("chosen", "i4"), ("best", "f8"),
                           ("second", "f8"), ("cut", "f8")])
DEC_SEARCH, DEC_CHAIN, DEC_SINPHI, DEC_EDGE = 0, 1, 2, 3

TRACE_DTYPE = np.dtype([("tracklet", "i4"), ("row", "i4"), ("chosen", "i4"), ("pad", "i4"), ("y_pred", "f8"),
                        ("dz_pred", "f8"), ("zref", "f8"), ("S00", "f8"), ("S01", "f8"), ("S11", "f8"), ("chi2", "f8")])


def build(force: bool = False) -> str:
    """Compile oracle/tpc_oracle.cpp -> oracle/libtpc_oracle.so (no-op if up to date)."""
    if (not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + f".tmp{os.getpid()}"
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-fvisibility=hidden", "-o", tmp, _SRC]
    if _cpu_has_fma():
        cmd.insert(1, "-mfma")      # std::fma -> vfmadd instead of a libm call; same (correctly rounded) result
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def _cpu_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return " fma " in line + " "
    except OSError:
        pass
    return False


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_sizeof_params.restype = C.c_int64
        L.orc_sizeof_trace.restype = C.c_int64
        assert L.orc_sizeof_params() == C.sizeof(OrcParams), "OrcParams layout mismatch"
        assert L.orc_sizeof_trace() == C.sizeof(TraceRec) == TRACE_DTYPE.itemsize, "TraceRec layout mismatch"
        for sfx in ("f32", "f64"):
            getattr(L, f"orc_grid_{sfx}").restype = C.c_int64
            getattr(L, f"orc_follow_{sfx}").restype = C.c_int64
            getattr(L, f"orc_neighbours_{sfx}").restype = None
            getattr(L, f"orc_fit_{sfx}").restype = None
            getattr(L, f"orc_propagate_{sfx}").restype = C.c_int
        L.orc_update_f32.restype = C.c_float
        L.orc_update_f64.restype = C.c_double
        L.orc_links.restype = C.c_int64
        L.orc_beamline.restype = None
        L.orc_select.restype = C.c_int64
        L.orc_sizeof_decision.restype = C.c_int64
        assert L.orc_sizeof_decision() == DECISION_DTYPE.itemsize, "DecRec layout mismatch"
        L.orc_set_arith.restype = None
        L.orc_get_arith.restype = C.c_int
        L.orc_decisions_begin.restype = None
        L.orc_decisions_end.restype = C.c_int64
        _lib = L
    return _lib


class arith:
    """with arith(fused=False): ...  -- evaluate every mad(a,b,c) of R12/R13 as a*b then +c (two roundings) instead
    of the fused multiply-add of the arithmetic contract.  Process-global, restored on exit."""

    def __init__(self, fused: bool):
        self.fused = bool(fused)

    def __enter__(self):
        self.prev = lib().orc_get_arith()
        lib().orc_set_arith(C.c_int(int(self.fused)))
        return self

    def __exit__(self, *exc):
        lib().orc_set_arith(C.c_int(self.prev))
        return False


class decisions:
    """with decisions(cap) as d: orc.follow(...) / orc.run(...);  d.log = every decision the follower took
    (DECISION_DTYPE records, in the order taken; d.dropped = decisions beyond cap)."""

    def __init__(self, cap: int):
        self.buf = np.zeros(int(cap), DECISION_DTYPE)
        self.log = self.buf[:0]
        self.dropped = 0

    def __enter__(self):
        lib().orc_decisions_begin(_ptr(self.buf), C.c_int64(self.buf.size))
        return self

    def __exit__(self, *exc):
        n = int(lib().orc_decisions_end())
        self.log = self.buf[:min(n, self.buf.size)]
        self.dropped = max(0, n - self.buf.size)
        return False


def make_params(p, precision: str = "f32") -> OrcParams:
    """Marshal a TpcParams-like object.  In f32 mode every real is first rounded to float32."""
    rnd = (lambda v: float(np.float32(v))) if precision == "f32" else float
    P = OrcParams()
    P.n_sectors, P.n_rows = int(p.n_sectors), int(p.n_rows)
    rx = np.asarray(p.row_x, dtype=np.float64)
    for i in range(P.n_rows):
        P.row_x[i] = rnd(rx[i])
    for name in ("tan_half", "kB", "sigma_y", "sigma_z", "z_lo", "z_hi", "cell_y", "cell_z", "ca_max_dydx",
                 "ca_max_dzdx", "ca_cut", "chi2_cut", "chi2_chain_cut", "win_max", "max_sinphi", "edge_margin"):
        setattr(P, name, rnd(getattr(p, name)))
    P.max_gap, P.min_hits, P.n_fit_passes = int(p.max_gap), int(p.min_hits), int(p.n_fit_passes)
    for i in range(5):
        P.cov0[i] = rnd(p.cov0[i])
    return P


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _real(precision):
    return (np.float32, "f32") if precision == "f32" else (np.float64, "f64")


def n_bins(p, precision="f32") -> int:
    P = make_params(p, precision)
    e = np.zeros(0, _real(precision)[0]); s = np.zeros(0, np.int32)
    return int(getattr(lib(), f"orc_grid_{_real(precision)[1]}")(C.byref(P), C.c_int64(0), _ptr(e), _ptr(e), _ptr(s),
                                                                   None, None, C.c_int64(0)))


def grid(p, y, z, sector_row, precision="f32"):
    """R7: returns (sorted_idx[n], bin_first[n_bins+1])."""
    rt, sfx = _real(precision)
    P = make_params(p, precision)
    y = np.ascontiguousarray(y, rt); z = np.ascontiguousarray(z, rt); sr = np.ascontiguousarray(sector_row, np.int32)
    nb = n_bins(p, precision)
    sorted_idx = np.empty(y.size, np.int32); bin_first = np.empty(nb + 1, np.int32)
    getattr(lib(), f"orc_grid_{sfx}")(C.byref(P), C.c_int64(y.size), _ptr(y), _ptr(z), _ptr(sr), _ptr(sorted_idx),
                                      _ptr(bin_first), C.c_int64(nb + 1))
    return sorted_idx, bin_first


def neighbours(p, y, z, sector_row, precision="f32", use_grid=True):
    """R9: returns (link_up[n], link_dn[n]) in original indices, -1 = none."""
    rt, sfx = _real(precision)
    P = make_params(p, precision)
    y = np.ascontiguousarray(y, rt); z = np.ascontiguousarray(z, rt); sr = np.ascontiguousarray(sector_row, np.int32)
    up = np.empty(y.size, np.int32); dn = np.empty(y.size, np.int32)
    getattr(lib(), f"orc_neighbours_{sfx}")(C.byref(P), C.c_int64(y.size), _ptr(y), _ptr(z), _ptr(sr),
                                            C.c_int(int(use_grid)), _ptr(up), _ptr(dn))
    return up, dn


def links(link_up, link_dn):
    """R10: returns (up_c, dn_c, starts)."""
    n = link_up.size
    up_c = np.empty(n, np.int32); dn_c = np.empty(n, np.int32); starts = np.empty(n, np.int32)
    ns = lib().orc_links(C.c_int64(n), _ptr(np.ascontiguousarray(link_up, np.int32)),
                         _ptr(np.ascontiguousarray(link_dn, np.int32)), _ptr(up_c), _ptr(dn_c), _ptr(starts))
    return up_c, dn_c, starts[:ns].copy()


R17_NAIVE, R17_PHASES, R17_WAVES = 0, 1, 2


def wave_test(p, y, z, sector_row, up_c, starts, precision="f32", use_grid=True):
    """R17 (i): waits[S] (bool) -- does start hit t have a plausible predecessor below it?"""
    rt, sfx = _real(precision)
    P = make_params(p, precision)
    y = np.ascontiguousarray(y, rt); z = np.ascontiguousarray(z, rt); sr = np.ascontiguousarray(sector_row, np.int32)
    starts = np.ascontiguousarray(starts, np.int32); up_c = np.ascontiguousarray(up_c, np.int32)
    waits = np.zeros(starts.size, np.uint8)
    fn = getattr(lib(), f"orc_wave_test_{sfx}")
    fn.restype = None
    fn(C.byref(P), C.c_int64(y.size), _ptr(y), _ptr(z), _ptr(sr), C.c_int(int(use_grid)), _ptr(up_c),
       C.c_int64(starts.size), _ptr(starts), _ptr(waits))
    return waits.astype(bool)


def follow(p, y, z, sector_row, up_c, starts, precision="f32", use_grid=True, want_state=False, trace_cap=0,
           r17_mode=R17_WAVES):
    """R14-R18: returns dict(row_hit[S, n_rows], n_hits[S], ran[S], state[S,21]?, trace?).
    r17_mode: 0 = every start hit followed in full, 1 = phases, 2 = phases + waves (R17; the default)."""
    rt, sfx = _real(precision)
    P = make_params(p, precision)
    y = np.ascontiguousarray(y, rt); z = np.ascontiguousarray(z, rt); sr = np.ascontiguousarray(sector_row, np.int32)
    starts = np.ascontiguousarray(starts, np.int32); up_c = np.ascontiguousarray(up_c, np.int32)
    S = starts.size
    row_hit = np.empty((S, P.n_rows), np.int32); n_hits = np.empty(S, np.int32)
    state = np.empty((S, 21), rt) if want_state else None
    trace = np.zeros(trace_cap, TRACE_DTYPE) if trace_cap else None
    ran = np.zeros(S, np.uint8)
    nt = getattr(lib(), f"orc_follow_{sfx}")(C.byref(P), C.c_int64(y.size), _ptr(y), _ptr(z), _ptr(sr),
                                             C.c_int(int(use_grid)), _ptr(up_c), C.c_int64(S), _ptr(starts),
                                             _ptr(row_hit), _ptr(n_hits), _ptr(state), _ptr(trace), C.c_int64(trace_cap),
                                             C.c_int(int(r17_mode)), _ptr(ran))
    out = dict(row_hit=row_hit, n_hits=n_hits, ran=ran.astype(bool))
    if want_state:
        out["state"] = state
    if trace_cap:
        out["trace"] = trace[:nt]
    return out


def select(n, n_rows, starts, row_hit, n_hits, min_hits):
    """R20: returns dict(cluster_track[n], trk_seed, trk_nhits, trk_first_hit, trk_hits)."""
    starts = np.ascontiguousarray(starts, np.int32); row_hit = np.ascontiguousarray(row_hit, np.int32)
    n_hits = np.ascontiguousarray(n_hits, np.int32)
    S = starts.size
    cluster_track = np.empty(n, np.int32)
    trk_seed = np.empty(S, np.int32); trk_nhits = np.empty(S, np.int32); trk_first = np.empty(S, np.int64)
    trk_hits = np.empty(max(n, 1), np.int32)
    K = lib().orc_select(C.c_int64(n), C.c_int(n_rows), C.c_int64(S), _ptr(starts), _ptr(row_hit), _ptr(n_hits),
                         C.c_int(int(min_hits)), _ptr(cluster_track), _ptr(trk_seed), _ptr(trk_nhits), _ptr(trk_first),
                         _ptr(trk_hits))
    nh = int(trk_nhits[:K].sum())
    return dict(cluster_track=cluster_track, trk_seed=trk_seed[:K].copy(), trk_nhits=trk_nhits[:K].copy(),
                trk_first_hit=trk_first[:K].copy(), trk_hits=trk_hits[:nh].copy())


def fit(p, y, z, sector_row, trk_nhits, trk_first_hit, trk_hits, precision="f32"):
    """R21-R22: returns dict(par[5,K], cov[15,K], xref, zref, chi2, ndf)."""
    rt, sfx = _real(precision)
    P = make_params(p, precision)
    y = np.ascontiguousarray(y, rt); z = np.ascontiguousarray(z, rt); sr = np.ascontiguousarray(sector_row, np.int32)
    nh = np.ascontiguousarray(trk_nhits, np.int32); fh = np.ascontiguousarray(trk_first_hit, np.int64)
    th = np.ascontiguousarray(trk_hits, np.int32)
    K = nh.size
    par = np.empty((5, K), rt); cov = np.empty((15, K), rt)
    xref = np.empty(K, rt); zref = np.empty(K, rt); chi2 = np.empty(K, rt); ndf = np.empty(K, np.int32)
    getattr(lib(), f"orc_fit_{sfx}")(C.byref(P), C.c_int64(y.size), _ptr(y), _ptr(z), _ptr(sr), C.c_int64(K), _ptr(nh),
                                     _ptr(fh), _ptr(th), _ptr(par), _ptr(cov), _ptr(xref), _ptr(zref), _ptr(chi2),
                                     _ptr(ndf))
    return dict(par=par, cov=cov, xref=xref, zref=zref, chi2=chi2, ndf=ndf)


def beamline(p, par, xref, zref, sector, v_drift=2.58):
    """R24: closest approach to the beam line of fp32 track states par[5,K] at xref: dict(phi0, z0, dca, t0) (fp32)."""
    P = make_params(p, "f32")          # the tracker's fp32-rounded field constant
    par = np.ascontiguousarray(par, np.float32)
    K = par.shape[1]
    xref = np.ascontiguousarray(xref, np.float32); zref = np.ascontiguousarray(zref, np.float32)
    sector = np.ascontiguousarray(sector, np.int32)
    out = {k: np.empty(K, np.float32) for k in ("phi0", "z0", "dca", "t0")}
    lib().orc_beamline(C.byref(P), C.c_int64(K), _ptr(par), C.c_int64(K), _ptr(xref), _ptr(zref), _ptr(sector),
                       C.c_double(v_drift), _ptr(out["phi0"]), _ptr(out["z0"]), _ptr(out["dca"]), _ptr(out["t0"]))
    return out


def collisions(t0, dca, t_lo, t_hi, w=1.0, dca_max=3.0, n_min=5, sector=None, side=0):
    """R25: dict(coll_time, coll_ntracks, coll_bin, trk_collision) from per-track t0 / dca (R24)."""
    t0 = np.ascontiguousarray(t0, np.float32); dca = np.ascontiguousarray(dca, np.float32)
    K = t0.size
    sector = np.zeros(K, np.int32) if sector is None else np.ascontiguousarray(sector, np.int32)
    nb = int(math.ceil((t_hi - t_lo) / w))
    ct = np.empty(max(nb, 1), np.float32); cn = np.empty(max(nb, 1), np.int32); cb = np.empty(max(nb, 1), np.int32)
    tc = np.empty(max(K, 1), np.int32)
    L = lib()
    L.orc_collisions.restype = C.c_int64
    n = L.orc_collisions(C.c_int64(K), _ptr(t0), _ptr(dca), _ptr(sector), C.c_int32(side), C.c_double(t_lo), C.c_double(w), C.c_int64(nb),
                         C.c_double(dca_max), C.c_int32(n_min), C.c_int64(ct.size), _ptr(ct), _ptr(cn), _ptr(cb), _ptr(tc))
    n = int(n)
    return dict(coll_time=ct[:n], coll_ntracks=cn[:n], coll_bin=cb[:n], trk_collision=tc[:K])


class OrcMergeParams(C.Structure):
    _fields_ = [("chi2_cut", C.c_double), ("dz_max", C.c_double), ("ce_tol", C.c_double), ("max_rows", C.c_int32),
                ("reserved", C.c_int32)]


#: R26 defaults: chi2 cut over 5 (4 across the electrode) parameters, largest row distance between the
#: two ends, z window between the ends [cm], tolerance of the electrode-crossing condition [cm]
MERGE_DEFAULTS = dict(chi2_cut=50.0, dz_max=64.0, ce_tol=1.0, max_rows=12)


def make_merge_params(mp=None, precision="f32") -> OrcMergeParams:
    d = dict(MERGE_DEFAULTS)
    if mp:
        d.update(mp if isinstance(mp, dict) else {k: getattr(mp, k) for k in MERGE_DEFAULTS})
    rnd = (lambda v: float(np.float32(v))) if precision == "f32" else float
    M = OrcMergeParams()
    M.chi2_cut, M.dz_max, M.ce_tol, M.max_rows = rnd(d["chi2_cut"]), rnd(d["dz_max"]), rnd(d["ce_tol"]), int(d["max_rows"])
    assert lib().orc_sizeof_merge_params() == C.sizeof(OrcMergeParams)
    return M


def track_rows(n_rows, sector_row, trk_nhits, trk_first_hit, trk_hits):
    """(sector, first row, last row) of every track from its hit list (rows ascend along a list)."""
    sr = np.asarray(sector_row)
    fh = np.asarray(trk_first_hit, np.int64); nh = np.asarray(trk_nhits, np.int64)
    if fh.size == 0:
        z = np.zeros(0, np.int32)
        return z, z, z
    first = sr[np.asarray(trk_hits)[fh]]
    last = sr[np.asarray(trk_hits)[fh + nh - 1]]
    return (first // n_rows).astype(np.int32), (first % n_rows).astype(np.int32), (last % n_rows).astype(np.int32)


def merge_match(p, par, cov, zref, sector, row_first, row_last, seed, mp=None, precision="f32", want_pairs=False):
    """R26 matching: dict(succ[K], pred[K] (track index or -1, reciprocal links only), succ_chi2[K] (chi2 of the best
    candidate successor, -1 = none), pair_chi2[K,K]? (chi2 of "b follows a", -1 = impossible))."""
    rt, sfx = _real(precision)
    P = make_params(p, precision); M = make_merge_params(mp, precision)
    par = np.ascontiguousarray(par, rt); cov = np.ascontiguousarray(cov, rt); zref = np.ascontiguousarray(zref, rt)
    K = par.shape[1]
    i32 = lambda a: np.ascontiguousarray(a, np.int32)
    sector, row_first, row_last, seed = i32(sector), i32(row_first), i32(row_last), i32(seed)
    succ = np.empty(K, np.int32); pred = np.empty(K, np.int32); sc = np.empty(K, rt)
    pairs = np.empty((K, K), rt) if want_pairs else None
    fn = getattr(lib(), f"orc_merge_match_{sfx}")
    fn.restype = None
    fn(C.byref(P), C.byref(M), C.c_int64(K), _ptr(par), _ptr(cov), _ptr(zref), _ptr(sector), _ptr(row_first), _ptr(row_last),
       _ptr(seed), _ptr(succ), _ptr(pred), _ptr(sc), _ptr(pairs))
    out = dict(succ=succ, pred=pred, succ_chi2=sc)
    if want_pairs:
        out["pair_chi2"] = pairs
    return out


def merge_fit(p, y, z, sector_row, fit, sector, trk_nhits, trk_first_hit, trk_hits, succ, pred, precision="f32"):
    """R26 refit of the chains: dict(trk_global[K], g_head[M], g_nseg, g_nhits, gpar[5,M], gcov[15,M], gxref, gzref,
    gchi2, gndf).  `fit` = the dict orc.fit returned for the sector-local tracks."""
    rt, sfx = _real(precision)
    P = make_params(p, precision)
    y = np.ascontiguousarray(y, rt); z = np.ascontiguousarray(z, rt); sr = np.ascontiguousarray(sector_row, np.int32)
    c = lambda a: np.ascontiguousarray(a, rt)
    i32 = lambda a: np.ascontiguousarray(a, np.int32)
    K = int(np.asarray(succ).size)
    pred = i32(pred); succ = i32(succ)
    Mg = int(np.count_nonzero(pred < 0))
    tg = np.empty(K, np.int32); gh = np.empty(Mg, np.int32); gs = np.empty(Mg, np.int32); gn = np.empty(Mg, np.int32)
    gpar = np.empty((5, Mg), rt); gcov = np.empty((15, Mg), rt)
    gx = np.empty(Mg, rt); gz = np.empty(Mg, rt); gc = np.empty(Mg, rt); gndf = np.empty(Mg, np.int32)
    fn = getattr(lib(), f"orc_merge_fit_{sfx}")
    fn.restype = C.c_int64
    par, cov, xref, zref, chi2 = c(fit["par"]), c(fit["cov"]), c(fit["xref"]), c(fit["zref"]), c(fit["chi2"])
    ndf = i32(fit["ndf"]); sector = i32(sector); nh = i32(trk_nhits); th = i32(trk_hits)
    fh = np.ascontiguousarray(trk_first_hit, np.int64)
    m = fn(C.byref(P), C.c_int64(y.size), _ptr(y), _ptr(z), _ptr(sr), C.c_int64(K), _ptr(par), _ptr(cov), _ptr(xref), _ptr(zref),
           _ptr(chi2), _ptr(ndf), _ptr(sector), _ptr(nh), _ptr(fh), _ptr(th), _ptr(succ), _ptr(pred), _ptr(tg), _ptr(gh), _ptr(gs),
           _ptr(gn), _ptr(gpar), _ptr(gcov), _ptr(gx), _ptr(gz), _ptr(gc), _ptr(gndf))
    assert int(m) == Mg
    return dict(trk_global=tg, g_head=gh, g_nseg=gs, g_nhits=gn, gpar=gpar, gcov=gcov, gxref=gx, gzref=gz, gchi2=gc, gndf=gndf)


def merge(p, y, z, sector_row, o, mp=None, precision="f32", want_pairs=False):
    """R26 on the output `o` of run(): matching + refit of the chains.  Returns the two dicts merged, plus the
    per-track (sector, row_first, row_last) it derived from the hit lists."""
    if int(p.n_fit_passes) % 2 != 0:
        raise ValueError("R26 takes every fitted state at the track's innermost hit: n_fit_passes must be even")
    sector, rf, rl = track_rows(int(p.n_rows), sector_row, o["trk_nhits"], o["trk_first_hit"], o["trk_hits"])
    m = merge_match(p, o["par"], o["cov"], o["zref"], sector, rf, rl, o["trk_seed"], mp, precision, want_pairs)
    f = merge_fit(p, y, z, sector_row, o, sector, o["trk_nhits"], o["trk_first_hit"], o["trk_hits"], m["succ"], m["pred"],
                  precision)
    return dict(trk_sector=sector, row_first=rf, row_last=rl, **m, **f)


class OrcFitOptions(C.Structure):
    _fields_ = [(nm, C.c_double) for nm in ("x0inv", "outlier_cut", "dedx", "eloss_sigma", "err_ang_y", "err_ang_z",
                                            "err_drift_y", "err_drift_z", "v_drift", "z_len")]


def fit_physics(p, y, z, sector_row, trk_nhits, trk_first_hit, trk_hits, x0inv=0.0, outlier_cut=0.0, precision="f32",
                dedx=0.0, eloss_sigma=0.0, err_ang_y=0.0, err_ang_z=0.0, err_drift_y=0.0, err_drift_z=0.0, v_drift=0.0,
                z_len=250.0, trk_t0=None):
    """R21-R22 with the R28 options (a: scattering noise per unit path, b: outlier rejection in the last pass, d: mean
    energy loss, e: angle- and drift-dependent cluster errors; trk_t0 = R24's time offsets for the drift length):
    dict(par, cov, xref, zref, chi2, ndf, hit_flag[n_hits])."""
    rt, sfx = _real(precision)
    P = make_params(p, precision)
    rnd = (lambda v: float(np.float32(v))) if precision == "f32" else float
    O = OrcFitOptions(*[rnd(v) for v in (x0inv, outlier_cut, dedx, eloss_sigma, err_ang_y, err_ang_z, err_drift_y, err_drift_z,
                                         v_drift, z_len)])
    t0 = None if trk_t0 is None else np.ascontiguousarray(trk_t0, rt)
    y = np.ascontiguousarray(y, rt); z = np.ascontiguousarray(z, rt); sr = np.ascontiguousarray(sector_row, np.int32)
    nh = np.ascontiguousarray(trk_nhits, np.int32); fh = np.ascontiguousarray(trk_first_hit, np.int64)
    th = np.ascontiguousarray(trk_hits, np.int32)
    K = nh.size
    par = np.empty((5, K), rt); cov = np.empty((15, K), rt)
    xref = np.empty(K, rt); zref = np.empty(K, rt); chi2 = np.empty(K, rt); ndf = np.empty(K, np.int32)
    flag = np.zeros(max(th.size, 1), np.uint8)
    fn = getattr(lib(), f"orc_fit_physics_{sfx}")
    fn.restype = None
    fn(C.byref(P), C.byref(O), C.c_int64(y.size), _ptr(y), _ptr(z), _ptr(sr), C.c_int64(K), _ptr(nh), _ptr(fh), _ptr(th), _ptr(t0),
       _ptr(par), _ptr(cov), _ptr(xref), _ptr(zref), _ptr(chi2), _ptr(ndf), _ptr(flag))
    return dict(par=par, cov=cov, xref=xref, zref=zref, chi2=chi2, ndf=ndf, hit_flag=flag[:th.size])


def tag_clusters(cluster_track, qpt, ndf, trk_nhits, trk_first_hit, trk_hits, hit_flag=None, qpt_max=10.0):
    """R28c: uint8 tag per cluster (bit 0 attached, bit 1 track not used for physics, bit 2 rejected hit)."""
    ct = np.ascontiguousarray(cluster_track, np.int32)
    qpt = np.ascontiguousarray(qpt, np.float32); ndf = np.ascontiguousarray(ndf, np.int32)
    nh = np.ascontiguousarray(trk_nhits, np.int32); fh = np.ascontiguousarray(trk_first_hit, np.int64)
    th = np.ascontiguousarray(trk_hits, np.int32)
    hf = None if hit_flag is None else np.ascontiguousarray(hit_flag, np.uint8)
    tag = np.empty(ct.size, np.uint8)
    fn = lib().orc_tag_clusters
    fn.restype = None
    fn(C.c_int64(ct.size), _ptr(ct), C.c_int64(nh.size), _ptr(qpt), _ptr(ndf), _ptr(nh), _ptr(fh), _ptr(th), _ptr(hf),
       C.c_double(qpt_max), _ptr(tag))
    return tag


def clusterize(p, sector_row, pad, time, adc, pad_width, time_width, peak_min=6, cap=None):
    """R27: clusters from digits: dict(y, z, q (fp32), sector_row, pad, time (peak cell)), ascending (sector_row, time, pad)."""
    P = make_params(p, "f32")
    i32 = lambda a: np.ascontiguousarray(a, np.int32)
    sr, pad, time, adc = i32(sector_row), i32(pad), i32(time), i32(adc)
    n = sr.size
    cap = int(cap if cap is not None else max(n, 1))
    out = dict(y=np.empty(cap, np.float32), z=np.empty(cap, np.float32), q=np.empty(cap, np.float32),
               sector_row=np.empty(cap, np.int32), pad=np.empty(cap, np.int32), time=np.empty(cap, np.int32))
    L = lib()
    L.orc_clusterize.restype = C.c_int64
    k = int(L.orc_clusterize(C.byref(P), C.c_int64(n), _ptr(sr), _ptr(pad), _ptr(time), _ptr(adc), C.c_double(pad_width),
                             C.c_double(time_width), C.c_int32(int(peak_min)), C.c_int64(cap), _ptr(out["y"]), _ptr(out["z"]),
                             _ptr(out["q"]), _ptr(out["sector_row"]), _ptr(out["pad"]), _ptr(out["time"])))
    out = {a: b[:min(k, cap)].copy() for a, b in out.items()}
    out["n_found"] = k
    return out


def pair_sides(tA, nA, tC, nC, dt_max=15.5, sigma_t=3.88, v_drift=2.58):
    """R29: dict(pair_of_a[nA], pair_of_c[nC], t[np], z_vertex[np]) from the per-side collision times / track counts."""
    tA = np.ascontiguousarray(tA, np.float32); tC = np.ascontiguousarray(tC, np.float32)
    nA = np.ascontiguousarray(nA, np.int32); nC = np.ascontiguousarray(nC, np.int32)
    pa = np.empty(max(tA.size, 1), np.int32); pc = np.empty(max(tC.size, 1), np.int32)
    t = np.empty(max(min(tA.size, tC.size), 1), np.float32); zv = np.empty_like(t)
    fn = lib().orc_pair_sides
    fn.restype = C.c_int64
    k = int(fn(C.c_int64(tA.size), _ptr(tA), _ptr(nA), C.c_int64(tC.size), _ptr(tC), _ptr(nC), C.c_double(dt_max),
               C.c_double(sigma_t), C.c_double(v_drift), _ptr(pa), _ptr(pc), _ptr(t), _ptr(zv)))
    return dict(pair_of_a=pa[:tA.size], pair_of_c=pc[:tC.size], t=t[:k], z_vertex=zv[:k])


def propagate(p, par5, cov15, dx, precision="f64"):
    """R12 primitive: returns (ok, par5', cov15', F[5,5])."""
    rt, sfx = _real(precision)
    P = make_params(p, precision)
    a = np.array(par5, rt); c = np.array(cov15, rt); F = np.zeros(25, rt)
    ct = C.c_float if sfx == "f32" else C.c_double
    ok = getattr(lib(), f"orc_propagate_{sfx}")(C.byref(P), _ptr(a), _ptr(c), ct(dx), _ptr(F))
    return bool(ok), a, c, F.reshape(5, 5)


def rotate(p, par5, cov15, x, delta, precision="f64"):
    """R26 rotation primitive: the state (par5, cov15) at x, expressed in the frame turned by `delta` rad.
    Returns (ok, par5', cov15', x')."""
    rt, sfx = _real(precision)
    P = make_params(p, precision)
    a = np.array(par5, rt); c = np.array(cov15, rt)
    ct = C.c_float if sfx == "f32" else C.c_double
    xx = ct(float(x))
    ok = getattr(lib(), f"orc_rotate_{sfx}")(C.byref(P), _ptr(a), _ptr(c), C.byref(xx), ct(math.cos(delta)), ct(math.sin(delta)))
    return bool(ok), a, c, float(xx.value)


def update(p, par5, cov15, ym, zm, precision="f64"):
    """R13 primitive: returns (chi2, par5', cov15')."""
    rt, sfx = _real(precision)
    P = make_params(p, precision)
    a = np.array(par5, rt); c = np.array(cov15, rt)
    ct = C.c_float if sfx == "f32" else C.c_double
    chi2 = getattr(lib(), f"orc_update_{sfx}")(C.byref(P), _ptr(a), _ptr(c), ct(ym), ct(zm))
    return float(chi2), a, c


def run(p, y, z, sector_row, precision="f32", use_grid=True, want_state=False, trace_cap=0, timings=None,
        r17_mode=R17_WAVES):
    """Whole hot path a1..a6.  Returns every stage's output (original cluster indices everywhere)."""
    t0 = time.perf_counter()
    out = {}
    if use_grid:
        out["sorted_idx"], out["bin_first"] = grid(p, y, z, sector_row, precision)
    t1 = time.perf_counter()
    up, dn = neighbours(p, y, z, sector_row, precision, use_grid)
    t2 = time.perf_counter()
    up_c, dn_c, starts = links(up, dn)
    t3 = time.perf_counter()
    fo = follow(p, y, z, sector_row, up_c, starts, precision, use_grid, want_state, trace_cap, r17_mode)
    t4 = time.perf_counter()
    se = select(int(np.asarray(y).size), int(p.n_rows), starts, fo["row_hit"], fo["n_hits"], p.min_hits)
    t5 = time.perf_counter()
    fi = fit(p, y, z, sector_row, se["trk_nhits"], se["trk_first_hit"], se["trk_hits"], precision)
    t6 = time.perf_counter()
    out.update(link_up=up, link_dn=dn, up_c=up_c, dn_c=dn_c, starts=starts, **fo, **se, **fi)
    if timings is not None:
        timings.update(grid=t1 - t0, neighbours=t2 - t1, links=t3 - t2, follow=t4 - t3, select=t5 - t4, fit=t6 - t5,
                       total=t6 - t0)
    return out
