"""Seeded synthetic TPC events: the five BASELINE.json configs made concrete.

This module is the *input recipe* (DESIGN.md "Input recipe").
It is shared by the CPU oracle tests and the CUDA path and holds none of the tracker's
arithmetic: it throws helices from vertices, intersects them with the straight pad rows of
the 18-gon TPC, smears, drops, adds noise and shuffles.  The helix is written in *global*
coordinates as a circle of signed curvature kappa = -kB*q/pT (R4); the tracker's own
(y, sinphi) propagation formulas are not used here, which is what makes pin I1 (a noiseless
helix recovers its generating parameters) a real cross-check.

No item of any public dataset is reproduced: the paper's inputs were ALICE raw Time Frames
(PAPER.md l.98), which are not available; these events borrow only their shape (36 sectors x
152 rows, 128-orbit TF, 50 kHz Poisson pile-up, drift-time/z equivalence).
"""
from __future__ import annotations

import math
import os
from dataclasses import dataclass, field

import numpy as np

from .params import KB, N_ROWS, SECTORS_PER_SIDE, V_DRIFT, TpcParams, default_row_x

TWO_PI = 2.0 * math.pi
Z_MAX = 250.0            # drift length per side, cm (BASELINE.json configs[0])
S_MAX = 0.9999           # |sin(phi_local)| beyond which a row crossing is not generated
ORBIT_US = 89.4          # BASELINE.json configs[4]


@dataclass
class Event:
    name: str
    params: TpcParams
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    q: np.ndarray
    sector_row: np.ndarray
    true_track: np.ndarray            # int32, -1 = noise
    trk: dict = field(default_factory=dict)   # per-track truth: qpt, phi, tanl, vx, vy, vz, t_us, collision
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.y.shape[0])


# ----------------------------------------------------------------------------------------
# kinematics samplers (A1, A3, A4)
# ----------------------------------------------------------------------------------------
def _sample_pt_exp(rng, n, tau=0.5, lo=0.1, hi=10.0):
    """pT ~ exp(-pT/tau) truncated to [lo, hi] by inverse CDF (A4)."""
    u = rng.random(n)
    a, b = math.exp(-lo / tau), math.exp(-hi / tau)
    return -tau * np.log(a - u * (a - b))


def _sample_tracks_pbpb(rng, n, frac_secondary=0.15, looper_frac=0.0, vz0=None):
    """configs[1] kinematics: 85 % primaries, 15 % secondaries (A3), exp pT, |eta|<0.9."""
    pt = _sample_pt_exp(rng, n)
    if looper_frac > 0.0:                      # A2: 10 % of tracks get pT uniform in [0.05, 0.2]
        loop = rng.random(n) < looper_frac
        pt = np.where(loop, rng.uniform(0.05, 0.2, n), pt)
    else:
        loop = np.zeros(n, bool)
    eta = rng.uniform(-0.9, 0.9, n)
    phi = rng.uniform(0.0, TWO_PI, n)
    charge = np.where(rng.random(n) < 0.5, -1.0, 1.0)
    sec = rng.random(n) < frac_secondary
    vr = np.where(sec, rng.uniform(0.0, 60.0, n), 0.0)
    va = rng.uniform(0.0, TWO_PI, n)
    if vz0 is None:
        vz = rng.normal(0.0, 5.0, n)           # one collision: every primary shares ... see caller
    else:
        vz = np.where(sec, rng.normal(0.0, 5.0, n), vz0)
    return dict(qpt=charge / pt, phi=phi, tanl=np.sinh(eta), vx=vr * np.cos(va), vy=vr * np.sin(va),
                vz=vz, looper=loop)


# ----------------------------------------------------------------------------------------
# helix / pad-row intersection in a sector-local frame (global-circle algebra)
# ----------------------------------------------------------------------------------------
def _alpha(sec18):
    """Centre azimuth of azimuthal sector 0..17 (R2)."""
    return (np.asarray(sec18, dtype=np.float64) + 0.5) * (TWO_PI / SECTORS_PER_SIDE)


def _crossing(t, idx, sec18, X, branch=1, turn=0):
    """Crossing of tracks t[idx] with the line x_local = X of azimuthal sector sec18.

    Circle through the vertex v with direction phi and curvature kappa = dphi/ds:
        p(s) = v + (1/kappa) * [ sin(phi+kappa s) - sin(phi), -(cos(phi+kappa s) - cos(phi)) ]
    In the frame rotated by alpha the direction angle is phi - alpha.  branch=+1 picks the
    crossing where the particle moves towards +x_local (cos > 0), branch=-1 the returning one.
    Returns (ok, y_local, z_true, s) with s the smallest positive path length (+ `turn` turns).
    """
    a = _alpha(sec18)
    ca, sa = np.cos(a), np.sin(a)
    vx, vy = t["vx"][idx], t["vy"][idx]
    vxl = vx * ca + vy * sa
    vyl = -vx * sa + vy * ca
    kap = t["kappa"][idx]
    phil = t["phi"][idx] - a
    sp, cp = np.sin(phil), np.cos(phil)
    S = sp + kap * (X - vxl)
    ok = np.abs(S) < S_MAX
    Sc = np.clip(S, -S_MAX, S_MAX)
    if branch > 0:
        end = np.arcsin(Sc)
        c2 = np.sqrt(1.0 - Sc * Sc)
    else:
        end = math.pi - np.arcsin(Sc)
        c2 = -np.sqrt(1.0 - Sc * Sc)
    sg = np.sign(kap)
    dphi = (np.mod((end - phil) * sg, TWO_PI) + TWO_PI * turn) * sg
    s = dphi / kap
    yl = vyl - (c2 - cp) / kap
    zt = t["vz"][idx] + t["tanl"][idx] * s
    return ok, yl, zt, s


def _trace_first_leg(t, row_x, tan_half, single_sector):
    """First outgoing leg of every track: (track, sector18, row, y_local, z_true) of each crossing."""
    n = t["kappa"].shape[0]
    allidx = np.arange(n)
    if single_sector:
        sec = np.zeros(n, np.int64)
        alive = np.ones(n, bool)
    else:
        best = np.full(n, np.inf)
        sec = np.full(n, -1, np.int64)
        y0max = row_x[0] * tan_half
        for j in range(SECTORS_PER_SIDE):
            ok, yl, zt, s = _crossing(t, allidx, np.full(n, j), row_x[0])
            ok &= (np.abs(yl) <= y0max) & (s < best)
            best = np.where(ok, s, best)
            sec = np.where(ok, j, sec)
        alive = sec >= 0
    s_prev = np.zeros(n)
    out_t, out_s, out_r, out_y, out_z = [], [], [], [], []
    for r in range(N_ROWS):
        idx = np.nonzero(alive)[0]
        if idx.size == 0:
            break
        X = row_x[r]
        ymax = X * tan_half
        ok, yl, zt, s = _crossing(t, idx, sec[idx], X)
        if not single_sector:
            shift = np.where(ok & (yl > ymax), 1, 0) - np.where(ok & (yl < -ymax), 1, 0)
            mv = np.nonzero(shift)[0]
            if mv.size:
                sec[idx[mv]] = (sec[idx[mv]] + shift[mv]) % SECTORS_PER_SIDE
                ok2, yl2, zt2, s2 = _crossing(t, idx[mv], sec[idx[mv]], X)
                ok[mv], yl[mv], zt[mv], s[mv] = ok2, yl2, zt2, s2
        zin = (np.abs(zt) <= Z_MAX) & ((zt >= 0.0) if single_sector else True)
        cont = ok & zin & (s > s_prev[idx])
        inside = cont & (np.abs(yl) <= ymax)
        if single_sector:
            cont = inside                       # A1: the track ends where it leaves the sector
        alive[idx[~cont]] = False
        s_prev[idx] = s
        k = np.nonzero(inside)[0]
        out_t.append(idx[k]); out_s.append(sec[idx[k]]); out_r.append(np.full(k.size, r))
        out_y.append(yl[k]); out_z.append(zt[k])
    return (np.concatenate(out_t), np.concatenate(out_s), np.concatenate(out_r),
            np.concatenate(out_y), np.concatenate(out_z))


def _trace_loopers(t, idx, row_x, tan_half, max_turns=2):
    """A2: outgoing and returning crossings of low-pT tracks for up to `max_turns` turns (brute force)."""
    out_t, out_s, out_r, out_y, out_z = [], [], [], [], []
    if idx.size == 0:
        z = np.zeros(0)
        return z.astype(np.int64), z.astype(np.int64), z.astype(np.int64), z, z
    smax = max_turns * TWO_PI / np.abs(t["kappa"][idx])
    for r in range(N_ROWS):
        X = row_x[r]
        ymax = X * tan_half
        for j in range(SECTORS_PER_SIDE):
            for branch in (1, -1):
                for turn in range(max_turns):
                    ok, yl, zt, s = _crossing(t, idx, np.full(idx.size, j), X, branch, turn)
                    ok &= (np.abs(yl) <= ymax) & (np.abs(zt) <= Z_MAX) & (s <= smax)
                    k = np.nonzero(ok)[0]
                    if k.size:
                        out_t.append(idx[k]); out_s.append(np.full(k.size, j)); out_r.append(np.full(k.size, r))
                        out_y.append(yl[k]); out_z.append(zt[k])
    if not out_t:
        z = np.zeros(0)
        return z.astype(np.int64), z.astype(np.int64), z.astype(np.int64), z, z
    return (np.concatenate(out_t), np.concatenate(out_s), np.concatenate(out_r),
            np.concatenate(out_y), np.concatenate(out_z))


# ----------------------------------------------------------------------------------------
# event assembly
# ----------------------------------------------------------------------------------------
def choose_cells(n, n_sectors, row_x, tan_half, z_lo, z_hi, occupancy=0.35, cz_min=5.5, lo=1.0, hi=8.0):
    """Grid cell (cell_y, cell_z) in cm for a mean bin occupancy of `occupancy` (R7; R8: results do not depend on it).

    Measured on the Time Frame of configs[4]: about three bins per cluster is the optimum --
    the follower and the CA finder test fewer candidates per lookup, the grid build pays for the extra bins.  The
    drift cell is kept >= 5.5 cm, the height of the CA window (2 * ca_max_dzdx * pitch = 5.3 cm), so that every
    window spans at most two z-bin rows; the rest of the area budget goes to y.  Quarter-cm steps: exact in fp32."""
    area = n_sectors * float(np.sum(2.0 * row_x.astype(np.float64) * tan_half)) * (z_hi - z_lo)
    cell_area = occupancy * area / max(n, 1)
    q = lambda v: float(np.float32(round(min(max(v, lo), hi) * 4.0) / 4.0))
    cz = q(max(math.sqrt(cell_area), cz_min))
    cy = q(cell_area / cz)
    return cy, cz


def _trace_signal(rng, t, t_us, sigma_y, sigma_z, dropout, single_sector, smear=True):
    """Trace tracks `t`, apply dropout (A5), the drift-time shift (R5) and smearing.

    Returns (track index, sector, row, y_local, z_meas) of every signal cluster; float64 y/z."""
    rx64 = default_row_x().astype(np.float64)
    tan_half = math.tan(math.radians(10.0))
    t = dict(t)
    t["kappa"] = -KB * t["qpt"]
    loop = t.get("looper", np.zeros(t["qpt"].shape[0], bool))
    norm = np.nonzero(~loop)[0]
    sub = {k: v[norm] for k, v in t.items()}
    a_t, a_s, a_r, a_y, a_z = _trace_first_leg(sub, rx64, tan_half, single_sector)
    a_t = norm[a_t]
    if loop.any():
        b = _trace_loopers(t, np.nonzero(loop)[0], rx64, tan_half)
        a_t, a_s, a_r, a_y, a_z = (np.concatenate([u, v]) for u, v in zip((a_t, a_s, a_r, a_y, a_z), b))
    # dropout per crossing (A5)
    if dropout > 0.0:
        keep = rng.random(a_t.size) >= dropout
        a_t, a_s, a_r, a_y, a_z = a_t[keep], a_s[keep], a_r[keep], a_y[keep], a_z[keep]
    side = np.where(a_z >= 0.0, 1.0, -1.0)
    sector = a_s + np.where(side > 0, 0, SECTORS_PER_SIDE)
    if single_sector:
        sector = np.zeros_like(a_s)
    zm = a_z - side * V_DRIFT * np.asarray(t_us)[a_t]     # R5
    if smear:
        a_y = a_y + rng.normal(0.0, sigma_y, a_t.size)
        zm = zm + rng.normal(0.0, sigma_z, a_t.size)
    return a_t, sector, a_r, a_y, zm


def _finish(name, rng, t, t_us, sig, noise_frac, single_sector, params_kw=None, shuffle=True):
    """Add noise (A5) and charge (A6), shuffle, choose the grid range/cell and build the Event."""
    a_t, sector, a_r, a_y, zm = sig
    row_x = default_row_x()
    rx64 = row_x.astype(np.float64)
    tan_half = math.tan(math.radians(10.0))
    n_sig = a_t.size
    n_sectors = 1 if single_sector else 2 * SECTORS_PER_SIDE
    # noise (A5): uniform over (sector,row), y across the row, z over that side's occupied range
    n_noise = int(round(noise_frac * n_sig))
    if n_noise > 0:
        ns = rng.integers(0, n_sectors, n_noise)
        nr = rng.integers(0, N_ROWS, n_noise)
        ny = rng.uniform(-1.0, 1.0, n_noise) * rx64[nr] * tan_half
        side = np.where(sector < SECTORS_PER_SIDE, 1.0, -1.0) if not single_sector else np.ones(n_sig)
        zeta = side * zm                                   # mirrored drift coordinate
        zl, zh = (float(zeta.min()), float(zeta.max())) if n_sig else (0.0, Z_MAX)
        del zeta, side
        nside = np.where(ns < SECTORS_PER_SIDE, 1.0, -1.0)
        nz = nside * rng.uniform(zl, zh, n_noise)
        sector = np.concatenate([sector, ns]); a_r = np.concatenate([a_r, nr])
        a_y = np.concatenate([a_y, ny]); zm = np.concatenate([zm, nz])
        a_t = np.concatenate([a_t, np.full(n_noise, -1)])
    n = a_t.size
    q = 20.0 + rng.exponential(30.0, n)                    # A6
    y32 = a_y.astype(np.float32); z32 = zm.astype(np.float32)
    sr = (sector * N_ROWS + a_r).astype(np.int32)
    tt = a_t.astype(np.int32); q32 = q.astype(np.float32)
    del a_y, zm, a_t, q
    if shuffle:
        perm = rng.permutation(n)
        y32, z32, sr, tt, q32 = y32[perm], z32[perm], sr[perm], tt[perm], q32[perm]
        del perm
    sgn = np.where(sr < SECTORS_PER_SIDE * N_ROWS, np.float32(1.0), np.float32(-1.0)) if not single_sector \
        else np.ones(n, np.float32)
    zeta = (sgn * z32).astype(np.float64)
    z_lo = float(np.floor(zeta.min() - 1.0)) if n else -1.0
    z_hi = float(np.ceil(zeta.max() + 1.0)) if n else Z_MAX + 1.0
    del zeta, sgn
    cell_y, cell_z = choose_cells(n, n_sectors, row_x, tan_half, z_lo, z_hi)
    kw = dict(n_sectors=n_sectors, z_lo=z_lo, z_hi=z_hi, cell_y=cell_y, cell_z=cell_z)
    kw.update(params_kw or {})
    p = TpcParams(**kw)
    trk = {k: np.asarray(v) for k, v in t.items()}
    trk["t_us"] = np.asarray(t_us)
    return Event(name=name, params=p, x=row_x[sr % N_ROWS], y=y32, z=z32, q=q32,
                 sector_row=sr, true_track=tt, trk=trk,
                 meta=dict(n_signal=int(n_sig), n_noise=int(n_noise)))


def _assemble(name, rng, t, t_us, sigma_y, sigma_z, dropout, noise_frac, single_sector, params_kw=None,
              smear=True, shuffle=True):
    """Trace all tracks, apply drift-time shift (R5), smear, drop, add noise (A5), shuffle."""
    sig = _trace_signal(rng, t, t_us, sigma_y, sigma_z, dropout, single_sector, smear)
    return _finish(name, rng, t, t_us, sig, noise_frac, single_sector, params_kw, shuffle)


def config0(seed=1, n_tracks=200, **kw):
    """configs[0]: one sector, 200 origin helices, 1/pT U[0.2,5], |eta| (A1), no noise, no time offset."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = n_tracks
    inv_pt = rng.uniform(0.2, 5.0, n)
    charge = np.where(rng.random(n) < 0.5, -1.0, 1.0)
    eta = np.abs(rng.uniform(-0.9, 0.9, n))
    phi = rng.uniform(0.0, math.radians(20.0), n)          # within sector 0 (alpha_0 = 10 deg +- 10 deg)
    t = dict(qpt=charge * inv_pt, phi=phi, tanl=np.sinh(eta), vx=np.zeros(n), vy=np.zeros(n), vz=np.zeros(n))
    return _assemble("c0", rng, t, np.zeros(n), 0.08, 0.10, 0.0, 0.0, True, **kw)


def config1(seed=2, n_tracks=5000, **kw):
    """configs[1]: one central Pb-Pb collision, full TPC, 2 % dropout, 5 % noise."""
    rng = np.random.Generator(np.random.PCG64(seed))
    vz0 = rng.normal(0.0, 5.0)
    t = _sample_tracks_pbpb(rng, n_tracks, vz0=vz0)
    return _assemble("c1", rng, t, np.zeros(n_tracks), 0.08, 0.10, 0.02, 0.05, False, **kw)


def _one_collision(args):
    """Tracks + signal clusters of one collision from its own counter-seeded stream (order-free, so the
    collisions can be generated by a process pool and the event is identical for any worker count)."""
    seed, ic, tc, m, dropout, looper_frac = args
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([int(seed), int(ic)])))
    vz0 = rng.normal(0.0, 5.0)
    t = _sample_tracks_pbpb(rng, int(m), looper_frac=looper_frac, vz0=vz0)
    a_t, sector, a_r, a_y, zm = _trace_signal(rng, t, np.full(int(m), tc), 0.08, 0.10, dropout, False)
    return t, (a_t.astype(np.int32), sector.astype(np.int8), a_r.astype(np.int16), a_y.astype(np.float32), zm)


def _pileup(name, seed, t_coll_us, mult, dropout, noise, looper_frac=0.0, workers=None, **kw):
    jobs = [(seed, ic, float(tc), int(m), dropout, looper_frac)
            for ic, (tc, m) in enumerate(zip(t_coll_us, mult)) if m > 0]
    total = sum(j[3] for j in jobs)
    if workers is None:
        workers = min(os.cpu_count() or 1, 32) if total > 100000 else 1
    if workers > 1:
        import multiprocessing as mp
        order = sorted(range(len(jobs)), key=lambda i: -jobs[i][3])       # big collisions first
        with mp.get_context("fork").Pool(workers) as pool:
            res = pool.map(_one_collision, [jobs[i] for i in order], chunksize=1)
        out = [None] * len(jobs)
        for i, r in zip(order, res):
            out[i] = r
    else:
        out = [_one_collision(j) for j in jobs]
    parts = [o[0] for o in out]
    t = {k: np.concatenate([p[k] for p in parts]) for k in parts[0]}
    t["collision"] = np.concatenate([np.full(j[3], j[1]) for j in jobs])
    t_us = np.concatenate([np.full(j[3], j[2]) for j in jobs])
    off = np.cumsum([0] + [j[3] for j in jobs])
    a_t = np.concatenate([o[1][0].astype(np.int64) + off[i] for i, o in enumerate(out)])
    sig = (a_t, np.concatenate([o[1][1] for o in out]).astype(np.int64),
           np.concatenate([o[1][2] for o in out]).astype(np.int64),
           np.concatenate([o[1][3] for o in out]), np.concatenate([o[1][4] for o in out]))
    del out, parts
    rng = np.random.Generator(np.random.PCG64(seed))
    return _finish(name, rng, t, t_us, sig, noise, False, kw.pop("params_kw", None), **kw), rng


def config2(seed=3, n_coll=200, mean_mult=30.0, window_us=1000.0, **kw):
    """configs[2]: pp-like continuous slice, collisions uniform over 1 ms, Poisson(30) tracks, 2 % noise."""
    r0 = np.random.Generator(np.random.PCG64(seed + 1000))
    tc = np.sort(r0.uniform(0.0, window_us, n_coll))
    mult = r0.poisson(mean_mult, n_coll)
    ev, _ = _pileup("c2", seed, tc, mult, 0.02, 0.02, **kw)
    return ev


def config3(seed=4, n_coll=5, n_tracks=5000, window_us=100.0, **kw):
    """configs[3]: 5 central collisions within one drift window, 10 % loopers, 20 % noise, 5 % dropout."""
    r0 = np.random.Generator(np.random.PCG64(seed + 1000))
    tc = np.sort(r0.uniform(0.0, window_us, n_coll))
    ev, _ = _pileup("c3", seed, tc, [n_tracks] * n_coll, 0.05, 0.20, looper_frac=0.10, **kw)
    return ev


def config4(seed=5, n_orbits=128, rate_khz=50.0, max_mult=5000, **kw):
    """configs[4]: one 50 kHz min-bias Pb-Pb Time Frame (A8), 2 % dropout (A5), 5 % noise."""
    r0 = np.random.Generator(np.random.PCG64(seed + 1000))
    T = n_orbits * ORBIT_US
    gaps = r0.exponential(1000.0 / rate_khz, int(T * rate_khz / 1000.0 * 1.5) + 64)
    tc = np.cumsum(gaps)
    tc = tc[tc < T]
    mult = np.floor(max_mult * r0.random(tc.size) ** 2).astype(np.int64)
    ev, _ = _pileup("c4", seed, tc, mult, 0.02, 0.05, **kw)
    ev.meta["tf_us"] = T
    return ev


def make_config(i: int, **kw) -> Event:
    return (config0, config1, config2, config3, config4)[i](**kw)


def single_helix(qpt, phi, tanl, vz=0.0, t_us=0.0, smear=False, seed=0):
    """One helix from the origin in the single-sector geometry (for pin I1); noiseless by default."""
    rng = np.random.Generator(np.random.PCG64(seed))
    t = dict(qpt=np.array([qpt], float), phi=np.array([phi], float), tanl=np.array([tanl], float),
             vx=np.zeros(1), vy=np.zeros(1), vz=np.array([vz], float))
    return _assemble("helix", rng, t, np.array([t_us], float), 0.08, 0.10, 0.0, 0.0, True, smear=smear)
