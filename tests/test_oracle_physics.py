"""Pins of R28 (process noise and outlier rejection in the refit, cluster tags), -m "not gpu", oracle only.
PAPER.md l.35 says why synchronous tracking exists (removing hits of tracks not used for physics) and gives no
formula.  What constrains the oracle:
  * the defaults (no material, no cut) reproduce R22 bit for bit
  * with material, the whole recursion is rebuilt here from the pinned primitives (orc.propagate: R12 with its
    Jacobian, pins I7; orc.update: R13, textbook pin) plus the scattering matrix written from the Highland formula in
    numpy -- this pins where and how Q enters
  * a hit displaced by 1.5 cm is rejected in the last pass, it alone, ndf loses 2, and the fit lands where the fit
    without that hit lands
  * the tags, on hand-made arrays
"""
import math

import numpy as np
import pytest

from helix_ref import KB_TRK
from paper_2106_03636_b200.synth import TpcParams, config0, single_helix

ROWX = np.asarray(TpcParams().row_x, np.float64)


def truth_list(ev):
    h = np.argsort(ev.sector_row % 152).astype(np.int32)
    return h


def test_defaults_reproduce_R22_bit_for_bit(orc):
    ev = config0()
    o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)
    f = orc.fit_physics(ev.params, ev.y, ev.z, ev.sector_row, o["trk_nhits"], o["trk_first_hit"], o["trk_hits"])
    for k in ("par", "cov", "xref", "zref", "chi2", "ndf"):
        assert np.array_equal(f[k], o[k]), k
    assert not f["hit_flag"].any()


def highland_q(par, arc, x0inv):
    s, tl, q = par[2], par[3], par[4]
    one = 1.0 + tl * tl
    L = abs(arc) * math.sqrt(one)
    th2 = 0.0136 ** 2 * q * q / one * L * x0inv
    Q = np.zeros((5, 5))
    Q[2, 2] = th2 * (1 - s * s) * one
    Q[3, 3] = th2 * one * one
    Q[3, 4] = Q[4, 3] = th2 * tl * q * one
    Q[4, 4] = th2 * tl * tl * q * q
    return Q


def full(c15):
    C = np.zeros((5, 5))
    C[np.tril_indices(5)] = c15
    return C + np.tril(C, -1).T


def test_process_noise_enters_as_F_C_Ft_plus_Q_after_every_transport(orc):
    ev = single_helix(1.5, math.radians(8.0), 0.5, vz=1.0, smear=True, seed=3)
    p = ev.params
    h = truth_list(ev)
    x0inv = 2e-4
    f = orc.fit_physics(p, ev.y, ev.z, ev.sector_row, [h.size], [0], h, x0inv=x0inv, precision="f64")
    base = orc.fit(p, ev.y, ev.z, ev.sector_row, [h.size], [0], h, "f64")
    assert np.all(np.diag(full(f["cov"][:, 0])) > np.diag(full(base["cov"][:, 0]))), "material must cost precision"
    # the same recursion from the primitives: seed = what R21 gives = the state the noise-free fit starts from; take it
    # from a one-pass run (n_fit_passes = 1 ends at the outermost hit; pass 2 of the real fit starts from there)
    rows = ev.sector_row[h] % 152
    y = ev.y.astype(np.float64); z = ev.z.astype(np.float64)
    zref = float(f["zref"][0])
    one = orc.fit_physics(p.with_(n_fit_passes=1), ev.y, ev.z, ev.sector_row, [h.size], [0], h, x0inv=x0inv, precision="f64")
    par = one["par"][:, 0].copy()
    C = np.diag(np.asarray(p.cov0, np.float64))
    chi2 = 0.0
    at = h.size - 1
    for k in range(h.size - 1, -1, -1):
        if k != at:
            dx = ROWX[rows[k]] - ROWX[rows[at]]
            s1 = par[2]
            ok, par, c15, F = orc.propagate(p, par, C[np.tril_indices(5)], dx, "f64")
            assert ok
            s2 = par[2]
            kap = -KB_TRK * par[4]
            arc = (math.asin(s2) - math.asin(s1)) / kap if abs(kap) > 1e-12 else dx / math.sqrt(1 - s1 * s1)
            C = full(c15) + highland_q(par, arc, x0inv)
            at = k
        c2, par, c15 = orc.update(p, par, C[np.tril_indices(5)], y[h[k]], z[h[k]] - zref, "f64")
        C = full(c15)
        chi2 += c2
    np.testing.assert_allclose(par, f["par"][:, 0], rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(C[np.tril_indices(5)], f["cov"][:, 0], rtol=1e-7, atol=1e-15)
    assert chi2 == pytest.approx(float(f["chi2"][0]), rel=1e-8)


def test_a_displaced_hit_is_rejected_in_the_last_pass(orc):
    ev = single_helix(-1.2, math.radians(11.0), 0.4, vz=2.0, smear=True, seed=5)
    p = ev.params
    h = truth_list(ev)
    k_bad = h.size // 2
    y = ev.y.copy()
    y[h[k_bad]] += 1.5
    f = orc.fit_physics(p, y, ev.z, ev.sector_row, [h.size], [0], h, outlier_cut=30.0, precision="f64")
    assert f["hit_flag"].sum() == 1 and f["hit_flag"][k_bad] == 1
    assert f["ndf"][0] == 2 * (h.size - 1) - 5
    h2 = np.delete(h, k_bad)
    ref = orc.fit(p, ev.y, ev.z, ev.sector_row, [h2.size], [0], h2, "f64")
    spoiled = orc.fit(p, y, ev.z, ev.sector_row, [h.size], [0], h, "f64")
    sig = np.sqrt(np.diag(full(ref["cov"][:, 0])))
    pull = np.abs(f["par"][:, 0] - ref["par"][:, 0]) / sig
    pull_spoiled = np.abs(spoiled["par"][:, 0] - ref["par"][:, 0]) / sig
    assert pull.max() < 0.05, "with the hit rejected the fit is the fit without it (the first pass only seeds the second)"
    assert pull_spoiled.max() > 1.0, "without the rejection the displaced hit pulls the fit by more than a sigma"
    assert f["chi2"][0] / f["ndf"][0] < 2.0 < spoiled["chi2"][0] / spoiled["ndf"][0]
    # no cut: nothing is ever rejected
    assert not orc.fit_physics(p, y, ev.z, ev.sector_row, [h.size], [0], h, precision="f64")["hit_flag"].any()


def test_cluster_tags(orc):
    ct = np.array([-1, 0, 0, 1, 1, 2, -1, 2], np.int32)
    qpt = np.array([0.5, -12.0, 3.0], np.float32)       # track 1 is a low-pT looper
    ndf = np.array([11, 9, -1], np.int32)               # the refit of track 2 failed
    nh = np.array([2, 2, 2], np.int32); fh = np.array([0, 2, 4], np.int64)
    hits = np.array([1, 2, 3, 4, 5, 7], np.int32)
    flag = np.array([0, 1, 0, 0, 0, 0], np.uint8)       # second hit of track 0 was rejected
    tag = orc.tag_clusters(ct, qpt, ndf, nh, fh, hits, flag, qpt_max=10.0)
    assert tag.tolist() == [0, 1, 1 | 4, 1 | 2, 1 | 2, 1 | 2, 0, 1 | 2]
    assert orc.tag_clusters(ct, qpt, ndf, nh, fh, hits, None, qpt_max=20.0).tolist() == [0, 1, 1, 1, 1, 3, 0, 3]


def test_tags_single_out_the_low_pt_loopers_of_a_pileup_event(orc):
    """R28c against the generator's truth on a configs[3]-like event (10 % of the particles are loopers with
    pT 0.05-0.2 GeV, A2): with qpt_max = 1 / (0.2 GeV) the clusters tagged "not used for physics" are, almost all of them,
    clusters of true low-pT particles, and most attached clusters of such particles are tagged."""
    from paper_2106_03636_b200.synth import config3
    ev = config3(n_coll=1, n_tracks=1500)
    o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)
    tag = orc.tag_clusters(o["cluster_track"], o["par"][4], o["ndf"], o["trk_nhits"], o["trk_first_hit"], o["trk_hits"], None,
                           qpt_max=5.0)
    tt = ev.true_track
    pt_true = np.where(tt >= 0, 1.0 / np.abs(ev.trk["qpt"][np.maximum(tt, 0)]), np.inf)
    attached = tag & 1 > 0
    removable = tag & 2 > 0
    low = (tt >= 0) & (pt_true < 0.2)
    high = (tt >= 0) & (pt_true > 0.3)
    assert low.sum() > 2000 and (attached & low).sum() > 500
    assert (removable & low & attached).sum() >= 0.85 * (attached & low).sum(), "attached looper clusters that escape the tag"
    assert (removable & high).sum() <= 0.01 * (attached & high).sum(), "clusters of physics tracks tagged for removal"
    assert not (removable & ~attached).any()


# ---------------------------------------------------------------------------------------------------------------------
# R28d (mean energy loss) and R28e (angle- and drift-dependent cluster errors)
# ---------------------------------------------------------------------------------------------------------------------
from helix_ref import truth_state_local  # noqa: E402
from paper_2106_03636_b200.synth import V_DRIFT  # noqa: E402

OPT_E = dict(err_ang_y=1.5, err_ang_z=0.8, err_drift_y=2e-4, err_drift_z=3e-4, v_drift=V_DRIFT, z_len=250.0)


def errors_of(p, par, z_raw, t0, side, o):
    """R28e written from its definition (numpy side of the pins)."""
    s, tl = par[2], par[3]
    d = max(0.0, o["z_len"] - abs(z_raw + side * o["v_drift"] * t0)) if t0 is not None else 0.0
    sy2 = p.sigma_y ** 2 * (1.0 + o["err_ang_y"] * s * s / (1.0 - s * s)) + o["err_drift_y"] * d
    sz2 = p.sigma_z ** 2 * (1.0 + o["err_ang_z"] * tl * tl) + o["err_drift_z"] * d
    return sy2, sz2


def test_new_options_off_reproduce_R28ab_bit_for_bit(orc):
    ev = config0()
    o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)
    lists = (o["trk_nhits"], o["trk_first_hit"], o["trk_hits"])
    a = orc.fit_physics(ev.params, ev.y, ev.z, ev.sector_row, *lists, x0inv=1e-4, outlier_cut=25.0)
    t0 = np.linspace(-3, 3, o["trk_nhits"].size)
    b = orc.fit_physics(ev.params, ev.y, ev.z, ev.sector_row, *lists, x0inv=1e-4, outlier_cut=25.0, eloss_sigma=0.3,
                        v_drift=V_DRIFT, trk_t0=t0)       # a straggling width and time offsets alone change nothing
    for k in a:
        assert np.array_equal(a[k], b[k]), k


def test_energy_loss_and_cluster_errors_enter_the_recursion_where_R28_says(orc):
    """The whole two-pass recursion rebuilt from the pinned primitives (orc.propagate, orc.update) with the scattering
    matrix, the momentum change and the two variances written here from their definitions."""
    t_us = 7.0
    ev = single_helix(1.5, math.radians(8.0), 0.5, vz=1.0, t_us=t_us, smear=True, seed=3)
    p = ev.params
    h = truth_list(ev)
    x0inv, dedx, esig = 2e-4, 1.5e-4, 0.4
    kw = dict(x0inv=x0inv, dedx=dedx, eloss_sigma=esig, trk_t0=[t_us], precision="f64", **OPT_E)
    f = orc.fit_physics(p, ev.y, ev.z, ev.sector_row, [h.size], [0], h, **kw)
    rows = ev.sector_row[h] % 152
    y = ev.y.astype(np.float64); z = ev.z.astype(np.float64)
    zref = float(f["zref"][0])
    # the R21 seed: a one-pass fit without any hit information is not available, so rebuild BOTH passes from the seed the
    # plain fit of the same hits starts from: par of a 1-pass fit depends on the options, the seed does not -- take the
    # seed from the state the oracle reports for n_fit_passes = 0 (no pass: par = seed)
    seed = orc.fit_physics(p.with_(n_fit_passes=0), ev.y, ev.z, ev.sector_row, [h.size], [0], h, **kw)["par"][:, 0].copy()
    par, chi2, at = seed, 0.0, 0
    for npass, order in enumerate((range(h.size), range(h.size - 1, -1, -1))):
        C = np.diag(np.asarray(p.cov0, np.float64))
        chi2 = 0.0
        direction = +1 if npass == 0 else -1
        for k in order:
            if k != at:
                dx = ROWX[rows[k]] - ROWX[rows[at]]
                s1 = par[2]
                kap = -KB_TRK * par[4]
                ok, par, c15, F = orc.propagate(p, par, C[np.tril_indices(5)], dx, "f64")
                assert ok
                arc = (math.asin(par[2]) - math.asin(s1)) / kap
                C = full(c15) + highland_q(par, arc, x0inv)
                dq = dedx * abs(arc) * abs(par[4]) * par[4]
                par = par.copy()
                par[4] += direction * dq
                C[4, 4] += (esig * dq) ** 2
                at = k
            sy2, sz2 = errors_of(p, par, z[h[k]], t_us, +1.0, OPT_E)
            c2, par, c15 = orc.update(p.with_(sigma_y=math.sqrt(sy2), sigma_z=math.sqrt(sz2)), par, C[np.tril_indices(5)],
                                      y[h[k]], z[h[k]] - zref, "f64")
            C = full(c15)
            chi2 += c2
    np.testing.assert_allclose(par, f["par"][:, 0], rtol=1e-8, atol=1e-11)
    np.testing.assert_allclose(C[np.tril_indices(5)], f["cov"][:, 0], rtol=1e-6, atol=1e-14)
    assert chi2 == pytest.approx(float(f["chi2"][0]), rel=1e-7)
    # and each option moves the result (none is silently ignored)
    for drop in ("dedx", "err_ang_y", "err_ang_z", "err_drift_y", "err_drift_z"):
        g = orc.fit_physics(p, ev.y, ev.z, ev.sector_row, [h.size], [0], h, **{**kw, drop: 0.0})
        assert not np.allclose(g["cov"][:, 0], f["cov"][:, 0], rtol=1e-6), drop


def losing_track(p, q0, s0, tl, dedx, sub=32):
    """Harness-side trajectory with d(1/|q|)/d(arc) = -dedx (beta = 1, direction unchanged by the loss): exact circle
    arcs over 1/32 of a row gap each, the closed-form momentum update after every arc.  Returns y, z at every row and q."""
    y, zz, s, q = 0.0, 0.0, s0, q0
    ys, zs, qs = [y], [zz], [q]
    for r in range(1, ROWX.size):
        step = (ROWX[r] - ROWX[r - 1]) / sub
        for _ in range(sub):
            kap = -KB_TRK * q
            s2 = s + kap * step
            y += (math.sqrt(1 - s * s) - math.sqrt(1 - s2 * s2)) / kap
            arc = (math.asin(s2) - math.asin(s)) / kap
            zz += tl * arc
            q = math.copysign(1.0 / (1.0 / abs(q) - dedx * abs(arc)), q)
            s = s2
        ys.append(y); zs.append(zz); qs.append(q)
    return np.array(ys), np.array(zs), np.array(qs)


def test_energy_loss_recovers_the_momentum_at_the_inner_end(orc):
    """A track that loses 2e-4 GeV/cm (a hundred times the gas, so that the effect dwarfs rounding): with dedx the
    inward pass arrives at the innermost row with the momentum the particle had THERE; without it the fit reports
    an average over the track.  Unsmeared hits, so chi2 measures the model alone."""
    ev = single_helix(2.0, math.radians(10.0), 0.3, smear=False)
    p = ev.params
    dedx, q0 = 2e-4, 2.0
    y, z, q = losing_track(p, q0, 0.02, 0.3, dedx)
    assert q[-1] / q0 > 1.05                                # the loss is a 5 % effect over the track
    sr = np.arange(ROWX.size, dtype=np.int32)
    h = sr.copy()
    on = orc.fit_physics(p, y, z + 5.0, sr, [h.size], [0], h, dedx=dedx, precision="f64")
    off = orc.fit_physics(p, y, z + 5.0, sr, [h.size], [0], h, precision="f64")
    assert on["xref"][0] == ROWX[0]
    err_on, err_off = abs(on["par"][4, 0] - q0), abs(off["par"][4, 0] - q0)
    assert err_on < 5e-4 * q0, err_on                       # what the first-order momentum step leaves
    assert err_off > 50 * err_on and err_off > 0.01 * q0, (err_on, err_off)
    assert on["chi2"][0] < 1e-3 * off["chi2"][0]
    # the sign convention: outward passes lose momentum.  A one-pass (outward) fit ends at the outer row with q there
    one = orc.fit_physics(p.with_(n_fit_passes=1), y, z + 5.0, sr, [h.size], [0], h, dedx=dedx, precision="f64")
    assert abs(one["par"][4, 0] - q[-1]) < 5e-4 * q[-1]


def test_cluster_error_model_gives_unit_pulls_on_hits_smeared_with_it(orc):
    """Hits smeared here with the R28e variances evaluated on the TRUE trajectory: chi2/ndf and the pull of y at the
    inner end come out at 1 with the model (and the right time offset), and do not with constant errors or with the
    time offset of the wrong sign (the drift length is then wrong by 2 v_d t)."""
    rng = np.random.default_rng(11)
    ratio = dict(model=[], const=[], wrong_t0=[])
    pulls = []
    for i in range(160):
        qpt = rng.choice([-1, 1]) * rng.uniform(0.3, 1.6)
        phi = math.radians(10.0 + rng.uniform(-5, 5))
        tanl = rng.uniform(0.05, 0.5)
        t_us = rng.uniform(6.0, 12.0)                       # z_true in [100, 225]: the wrong sign adds 2 v_d t to every drift length
        ev = single_helix(qpt, phi, tanl, vz=100.0, t_us=t_us, smear=False)
        p = ev.params
        h = truth_list(ev)
        if h.size < 60:                                     # left the sector early
            continue
        rows = ev.sector_row[h] % 152
        y = ev.y.astype(np.float64); z = ev.z.astype(np.float64)
        for k, r in zip(h, rows):
            tr = truth_state_local(qpt, phi, tanl, 0.0, 0.0, 100.0, 0, ROWX[r])
            sy2, sz2 = errors_of(p, tr, z[k], t_us, +1.0, OPT_E)
            y[k] += rng.normal(0.0, math.sqrt(sy2)); z[k] += rng.normal(0.0, math.sqrt(sz2))
        args = (p, y, z, ev.sector_row, [h.size], [0], h)
        m = orc.fit_physics(*args, trk_t0=[t_us], precision="f64", **OPT_E)
        c = orc.fit_physics(*args, precision="f64")
        w = orc.fit_physics(*args, trk_t0=[-t_us], precision="f64", **OPT_E)
        for nm, f in (("model", m), ("const", c), ("wrong_t0", w)):
            ratio[nm].append(f["chi2"][0] / f["ndf"][0])
        tr0 = truth_state_local(qpt, phi, tanl, 0.0, 0.0, 100.0, 0, float(m["xref"][0]))
        pulls.append((m["par"][0, 0] - tr0[0]) / math.sqrt(m["cov"][0, 0]))
    # medians: a few short, steep tracks start from a poor three-point seed with these large errors and stay off
    mean = {k: float(np.median(v)) for k, v in ratio.items()}
    assert len(pulls) > 120
    assert 0.96 < mean["model"] < 1.04, mean
    assert mean["const"] > 2.0, mean
    assert mean["wrong_t0"] < 0.9, mean                     # drift lengths, hence errors, overestimated
    pulls = np.sort(np.asarray(pulls))[3:-3]
    assert 0.8 < float(np.std(pulls)) < 1.15 and abs(float(np.mean(pulls))) < 0.25
