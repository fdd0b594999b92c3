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
