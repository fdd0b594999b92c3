"""Pins of R26 (merging of sector-local tracks across sector edges, the central electrode and long holes,
and the refit of the merged hit list), -m "not gpu", oracle only.

PAPER.md only says that the full TPC is tracked (l.35, l.60); R26 is a reading.  What constrains it here comes from
geometry and statistics, never from a run of the CUDA path:
  * a noiseless helix that crosses a 20-degree edge is found as one track per sector, the pieces are linked, the
    global track holds every cluster, and its refit returns the generating q/pT, tan(lambda), direction and vertex z
  * the same across the central electrode, with a non-zero collision time (the two sides measure z_true -+ v_d t)
  * two different tracks that end / start at the same edge are not linked (by the chi2 if they share curvature and
    dip, by the (tanlambda, q/pT) gate -- a necessary condition of the chi2 cut -- otherwise)
  * relabelling the sectors (rotation by 20 degrees, A <-> C mirror) relabels the links and nothing else
  * with the configs' smearing the chi2 of true links is chi2-distributed with 5 (4 across the electrode) degrees of
    freedom -- this pins the rotation Jacobian, the transported covariance and the Cholesky chi2 in one number
  * succ / pred are the reciprocal arg-mins of the pair chi2 matrix (brute force in numpy)
  * on a central collision every link joins pieces of one true particle, and nearly all true splits are recovered
"""
import math

import numpy as np
import pytest

from helix_ref import KB_TRK, to_beamline
from paper_2106_03636_b200.synth import TpcParams
from paper_2106_03636_b200.synth import generator as gen

NR = 152


def tracks_event(t, t_us=None, smear=False, dropout=0.0, seed=0):
    """Full-TPC event from explicit true tracks (dict of arrays: qpt, phi, tanl, vx, vy, vz)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = len(t["qpt"])
    t = {k: np.asarray(v, float) for k, v in t.items()}
    t_us = np.zeros(n) if t_us is None else np.asarray(t_us, float)
    return gen._assemble("merge", rng, t, t_us, 0.08, 0.10, dropout, 0.0, False, smear=smear)


def one(qpt, phi_deg, tanl, vz=0.0):
    return dict(qpt=[qpt], phi=[math.radians(phi_deg)], tanl=[tanl], vx=[0.0], vy=[0.0], vz=[vz])


def run_merge(orc, ev, prec="f64", **mp):
    o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, prec, True)
    m = orc.merge(ev.params, ev.y, ev.z, ev.sector_row, o, mp or None, prec, want_pairs=True)
    return o, m


def chains(m):
    out = []
    for h in np.nonzero(m["pred"] < 0)[0]:
        c = [int(h)]
        while m["succ"][c[-1]] >= 0:
            c.append(int(m["succ"][c[-1]]))
        out.append(c)
    return out


# ------------------------------------------------------------------------------------------------------------
# one noiseless helix across a sector edge
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("qpt,phi_deg,tanl,vz", [(2.0, 12.0, 0.4, 3.0), (-2.5, 47.0, -0.6, -4.0), (3.0, 355.0, 0.2, 0.0)])
def test_noiseless_helix_across_a_sector_edge_is_one_global_track(orc, qpt, phi_deg, tanl, vz):
    ev = tracks_event(one(qpt, phi_deg, tanl, vz))
    sectors = np.unique(ev.sector_row // NR)
    assert sectors.size >= 2, "the test track must cross an edge"
    o, m = run_merge(orc, ev)
    K = o["trk_seed"].size
    assert K == sectors.size, "one sector-local track per sector"
    ch = chains(m)
    assert len(ch) == 1 and len(ch[0]) == K, "all pieces linked into one chain"
    assert m["g_nhits"][0] == int(o["trk_nhits"].sum()) == ev.n, "the global track holds every cluster"
    # the chain runs outward: first rows ascend, neighbouring sectors
    rf = m["row_first"][ch[0]]
    assert np.all(np.diff(rf) > 0)
    assert np.all(m["succ_chi2"][ch[0][:-1]] < 1e-6), "noiseless: the pieces agree exactly"
    # refit of the merged hit list: generating parameters back (the pieces alone see 10-60 rows, the chain all of them)
    par = m["gpar"][:, 0]
    assert m["gndf"][0] == 2 * ev.n - 5 and m["gchi2"][0] < 1e-4
    assert par[4] == pytest.approx(qpt, rel=1e-5)
    assert par[3] == pytest.approx(tanl, rel=1e-5)
    head_sector = int(m["trk_sector"][ch[0][0]])
    phi0, z0, dca = to_beamline(par, m["gxref"][0], m["gzref"][0] + par[1], head_sector)
    assert abs((phi0 - math.radians(phi_deg) + math.pi) % (2 * math.pi) - math.pi) < 1e-5
    assert abs(z0 - vz) < 1e-3 and dca < 1e-3


def test_noiseless_helix_across_the_central_electrode(orc):
    """vz = +60 cm, tan(lambda) = -0.35: z_true falls through 0 near x = 165 cm, inside the TPC; collision at t = 7 us, so side A
    measures z_true - v_d t and side C z_true + v_d t (R5): the pieces differ by 2 v_d t = 36 cm in z and still link,
    and the refit (time offset free per side) returns the curvature and the dip angle."""
    t_us = 7.0
    ev = tracks_event(one(1.2, 15.0, -0.35, 60.0), t_us=[t_us])
    sec = np.unique(ev.sector_row // NR)
    assert (sec < 18).any() and (sec >= 18).any()
    o, m = run_merge(orc, ev)
    ch = chains(m)
    assert len(ch) == 1 and len(ch[0]) == o["trk_seed"].size >= 2
    sides = m["trk_sector"][ch[0]] < 18
    assert sides[0] and not sides[-1], "the chain starts on side A and ends on side C"
    k = int(np.nonzero(np.diff(sides.astype(int)))[0][0])
    a, b = ch[0][k], ch[0][k + 1]
    # the z jump between the two sides is 2 v_d t
    za = o["zref"][a] + o["par"][1, a]; zb = o["zref"][b] + o["par"][1, b]
    dxs = gen.default_row_x()[m["row_first"][b]] - gen.default_row_x()[m["row_first"][a]]
    assert m["g_nhits"][0] == ev.n
    assert m["gpar"][4, 0] == pytest.approx(1.2, rel=1e-5) and m["gpar"][3, 0] == pytest.approx(-0.35, rel=1e-5)
    assert m["gndf"][0] == 2 * ev.n - 5 - 1, "one z residual is spent on the free offset of the second side"
    # time from the electrode crossing: z_C - z_A = 2 v_d t at the same point of the track
    st = orc.propagate(ev.params, o["par"][:, a], o["cov"][:, a], float(dxs), "f64")
    assert st[0]
    z_a_at_xb = o["zref"][a] + st[1][1]
    assert (zb - z_a_at_xb) / (2 * gen.V_DRIFT) == pytest.approx(t_us, abs=1e-3)


@pytest.mark.parametrize("t_us", [40.0, 5000.0])
def test_electrode_link_at_the_collision_times_of_a_time_frame(orc, t_us):
    """The two sides measure z_true -+ v_d t, so across the electrode the z window is on z_A + z_B (= 2 z_true, small
    near the electrode), never on z_B - z_A (= 2 v_d t: 206 cm at 40 us, 258 m at 5000 us -- the collision times of a
    Time Frame run up to 1.1e4 us, R3).  Same helix as above at such times: linked, refit as before, 2 v_d t read back."""
    assert 2 * gen.V_DRIFT * t_us > 3 * 64.0, "the jump must be far outside dz_max for this to pin the sign"
    ev = tracks_event(one(1.2, 15.0, -0.35, 60.0), t_us=[t_us])
    o, m = run_merge(orc, ev)
    ch = chains(m)
    assert len(ch) == 1 and len(ch[0]) == o["trk_seed"].size >= 2
    sides = m["trk_sector"][ch[0]] < 18
    k = int(np.nonzero(np.diff(sides.astype(int)))[0][0])
    a, b = ch[0][k], ch[0][k + 1]
    assert m["g_nhits"][0] == ev.n and m["gndf"][0] == 2 * ev.n - 6
    assert m["gpar"][4, 0] == pytest.approx(1.2, rel=1e-5) and m["gpar"][3, 0] == pytest.approx(-0.35, rel=1e-5)
    zb = o["zref"][b] + o["par"][1, b]
    dxs = gen.default_row_x()[m["row_first"][b]] - gen.default_row_x()[m["row_first"][a]]
    st = orc.propagate(ev.params, o["par"][:, a], o["cov"][:, a], float(dxs), "f64")
    assert st[0]
    assert (zb - (o["zref"][a] + st[1][1])) / (2 * gen.V_DRIFT) == pytest.approx(t_us, rel=1e-6, abs=1e-3)


def test_same_side_pieces_with_mirrored_z_are_not_linked(orc):
    """Inside one side the window is on z_B - z_A.  Two particles on the same circle in the bending plane, flat in z
    (tan lambda = 0.01), one measured at z = +40 cm and one -- a later collision -- at z = -40 cm on the same side; the
    first keeps its clusters below row 70, the second those above row 75.  Every test of R26 but the z window would pass
    (same sector, 7 rows apart, same tan lambda and q/pT, same y and direction): z_B + z_A = 0 but z_B - z_A = -80 cm,
    beyond dz_max = 64 -- not compared.  Control: the second particle at z = +40 as well -- linked."""
    from types import SimpleNamespace
    t_shift = 80.0 / gen.V_DRIFT                          # side A measures z_true - v_d t
    for z2, linked in ((-40.0, False), (40.0, True)):
        t = dict(qpt=[0.3, 0.3], phi=[math.radians(10.0)] * 2, tanl=[0.01, 0.01], vx=[0.0, 0.0], vy=[0.0, 0.0], vz=[40.0, 40.0])
        full = tracks_event(t, t_us=[0.0, t_shift if z2 < 0 else 0.0])
        row = full.sector_row % NR
        assert np.all(full.sector_row // NR == 0)
        keep = ((full.true_track == 0) & (row < 70)) | ((full.true_track == 1) & (row > 75))
        ev = SimpleNamespace(params=full.params, y=full.y[keep], z=full.z[keep], sector_row=full.sector_row[keep])
        assert abs(float(np.median(ev.z[row[keep] > 75])) - z2) < 3.0      # 40 cm + 0.01 x path, shifted
        o, m = run_merge(orc, ev)
        assert o["trk_seed"].size == 2
        a, b = np.argsort(m["row_first"])
        assert m["row_last"][a] == 69 and m["row_first"][b] == 76
        if linked:
            assert m["succ"][a] == b and m["pred"][b] == a and 0.0 <= m["pair_chi2"][a, b] < 1e-6
        else:
            assert m["succ"][a] == -1 and m["pred"][b] == -1 and m["pair_chi2"][a, b] == -1.0


# ------------------------------------------------------------------------------------------------------------
# the rotation primitive
# ------------------------------------------------------------------------------------------------------------
def exact_rotation_map(orc, p, v, x0, delta, x_fixed):
    """The map R26's rotation stands for, built from plane geometry and the pinned R12 only: the state v = (y, z, sinphi,
    tanlambda, q/pT) at the plane x0 of the old frame -> the state of the same helix at the FIXED plane x_fixed of the frame
    turned by delta."""
    y, z, s, tl, q = v
    cd, sd = math.cos(delta), math.sin(delta)
    xr, yr = x0 * cd + y * sd, y * cd - x0 * sd
    sr = s * cd - math.sqrt(1.0 - s * s) * sd
    ok, par, _, _ = orc.propagate(p, [yr, z, sr, tl, q], np.zeros(15), x_fixed - xr, "f64")
    assert ok
    return par


@pytest.mark.parametrize("delta_deg", [20.0, -20.0])
@pytest.mark.parametrize("v,x0", [((38.0, 12.0, 0.25, 0.6, 1.5), 150.0), ((-25.0, -40.0, -0.3, -1.1, -2.5), 110.0),
                                  ((5.0, 100.0, 0.05, 0.2, 0.2), 220.0)])
def test_rotation_jacobian_against_finite_differences(orc, v, x0, delta_deg):
    """orc.rotate: (i) point and direction are the plane rotation; (ii) the covariance is D C D with D the DIAGONAL of the
    Jacobian of the exact map -- taken here from central differences, not from a formula -- entry by entry; (iii) the exact
    map has two more non-zero entries, dz'/dy = -sin(delta) tanl / cosphi' and dsinphi'/dy = -sin(delta) kappa, which R26
    drops (R26 says so): their size is measured here so that the approximation is a stated number."""
    p = TpcParams()
    delta = math.radians(delta_deg)
    v = np.array(v, float)
    rng = np.random.default_rng(26)
    A = rng.normal(size=(5, 5)) * np.array([0.1, 0.1, 0.01, 0.01, 0.05])[:, None]
    Cm = A @ A.T + np.diag([1e-3, 1e-3, 1e-5, 1e-5, 1e-4])
    c15 = np.array([Cm[i, j] for i in range(5) for j in range(i + 1)])
    ok, par, cov, xn = orc.rotate(p, v, c15, x0, delta, "f64")
    assert ok
    cd, sd = math.cos(delta), math.sin(delta)
    assert xn == pytest.approx(x0 * cd + v[0] * sd, rel=1e-14)
    want = exact_rotation_map(orc, p, v, x0, delta, xn)
    assert np.allclose(par, want, rtol=0, atol=1e-12), "(i) the rotated state is the helix at the plane x' = xn"
    J = np.zeros((5, 5))
    for j, h in enumerate([1e-4, 1e-4, 1e-6, 1e-6, 1e-6]):
        e = np.zeros(5); e[j] = h
        J[:, j] = (exact_rotation_map(orc, p, v + e, x0, delta, xn) - exact_rotation_map(orc, p, v - e, x0, delta, xn)) / (2 * h)
    D = np.diag(J)
    Cn = np.zeros((5, 5))
    for i in range(5):
        for j in range(i + 1):
            Cn[i, j] = Cn[j, i] = cov[i * (i + 1) // 2 + j]
    assert np.allclose(Cn, D[:, None] * Cm * D[None, :], rtol=2e-7, atol=0), "(ii) C' = D C D, D = diag of the exact Jacobian"
    assert abs(D[0] - 1) > 0.01 and abs(D[2] - 1) > 0.01 and np.allclose(D[[1, 3, 4]], 1.0, atol=1e-9)
    # (iii) what the diagonal form leaves out
    cn = math.sqrt(1.0 - par[2] ** 2)
    kappa = -KB_TRK * v[4]
    off = J - np.diag(D)
    assert off[1, 0] == pytest.approx(-sd * v[3] / cn, rel=1e-6)
    assert off[2, 0] == pytest.approx(-sd * kappa, rel=1e-5, abs=1e-10)
    off[1, 0] = off[2, 0] = 0.0
    assert np.abs(off).max() < 1e-7, "no other entry"


def test_different_tracks_at_the_same_edge_are_not_linked(orc):
    """Two particles of the SAME curvature and dip leave a sector through the same edge, 0.6 degrees and 7 cm in z
    apart: the piece of one in the first sector and the piece of the other in the second pass every window and the
    (tanlambda, q/pT) gate of R26 -- they are compared, and it is the chi2 (position and direction) that keeps them
    apart; each particle's own pieces link.  A pair that differs in curvature instead never reaches the chi2 (gate)."""
    t = dict(qpt=[2.0, 2.0], phi=[math.radians(12.0), math.radians(12.6)], tanl=[0.4, 0.4], vx=[0.0, 0.0], vy=[0.0, 0.0],
             vz=[3.0, 10.0])
    ev = tracks_event(t)
    o, m = run_merge(orc, ev)
    lab = np.array([np.bincount(ev.true_track[o["trk_hits"][f:f + n]]).argmax()
                    for f, n in zip(o["trk_first_hit"], o["trk_nhits"])])
    assert (lab == 1).sum() >= 2 and (lab == 0).sum() >= 2
    a = np.nonzero(m["succ"] >= 0)[0]
    assert a.size >= 2 and np.all(lab[a] == lab[m["succ"][a]]), "only pieces of the same particle are linked"
    cross = np.concatenate([m["pair_chi2"][np.ix_(lab == 0, lab == 1)].ravel(), m["pair_chi2"][np.ix_(lab == 1, lab == 0)].ravel()])
    assert (cross > 50.0).any(), "the cross pairs were looked at: a finite chi2, far above the cut"
    assert not ((cross >= 0) & (cross < 50.0)).any()
    # other curvature (q/pT 2.0 and 2.1): removed by the gate, chi2 never formed, own pieces still linked
    t["qpt"] = [2.0, 2.1]; t["phi"] = [math.radians(12.0)] * 2; t["tanl"] = [0.4, 0.5]; t["vz"] = [3.0, 3.0]
    ev = tracks_event(t)
    o, m = run_merge(orc, ev)
    lab = np.array([np.bincount(ev.true_track[o["trk_hits"][f:f + n]]).argmax()
                    for f, n in zip(o["trk_first_hit"], o["trk_nhits"])])
    a = np.nonzero(m["succ"] >= 0)[0]
    assert a.size == 2 and np.all(lab[a] == lab[m["succ"][a]])
    assert np.all(m["pair_chi2"][np.ix_(lab == 0, lab == 1)] == -1) and np.all(m["pair_chi2"][np.ix_(lab == 1, lab == 0)] == -1)


def test_links_follow_a_relabelling_of_the_sectors(orc):
    """Rotation by 20 degrees (sector s -> s + 1 on its side) and the A <-> C mirror (z -> -z) are symmetries of the
    geometry (R2): the same pairs are linked, with the same chi2."""
    rng = np.random.Generator(np.random.PCG64(5))
    n = 60
    t = dict(qpt=rng.choice([-1, 1], n) / rng.uniform(0.3, 1.5, n), phi=rng.uniform(0, 2 * math.pi, n),
             tanl=rng.uniform(-0.8, 0.8, n), vx=np.zeros(n), vy=np.zeros(n), vz=rng.normal(0, 5, n))
    ev = tracks_event(t, smear=True, seed=6)
    p = ev.params
    o, m = run_merge(orc, ev, "f64")
    s, r = ev.sector_row // NR, ev.sector_row % NR

    def links(o_, m_):
        seeds = o_["trk_seed"]
        return {(int(seeds[a]), int(seeds[b])): float(m_["succ_chi2"][a]) for a, b in enumerate(m_["succ"]) if b >= 0}

    ref = links(o, m)
    assert len(ref) > 20
    rot = ((s % 18 + 1) % 18 + 18 * (s // 18)) * NR + r
    o2 = orc.run(p, ev.y, ev.z, rot.astype(np.int32), "f64", True)
    m2 = orc.merge(p, ev.y, ev.z, rot.astype(np.int32), o2, None, "f64")
    got = links(o2, m2)
    assert got.keys() == ref.keys()
    assert all(got[k] == pytest.approx(ref[k], rel=1e-9, abs=1e-12) for k in ref)
    mir = ((s + 18) % 36) * NR + r
    pm = p.with_(z_lo=-float(p.z_hi), z_hi=-float(p.z_lo)) if False else p
    o3 = orc.run(pm, ev.y, -ev.z, mir.astype(np.int32), "f64", True)
    m3 = orc.merge(pm, ev.y, -ev.z, mir.astype(np.int32), o3, None, "f64")
    got = links(o3, m3)
    assert got.keys() == ref.keys()
    assert all(got[k] == pytest.approx(ref[k], rel=1e-9, abs=1e-12) for k in ref)


# ------------------------------------------------------------------------------------------------------------
# statistics: the chi2 of true links, the arg-mins, efficiency and purity of the links
# ------------------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def busy(orc):
    from paper_2106_03636_b200.synth import config1
    ev = config1(n_tracks=1500)
    o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)
    m = orc.merge(ev.params, ev.y, ev.z, ev.sector_row, o, None, "f32")
    lab = np.array([np.bincount(ev.true_track[o["trk_hits"][f:f + n]] + 1).argmax() - 1
                    for f, n in zip(o["trk_first_hit"], o["trk_nhits"])])
    return ev, o, m, lab


def test_chi2_of_true_links_has_five_degrees_of_freedom(busy):
    ev, o, m, lab = busy
    a = np.nonzero(m["succ"] >= 0)[0]
    b = m["succ"][a]
    same_side = (m["trk_sector"][a] < 18) == (m["trk_sector"][b] < 18)
    c2 = m["succ_chi2"][a][same_side & (lab[a] == lab[b])]
    assert c2.size > 500
    # chi2(5): mean 5, median 4.35, 90 % quantile 9.24; a wrong Jacobian or covariance moves these by factors
    assert np.mean(c2) == pytest.approx(5.0, rel=0.2)
    assert np.median(c2) == pytest.approx(4.35, rel=0.2)
    assert np.quantile(c2, 0.9) == pytest.approx(9.24, rel=0.25)


def test_links_are_pure_and_recover_the_true_splits(busy):
    ev, o, m, lab = busy
    a = np.nonzero(m["succ"] >= 0)[0]
    b = m["succ"][a]
    assert np.all(lab[a] >= 0) and np.count_nonzero(lab[a] != lab[b]) <= 0.005 * a.size, "wrong links"
    splits = sum(c - 1 for c in np.bincount(lab[lab >= 0]) if c > 0)
    assert a.size >= 0.95 * splits, f"only {a.size} of {splits} true splits linked"
    # bookkeeping of the global tracks
    K = o["trk_seed"].size
    M = m["g_head"].size
    assert M == K - a.size and int(m["g_nhits"].sum()) == int(o["trk_nhits"].sum())
    assert np.array_equal(np.bincount(m["trk_global"], minlength=M), m["g_nseg"])
    single = m["g_nseg"] == 1
    h = m["g_head"][single]
    assert np.array_equal(m["gpar"][:, single], o["par"][:, h]) and np.array_equal(m["gndf"][single], o["ndf"][h])
    merged_ok = (~single) & (m["gndf"] > 0)
    assert merged_ok.sum() >= 0.97 * (~single).sum(), "merged refits that ran into max_sinphi"
    assert np.median(m["gchi2"][merged_ok] / m["gndf"][merged_ok]) == pytest.approx(1.0, abs=0.1)
    # a merged track measures the curvature better than its head alone did
    hm = m["g_head"][merged_ok]
    assert np.median(m["gcov"][14, merged_ok] / o["cov"][14, hm]) < 0.5


def test_succ_and_pred_are_reciprocal_argmins_of_the_pair_chi2(orc):
    rng = np.random.Generator(np.random.PCG64(11))
    n = 40
    t = dict(qpt=rng.choice([-1, 1], n) / rng.uniform(0.25, 1.0, n), phi=rng.uniform(0, 2 * math.pi, n),
             tanl=rng.uniform(-0.8, 0.8, n), vx=np.zeros(n), vy=np.zeros(n), vz=rng.normal(0, 5, n))
    ev = tracks_event(t, smear=True, dropout=0.02, seed=12)
    o, m = run_merge(orc, ev, "f32")
    C = m["pair_chi2"].astype(np.float64)
    K = C.shape[0]
    ok = (C >= 0) & (C < 50.0)
    big = np.where(ok, C, np.inf)
    seeds = o["trk_seed"]
    exp_succ = np.full(K, -1); exp_pred = np.full(K, -1)
    for a in range(K):
        if ok[a].any():
            best = big[a].min()
            cand = np.nonzero(big[a] == best)[0]
            exp_succ[a] = cand[np.argmin(seeds[cand])]
    for b in range(K):
        if ok[:, b].any():
            best = big[:, b].min()
            cand = np.nonzero(big[:, b] == best)[0]
            exp_pred[b] = cand[np.argmin(seeds[cand])]
    link = np.array([exp_succ[a] if exp_succ[a] >= 0 and exp_pred[exp_succ[a]] == a else -1 for a in range(K)])
    assert np.array_equal(m["succ"], link)
    back = np.full(K, -1)
    back[link[link >= 0]] = np.nonzero(link >= 0)[0]
    assert np.array_equal(m["pred"], back)
    assert (link >= 0).sum() >= 10
    # windows of R26: no pair outside 1 <= first row of b - last row of a <= max_rows has a chi2
    dr = m["row_first"][None, :] - m["row_last"][:, None]
    assert np.all(C[(dr < 1) | (dr > 12)] == -1.0)
