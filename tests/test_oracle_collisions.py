"""Pins of the oracle's R25 (collisions from per-track time offsets, R25) against what the definition and
statistics fix, none re-using the oracle's code path:
  * well-separated Gaussian bunches of t0 at known times are each found exactly once, with the bunch mean as time
    and every bunch member assigned to it;
  * the histogram definition written out with numpy primitives (np.histogram / np.convolve) gives the same peaks;
  * shifting all times by a whole number of bins shifts the collisions and changes nothing else;
  * unused tracks (NaN, displaced, out of range) are ignored and unassigned; too few tracks make no collision.
"""
import numpy as np
import pytest


def _bunches(rng, times, n, sigma=1.9):
    t = np.concatenate([rng.normal(c, sigma, n) for c in times]).astype(np.float32)
    lab = np.repeat(np.arange(len(times)), n)
    return t, lab


def test_R25_separated_bunches_found_once_with_their_mean(orc):
    rng = np.random.default_rng(25)
    times = np.array([40.0, 95.0, 131.0, 300.0, 555.5, 900.0])
    t, lab = _bunches(rng, times, 80)
    r = orc.collisions(t, np.zeros_like(t), 0.0, 1000.0)
    assert r["coll_time"].size == times.size
    assert np.all(np.diff(r["coll_time"]) > 0)
    for c, tc in enumerate(times):
        assert abs(r["coll_time"][c] - tc) < 4 * 1.9 / np.sqrt(60)       # mean of >= 60 members, 4 sigma
        members = r["trk_collision"][lab == c]
        assert np.count_nonzero(members == c) >= 76                      # within 5 bins = 2.6 sigma: >= 95 % of 80
        assert np.all((members == c) | (members == -1))
    assert np.all((r["coll_ntracks"] > 50) & (r["coll_ntracks"] <= 80))


def test_R25_equals_the_definition_written_with_numpy(orc):
    rng = np.random.default_rng(26)
    t = np.concatenate([rng.uniform(0, 400, 300), rng.normal(120.0, 1.9, 40), rng.normal(127.0, 1.9, 25),
                        rng.normal(250.3, 1.9, 12)]).astype(np.float32)
    dca = rng.uniform(0, 4, t.size).astype(np.float32)
    r = orc.collisions(t, dca, 0.0, 400.0, w=1.0, dca_max=3.0, n_min=5)
    use = dca <= 3.0
    h, _ = np.histogram(t[use].astype(np.float64), bins=400, range=(0.0, 400.0))
    s = np.convolve(h, np.ones(5, int), mode="same")
    sp = np.concatenate([np.zeros(3, int), s, np.zeros(3, int)])
    peaks = [b for b in range(400) if s[b] >= 5 and all(s[b] > sp[b + 3 - j] and s[b] >= sp[b + 3 + j] for j in (1, 2, 3))]
    assert list(r["coll_bin"]) == peaks and len(peaks) >= 3
    assert list(r["coll_ntracks"]) == [int(s[b]) for b in peaks]
    for c, b in enumerate(peaks):
        m = use & (np.floor(t.astype(np.float64)) >= b - 2) & (np.floor(t.astype(np.float64)) <= b + 2)
        assert r["coll_time"][c] == pytest.approx(t[m].astype(np.float64).mean(), abs=2e-3)   # 1/1024 us quantisation
    assert np.all(r["trk_collision"][~use] == -1)


def test_R25_shift_by_whole_bins(orc):
    rng = np.random.default_rng(27)
    t, _ = _bunches(rng, [50.0, 70.0, 200.0], 40)
    t = np.round(t * 64) / 64          # exact in fp32 after the shift
    a = orc.collisions(t, np.zeros_like(t), 0.0, 300.0)
    b = orc.collisions((t + 37.0).astype(np.float32), np.zeros_like(t), 0.0, 337.0)
    assert np.array_equal(a["coll_bin"] + 37, b["coll_bin"])
    assert np.array_equal(a["coll_ntracks"], b["coll_ntracks"]) and np.array_equal(a["trk_collision"], b["trk_collision"])
    assert np.allclose(a["coll_time"] + 37.0, b["coll_time"], atol=1e-4)


def test_R25_ignores_unusable_tracks_and_small_groups(orc):
    t = np.array([10.0, 10.2, 10.4, 9.9, np.nan, 500.0, -3.0, 10.1], np.float32)      # 4 usable near 10 + one displaced
    dca = np.array([0, 0, 0, 0, 0, 0, 0, 9.0], np.float32)
    r = orc.collisions(t, dca, 0.0, 100.0, n_min=5)
    assert r["coll_time"].size == 0 and np.all(r["trk_collision"] == -1)
    r = orc.collisions(t, dca, 0.0, 100.0, n_min=4)
    assert r["coll_time"].size == 1 and r["coll_ntracks"][0] == 4
    assert list(r["trk_collision"]) == [0, 0, 0, 0, -1, -1, -1, -1]


def test_R25_side_selection_separates_the_two_halves_of_a_collision(orc):
    """R5/R24: side A sees a collision at t - z_v/v_d, side C at t + z_v/v_d; clustered per side each half is one
    clean bunch, and the pair gives back t and z_v."""
    rng = np.random.default_rng(28)
    t_c, zv, vd = 200.0, 9.0, 2.58
    tA = rng.normal(t_c - zv / vd, 0.3, 60); tC = rng.normal(t_c + zv / vd, 0.3, 70)
    t = np.concatenate([tA, tC]).astype(np.float32)
    sector = np.concatenate([rng.integers(0, 18, 60), rng.integers(18, 36, 70)]).astype(np.int32)
    a = orc.collisions(t, np.zeros_like(t), 0.0, 400.0, sector=sector, side=1)
    c = orc.collisions(t, np.zeros_like(t), 0.0, 400.0, sector=sector, side=-1)
    assert a["coll_time"].size == 1 and c["coll_time"].size == 1
    assert a["coll_ntracks"][0] == 60 and c["coll_ntracks"][0] == 70
    assert np.all(a["trk_collision"][:60] == 0) and np.all(a["trk_collision"][60:] == -1)
    assert 0.5 * (a["coll_time"][0] + c["coll_time"][0]) == pytest.approx(t_c, abs=0.15)
    assert 0.5 * (c["coll_time"][0] - a["coll_time"][0]) * vd == pytest.approx(zv, abs=0.4)


# ------------------------------------------------------------------------------------------------------------
# R29: pairing of the two sides' collisions into (t, z_vertex)
# ------------------------------------------------------------------------------------------------------------
def _two_sides(rng, n_coll, rate_us, sigma_z=5.0, vd=2.58):
    t = np.cumsum(rng.exponential(rate_us, n_coll)) + 50.0
    zv = rng.normal(0.0, sigma_z, n_coll)
    mult = rng.integers(20, 400, n_coll)
    nA = rng.binomial(mult, 0.5); nC = mult - nA
    return t, zv, (t - zv / vd).astype(np.float32), nA.astype(np.int32), (t + zv / vd).astype(np.float32), nC.astype(np.int32)


def test_R29_pairs_give_back_time_and_vertex(orc):
    """Collisions 20 us apart on average (50 kHz), vertex spread 5 cm: the two halves are 2 z_v / v_d <= ~12 us apart;
    the reciprocal arg-min of (dt / sigma_t)^2 + (n_A - n_C)^2 / (n_A + n_C + 1) pairs 85 % of them correctly at this
    pile-up (every collision at a tenth of the rate), and a correct pair returns t and z_v exactly (up to fp32)."""
    rng = np.random.default_rng(40)
    t, zv, tA, nA, tC, nC = _two_sides(rng, 400, 20.0)
    permC = rng.permutation(400)                      # the C list in another order: the pairing is by value
    r = orc.pair_sides(tA, nA, tC[permC], nC[permC])
    inv = np.empty(400, np.int64); inv[permC] = np.arange(400)
    good = r["pair_of_a"] == inv
    assert good.mean() > 0.80
    t2, zv2, tA2, nA2, tC2, nC2 = _two_sides(rng, 200, 200.0)
    r2 = orc.pair_sides(tA2, nA2, tC2, nC2)
    ok2 = r2["pair_of_a"] == np.arange(200)
    assert ok2.mean() > 0.97                     # a few gaps of the Poisson process are still shorter than the window
    paired = np.nonzero(r2["pair_of_a"] >= 0)[0]
    np.testing.assert_allclose(r2["z_vertex"][ok2[paired]], zv2[paired][ok2[paired]], atol=2e-2)
    idx = np.nonzero(r["pair_of_a"] >= 0)[0]
    assert np.array_equal(r["pair_of_c"][r["pair_of_a"][idx]], idx), "the two partner tables must agree"
    ok = good[idx]
    np.testing.assert_allclose(r["t"][ok], t[idx][ok], atol=2e-3)
    np.testing.assert_allclose(r["z_vertex"][ok], zv[idx][ok], atol=5e-3)


def test_R29_is_the_reciprocal_argmin_of_the_stated_cost(orc):
    rng = np.random.default_rng(41)
    t, zv, tA, nA, tC, nC = _two_sides(rng, 120, 6.0)     # heavy pile-up: many admissible partners
    dt_max, sig = 15.5, 3.88
    r = orc.pair_sides(tA, nA, tC, nC, dt_max, sig)
    dt = tC.astype(np.float64)[None, :] - tA.astype(np.float64)[:, None]
    dn = nA.astype(np.float64)[:, None] - nC.astype(np.float64)[None, :]
    cost = (dt / sig) ** 2 + dn * dn / (nA[:, None] + nC[None, :] + 1.0)
    cost = np.where(np.abs(dt) <= dt_max, cost, np.inf)
    bc = np.where(np.isfinite(cost).any(1), cost.argmin(1), -1)
    ba = np.where(np.isfinite(cost).any(0), cost.argmin(0), -1)
    want = np.array([j if j >= 0 and ba[j] == i else -1 for i, j in enumerate(bc)])
    assert np.array_equal(r["pair_of_a"], want) and (want >= 0).sum() > 60
    # nothing outside the window is ever paired; a lone half stays unpaired
    lone = orc.pair_sides([100.0], [50], [130.0], [50])
    assert lone["pair_of_a"][0] == -1 and lone["t"].size == 0
    one = orc.pair_sides([100.0], [50], [107.0], [48])
    assert one["pair_of_a"][0] == 0 and one["t"][0] == pytest.approx(103.5) and one["z_vertex"][0] == pytest.approx(2.58 * 3.5)
