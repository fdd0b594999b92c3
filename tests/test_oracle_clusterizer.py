"""Pins of R27 (TPC clusterizer on digits -- peaks in (pad, time), 3 x 3 centre of gravity), -m "not gpu",
oracle only.  PAPER.md names the step (l.35, l.98) and gives no algorithm; what constrains the oracle here:
  * the definition written a second time, densely, in numpy (arrays + shifts instead of sorted cells + look-ups),
    compared cluster for cluster and bit for bit
  * hand-made cases: a plateau gives exactly one peak (the earlier cell), a missing neighbour counts as zero, two
    digits of one cell add up, peak_min; digits of ADC <= 0 change nothing, wherever they sit
  * an isolated Gaussian deposit comes back where it was put (closed form of the response: the 3-cell centre of
    gravity of a sampled Gaussian), translation by whole cells moves the clusters by whole cells
  * end to end: digits of configs[0] -> clusters -> the tracker finds the tracks it finds on the true clusters
"""
import numpy as np
import pytest

from paper_2106_03636_b200.synth import TpcParams, config0, digitize
from paper_2106_03636_b200.synth.digitizer import Digits

P1 = TpcParams(n_sectors=1, z_lo=-1.0, z_hi=251.0)
PW, TW = 0.5, 0.25


def dense_reference(p, sr, pad, time, adc, pw, tw, peak_min):
    """R27 on dense per-row arrays: returns sorted list of (sector_row, time, pad, S, y, z) with y, z in fp32."""
    out = []
    f = np.float32
    X = np.asarray(p.row_x, np.float32)
    for s in np.unique(sr):
        m = (sr == s) & (adc > 0)
        if not m.any():
            continue
        P, T = int(pad[m].max()) + 3, int(time[m].max()) + 3
        a = np.zeros((T + 2, P + 2), np.int64)                 # one cell of zeros all around
        np.add.at(a, (time[m] + 1, pad[m] + 1), adc[m])
        c = a[1:-1, 1:-1]
        peak = c >= peak_min
        S = np.zeros_like(c); Sp = np.zeros_like(c); St = np.zeros_like(c)
        for dt in (-1, 0, 1):
            for dp in (-1, 0, 1):
                b = a[1 + dt:a.shape[0] - 1 + dt, 1 + dp:a.shape[1] - 1 + dp]
                if (dt, dp) != (0, 0):
                    peak &= (c > b) if (dt < 0 or (dt == 0 and dp < 0)) else (c >= b)
                S += b; Sp += b * dp; St += b * dt
        tt, pp = np.nonzero(peak)
        r = int(s) % int(p.n_rows); sector = int(s) // int(p.n_rows)
        ymax = f(X[r] * f(p.tan_half))
        side = f(1.0) if sector < 18 else f(-1.0)
        for t0, p0 in zip(tt, pp):
            s_, sp_, st_ = S[t0, p0], Sp[t0, p0], St[t0, p0]
            y = f(f(f(f(p0) + f(0.5)) + f(f(sp_) / f(s_))) * f(pw)) - ymax
            zeta = f(f(f(f(t0) + f(0.5)) + f(f(st_) / f(s_))) * f(tw)) + f(p.z_lo)
            out.append((int(s), int(t0), int(p0), int(s_), f(y), f(side * zeta)))
    return sorted(out)


def as_tuples(c):
    return [(int(s), int(t), int(p), int(q), y, z) for s, t, p, q, y, z in
            zip(c["sector_row"], c["time"], c["pad"], c["q"], c["y"], c["z"])]


def digits_of(cells):
    """cells: list of (sector_row, pad, time, adc)."""
    a = np.array(cells, np.int32).reshape(-1, 4)
    return a[:, 0].copy(), a[:, 1].copy(), a[:, 2].copy(), a[:, 3].copy()


def test_equals_the_dense_numpy_definition(orc):
    ev = config0(seed=3, n_tracks=40)
    d = digitize(ev, seed=1)
    assert d.n > 3000
    c = orc.clusterize(ev.params, d.sector_row, d.pad, d.time, d.adc, d.pad_width, d.time_width, peak_min=6)
    ref = dense_reference(ev.params, d.sector_row, d.pad, d.time, d.adc, d.pad_width, d.time_width, 6)
    got = as_tuples(c)
    assert len(got) == len(ref) == c["n_found"] > 500
    assert got == ref, "peaks, charge sums or fp32 positions differ from the dense definition"


def test_plateau_missing_neighbours_duplicates_and_peak_min(orc):
    s = 5
    # two equal neighbours in pad at the same time: the earlier (lower pad) is the one peak
    sr, pad, tim, adc = digits_of([(s, 10, 20, 50), (s, 11, 20, 50)])
    c = orc.clusterize(P1, sr, pad, tim, adc, PW, TW, peak_min=6)
    assert as_tuples(c)[0][:4] == (s, 20, 10, 100) and c["n_found"] == 1
    # ... equal neighbours in time: the earlier time bin wins
    sr, pad, tim, adc = digits_of([(s, 10, 20, 50), (s, 10, 21, 50), (s, 11, 21, 50)])
    c = orc.clusterize(P1, sr, pad, tim, adc, PW, TW, peak_min=6)
    assert c["n_found"] == 1 and as_tuples(c)[0][:4] == (s, 20, 10, 150)
    # a lone digit at pad 0, time 0: neighbours outside the row count as zero
    sr, pad, tim, adc = digits_of([(s, 0, 0, 9)])
    c = orc.clusterize(P1, sr, pad, tim, adc, PW, TW, peak_min=6)
    assert c["n_found"] == 1 and c["q"][0] == 9.0
    ymax = np.float32(np.float32(P1.row_x[s]) * np.float32(P1.tan_half))
    assert c["y"][0] == np.float32(np.float32(0.5) * np.float32(PW)) - ymax
    assert c["z"][0] == np.float32(np.float32(0.5) * np.float32(TW)) + np.float32(P1.z_lo)
    # below peak_min: nothing; two digits of the same cell add up and pass it
    assert orc.clusterize(P1, sr, pad, tim, np.array([5], np.int32), PW, TW, peak_min=6)["n_found"] == 0
    sr, pad, tim, adc = digits_of([(s, 7, 7, 3), (s, 7, 7, 4)])
    c = orc.clusterize(P1, sr, pad, tim, adc, PW, TW, peak_min=6)
    assert c["n_found"] == 1 and c["q"][0] == 7.0
    # centre of gravity by hand: 10 at (p, t) = (4, 4), 6 at (5, 4), 2 at (4, 5): S = 18, Sp = 6, St = 2
    sr, pad, tim, adc = digits_of([(s, 4, 4, 10), (s, 5, 4, 6), (s, 4, 5, 2)])
    c = orc.clusterize(P1, sr, pad, tim, adc, PW, TW, peak_min=6)
    assert c["n_found"] == 1
    assert c["y"][0] == pytest.approx((4.5 + 6 / 18) * PW - float(ymax), abs=1e-5)
    assert c["z"][0] == pytest.approx((4.5 + 2 / 18) * TW + P1.z_lo, abs=1e-5)


def test_digits_without_charge_are_ignored(orc):
    """R27: a digit of ADC <= 0 is not a zero-suppressed digit.  By hand: a peak of 6 between two digits of -3 would have
    S = 0 (centre of gravity 0/0); with the rule it is the lone digit of the third case above.  On a digitised event:
    zero and negative digits sprinkled on empty cells, on cells next to peaks and on occupied cells leave every cluster as
    it was."""
    s = 5
    ymax = np.float32(np.float32(P1.row_x[s]) * np.float32(P1.tan_half))
    sr, pad, tim, adc = digits_of([(s, 10, 20, 6), (s, 9, 20, -3), (s, 11, 20, -3), (s, 10, 21, 0)])
    c = orc.clusterize(P1, sr, pad, tim, adc, PW, TW, peak_min=6)
    assert c["n_found"] == 1 and as_tuples(c)[0][:4] == (s, 20, 10, 6)
    assert c["y"][0] == np.float32(np.float32(10.5) * np.float32(PW)) - ymax
    assert c["z"][0] == np.float32(np.float32(20.5) * np.float32(TW)) + np.float32(P1.z_lo)
    # a negative digit on an occupied cell does not lower it: 4 + (-2) stays a peak of 4 (= peak_min), 7 + (-5) one of 7
    sr, pad, tim, adc = digits_of([(s, 3, 3, 4), (s, 3, 3, -2), (s, 30, 30, 7), (s, 30, 30, -5)])
    c = orc.clusterize(P1, sr, pad, tim, adc, PW, TW, peak_min=4)
    assert c["n_found"] == 2 and sorted(c["q"].tolist()) == [4.0, 7.0]
    ev = config0()
    d = digitize(ev)
    base = orc.clusterize(ev.params, d.sector_row, d.pad, d.time, d.adc, d.pad_width, d.time_width)
    rng = np.random.default_rng(27)
    k = rng.integers(0, d.sector_row.size, 5000)
    extra_sr = d.sector_row[k]
    extra_pad = np.clip(d.pad[k] + rng.integers(-1, 2, k.size), 0, 65535).astype(np.int32)
    extra_time = np.clip(d.time[k] + rng.integers(-1, 2, k.size), 0, None).astype(np.int32)
    extra_adc = rng.integers(-40, 1, k.size).astype(np.int32)
    cat = lambda a, b: np.concatenate([a, b]).astype(np.int32)
    more = orc.clusterize(ev.params, cat(d.sector_row, extra_sr), cat(d.pad, extra_pad), cat(d.time, extra_time),
                          cat(d.adc, extra_adc), d.pad_width, d.time_width)
    assert more["n_found"] == base["n_found"] > 1000
    for key in ("y", "z", "q", "sector_row", "pad", "time"):
        assert np.array_equal(more[key], base[key]), key
    assert np.isfinite(more["y"]).all() and np.isfinite(more["z"]).all()


def test_isolated_deposit_comes_back_and_whole_cell_shifts(orc):
    """One cluster of charge 5000 at 25 sub-cell positions: the reconstructed position is the 3-cell centre of gravity
    of the sampled Gaussian response, within ADC truncation (1 / peak ADC) -- and within 0.06 cells of the truth."""
    from types import SimpleNamespace
    row = 40
    X = np.asarray(P1.row_x, np.float64)
    ymax = X[row] * float(P1.tan_half)
    sp, st = 0.45, 0.55
    for fu in (0.1, 0.3, 0.5, 0.7, 0.9):
        for fv in (0.05, 0.35, 0.5, 0.65, 0.95):
            u, v = 30 + fu, 200 + fv
            ev = SimpleNamespace(params=P1, sector_row=np.array([row], np.int32),
                                 y=np.array([u * PW - ymax], np.float32), z=np.array([v * TW + P1.z_lo], np.float32),
                                 q=np.array([5000.0], np.float32))
            d = digitize(ev, PW, TW, sp, st, threshold=1, shuffle=False)
            c = orc.clusterize(P1, d.sector_row, d.pad, d.time, d.adc, PW, TW, peak_min=6)
            assert c["n_found"] == 1
            # expected: centre of gravity of the response sampled at the 3 cell centres around the peak cell
            p0, t0 = int(np.floor(u)), int(np.floor(v))
            wp = np.exp(-0.5 * ((p0 + np.arange(-1, 2) + 0.5 - u) / sp) ** 2)
            wt = np.exp(-0.5 * ((t0 + np.arange(-1, 2) + 0.5 - v) / st) ** 2)
            u_exp = p0 + 0.5 + (wp * np.arange(-1, 2)).sum() / wp.sum()
            v_exp = t0 + 0.5 + (wt * np.arange(-1, 2)).sum() / wt.sum()
            u_rec = (float(c["y"][0]) + ymax) / PW
            v_rec = (float(c["z"][0]) - P1.z_lo) / TW
            assert abs(u_rec - u_exp) < 0.01 and abs(v_rec - v_exp) < 0.01
            assert abs(u_rec - u) < 0.06 and abs(v_rec - v) < 0.08
    # translation by whole cells: same peaks and charges, positions moved by whole cells
    ev = config0(seed=4, n_tracks=10)
    d = digitize(ev, seed=2)
    a = orc.clusterize(ev.params, d.sector_row, d.pad, d.time, d.adc, PW, TW)
    b = orc.clusterize(ev.params, d.sector_row, d.pad + 3, d.time + 7, d.adc, PW, TW)
    assert np.array_equal(a["pad"] + 3, b["pad"]) and np.array_equal(a["time"] + 7, b["time"]) and np.array_equal(a["q"], b["q"])
    np.testing.assert_allclose(b["y"] - a["y"], 3 * PW, atol=2e-5)
    np.testing.assert_allclose(b["z"] - a["z"], 7 * TW, atol=2e-4)


def test_tracks_from_digits_are_the_tracks_from_clusters(orc):
    ev = config0()
    d = digitize(ev)
    c = orc.clusterize(ev.params, d.sector_row, d.pad, d.time, d.adc, d.pad_width, d.time_width)
    assert 0.95 * ev.n <= c["n_found"] <= ev.n, "nearly every deposit is a cluster again (close pairs merge)"
    o_true = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)
    o_dig = orc.run(ev.params, c["y"], c["z"], c["sector_row"], "f32", True)
    assert o_dig["trk_seed"].size >= 0.95 * o_true["trk_seed"].size
    assert (o_dig["cluster_track"] >= 0).sum() >= 0.93 * (o_true["cluster_track"] >= 0).sum()
    # resolution: the reconstructed cluster nearest to a true one (same row) is within a third of a pad for 95 %
    near = []
    for r in np.unique(ev.sector_row):
        a = np.nonzero(ev.sector_row == r)[0]; b = np.nonzero(c["sector_row"] == r)[0]
        if b.size:
            dd = np.hypot(c["y"][b][None, :] - ev.y[a][:, None], c["z"][b][None, :] - ev.z[a][:, None])
            near.append(dd.min(axis=1))
    near = np.concatenate(near)
    assert np.quantile(near, 0.95) < PW / 3
