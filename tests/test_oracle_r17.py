"""Pins of R17 as the oracle implements it (R17: phases and waves), -m "not gpu", oracle only.

PAPER.md fixes nothing here (l.47 only says the tracker derives from the Run-2 HLT tracker), so R17 is a reading,
and these tests are what constrains it: every expected value below is derived BY HAND from the text of R17 on
hand-built straight-line inputs (a straight line is a helix of q/pT = 0), never from a run of the oracle or of
the CUDA path.  The R17 `mode` argument of the oracle (0 = every start hit followed in full, as SURVEY.md §8(c)
R17 first read; 1 = phases; 2 = phases + waves, the method the CUDA path implements) lets the amended reading be
measured against the original one.

Which pin constrains which line of the oracle (oracle/tpc_oracle.cpp):

  Follower::has_predecessor (the wave test, R17 (i))
    slopes my, mz from (h1, h0) and the minus sign of the backward line ... test_wave_test_follows_the_backward_line
    k runs to max_gap + 3 (not + 2, not + 4) .............................. test_wave_test_row_range
    `r < 0` stops the scan ................................................. test_wave_test_start_hit_on_row_one
    |dy| <= 4 sigma_y (k+1) and |dz| <= 4 sigma_z (k+1), both, inclusive .... test_wave_test_tolerance_edges
    only clusters with up' == -2 count (not -1, not >= 0) ................... test_wave_test_row_range (g = max_gap+1:
                                                                              an unlinked cluster sits in the window),
                                                                              test_wave_test_ignores_chain_middles
    same sector only ....................................................... test_wave_test_is_sector_local
    grid and brute-force back ends agree (R8) .............................. every wave-test pin runs both
  follow_impl (the wave loop, R17 (ii)-(iv))
    first wave = the start hits that do not wait; a waiting start hit that an upward leg of the first wave marked
    never runs and is absorbed ............................................. test_R17_clean_fragments
    second wave = waiting and unmarked start hits, and they are followed in full ("a wrong wait costs only time")
                                                                              test_R17_wrong_wait_runs_in_second_wave
    the list of a wave is fixed before the wave runs; marks made in the second wave absorb too
                                                                              test_R17_marks_of_the_second_wave_absorb
    a start hit that ran in the first wave and was marked in the same wave is absorbed, and its own marks stand
                                                                              test_R17_ran_and_marked_in_the_same_wave
    whether a fragment ran decides the fate of the next one (wait vs no wait: mode 2 vs mode 1)
                                                                              test_R17_kinked_track_three_fragments
    failure mode: the picker dies right after the start hit it attached -> the upper part of that track is lost
                                                                              test_R17_failure_mode_picker_dies,
                                                                              test_R17_modes_physics (bounds how often)
  physics cost of the amended reading (R17 table) ................. test_R17_modes_physics
  the oracle's output on configs[0] is the stored summary ................... test_config0_reproduces_golden_summary
"""
import hashlib
import os

import numpy as np
import pytest

from paper_2106_03636_b200.synth import TpcParams, config0, config1, config3, default_row_x

from truth_metrics import physics_summary

ROWX = default_row_x().astype(np.float64)
NR = 152
P1 = TpcParams(n_sectors=1, z_lo=-1.0, z_hi=251.0, cell_y=2.0, cell_z=5.5)
P36 = TpcParams(n_sectors=36, z_lo=-1.0, z_hi=251.0, cell_y=2.0, cell_z=5.5)
SIG_Y, SIG_Z = float(P1.sigma_y), float(P1.sigma_z)
MAX_GAP = int(P1.max_gap)
MY, MZ = 0.1, 0.3            # slopes dy/dx, dz/dx of the default line


def line(rows, r_ref, y_ref, z_ref, my=MY, mz=MZ, sector=0):
    """Clusters of a straight line through (ROWX[r_ref], y_ref, z_ref) on the given pad rows."""
    rows = np.asarray(list(rows))
    dx = ROWX[rows] - ROWX[r_ref]
    return rows + NR * sector, y_ref + my * dx, z_ref + mz * dx


def build(parts):
    sr = np.concatenate([p[0] for p in parts]).astype(np.int32)
    return np.concatenate([p[1] for p in parts]), np.concatenate([p[2] for p in parts]), sr


def waits_by_row(orc, P, y, z, sr, grid):
    """{row of the start hit: waits?}"""
    up, dn = orc.neighbours(P, y, z, sr, "f64", grid)
    up_c, _, starts = orc.links(up, dn)
    w = orc.wave_test(P, y, z, sr, up_c, starts, "f64", grid)
    return {int(sr[s]) % NR: bool(v) for s, v in zip(starts, w)}


def two_fragments(gap, dy=0.0, dz=0.0, my=MY, mz=MZ, last_lower=50):
    """Lower fragment rows 10..last_lower, `gap` missing rows, upper fragment of 25 rows displaced by (dy, dz).
    R9: the last cluster of the lower fragment and the first of the upper one have no (up, down) pair, hence no
    links: the lower chain's top (up' = -2) is on row last_lower - 1, the upper start hit on row first_upper + 1,
    i.e. gap + 3 rows above it.  Returns (y, z, sr, row of the upper start hit)."""
    first_upper = last_lower + gap + 1
    lower = line(range(10, last_lower + 1), 10, 5.0, 50.0, my, mz)
    upper = line(range(first_upper, first_upper + 25), 10, 5.0 + dy, 50.0 + dz, my, mz)
    return (*build([lower, upper]), first_upper + 1)


# ---------------------------------------------------------------------------------------------------------
# the wave test (Follower::has_predecessor)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("grid", [True, False])
def test_wave_test_row_range(orc, grid):
    """R17 (i): k = 1 .. max_gap + 3.  g missing rows put the lower chain's top g + 3 rows below the start hit, so
    every gap an upward leg can bridge (g <= max_gap) makes the upper start hit wait, and g = max_gap + 1 does not:
    there the row at k = max_gap + 3 holds the lower fragment's LAST cluster, exactly on the line but without links
    (up' = -1, not a chain top), and the chain top is one row out of range."""
    for g in range(1, MAX_GAP + 3):
        y, z, sr, r0 = two_fragments(g)
        w = waits_by_row(orc, P1, y, z, sr, grid)
        assert w[11] is False, "the lowest fragment has nothing below it"
        assert w[r0] is (g <= MAX_GAP), f"gap of {g} rows: chain top {g + 3} rows below the start hit"


@pytest.mark.parametrize("grid", [True, False])
def test_wave_test_tolerance_edges(orc, grid):
    """|dy| <= 4 sigma_y (k + 1) and |dz| <= 4 sigma_z (k + 1): a fragment displaced parallel to the lower one by d has
    its backward line pass the chain top at distance d exactly; inside by 1e-9 relative -> waits, outside -> not."""
    g = 2
    k = g + 3
    ty, tz = 4.0 * SIG_Y * (k + 1), 4.0 * SIG_Z * (k + 1)
    for sgn in (1.0, -1.0):
        for name, tol in (("dy", ty), ("dz", tz)):
            inside = two_fragments(g, **{name: sgn * tol * (1 - 1e-9)})
            outside = two_fragments(g, **{name: sgn * tol * (1 + 1e-9)})
            assert waits_by_row(orc, P1, *inside[:3], grid)[inside[3]] is True, (name, sgn)
            assert waits_by_row(orc, P1, *outside[:3], grid)[outside[3]] is False, (name, sgn)
    # both conditions must hold: well inside in y, just outside in z
    y, z, sr, r0 = two_fragments(g, dy=0.5 * ty, dz=tz * (1 + 1e-9))
    assert waits_by_row(orc, P1, y, z, sr, grid)[r0] is False
    # the tolerance grows with k: a displacement that fails at k = 5 passes at k = 7 (g = 4)
    y, z, sr, r0 = two_fragments(MAX_GAP, dy=ty * 1.2)
    assert waits_by_row(orc, P1, y, z, sr, grid)[r0] is True


@pytest.mark.parametrize("grid", [True, False])
def test_wave_test_follows_the_backward_line(orc, grid):
    """The prediction on row r0 - k is the straight line through the start hit and its up-neighbour, continued
    backwards.  With steep slopes a mirrored or slope-less prediction misses by centimetres: at k = 7 (7.4 cm) the
    slopes 0.5 / -0.9 move the line by 3.7 / 6.7 cm, the tolerances are 2.56 / 3.2 cm."""
    y, z, sr, r0 = two_fragments(MAX_GAP, my=0.5, mz=-0.9)
    assert waits_by_row(orc, P1, y, z, sr, grid)[r0] is True
    # and a lower chain that lies on the MIRRORED line (slopes of opposite sign through the start hit) is not seen
    upper = line(range(60, 85), 61, 0.0, 100.0, 0.5, -0.9)
    mirrored = line(range(30, 56), 61, 0.0, 100.0, -0.5, 0.9)
    y, z, sr = build([mirrored, upper])
    w = waits_by_row(orc, P1, y, z, sr, grid)
    assert w[61] is False


@pytest.mark.parametrize("grid", [True, False])
def test_wave_test_ignores_chain_middles(orc, grid):
    """A cluster inside the window only counts if it is the TOP of a chain (up' == -2).  Another track crossing the
    backward line k rows below the start hit puts linked clusters (up' >= 0) right on the prediction."""
    upper = line(range(60, 85), 60, 0.0, 100.0)
    for k in (3, 5):
        xr = 61 - k
        yx = 0.0 + MY * (ROWX[xr] - ROWX[60])
        zx = 100.0 + MZ * (ROWX[xr] - ROWX[60])
        crossing = line(range(xr - 15, xr + 12), xr, yx, zx, MY + 1.0, MZ)     # its own top is 10 rows above
        y, z, sr = build([upper, crossing])
        w = waits_by_row(orc, P1, y, z, sr, grid)
        assert w[61] is False, f"crossing chain at k = {k}"


@pytest.mark.parametrize("grid", [True, False])
def test_wave_test_is_sector_local(orc, grid):
    lower1 = line(range(10, 51), 10, 5.0, 50.0, sector=1)
    lower0 = line(range(10, 51), 10, 5.0, 50.0, sector=0)
    upper0 = line(range(53, 78), 10, 5.0, 50.0, sector=0)
    y, z, sr = build([lower1, upper0])
    assert waits_by_row(orc, P36, y, z, sr, grid)[54] is False, "same local coordinates, other sector"
    y, z, sr = build([lower0, upper0])
    assert waits_by_row(orc, P36, y, z, sr, grid)[54] is True


@pytest.mark.parametrize("grid", [True, False])
def test_wave_test_start_hit_on_row_one(orc, grid):
    y, z, sr = build([line(range(0, 25), 0, 5.0, 50.0)])
    assert waits_by_row(orc, P1, y, z, sr, grid) == {1: False}, "nothing below row 0 to look at"


# ---------------------------------------------------------------------------------------------------------
# the wave loop (follow_impl)
# ---------------------------------------------------------------------------------------------------------
def run_modes(orc, P, y, z, sr):
    """mode -> (rows of the start hits ascending, ran, n_hits, {seed row: set of cluster indices}) ."""
    out = {}
    for mode in (orc.R17_NAIVE, orc.R17_PHASES, orc.R17_WAVES):
        o = orc.run(P, y, z, sr, "f64", True, r17_mode=mode)
        order = np.argsort(sr[o["starts"]])
        tracks = {}
        for k in range(o["trk_seed"].size):
            a = int(o["trk_first_hit"][k])
            tracks[int(sr[o["trk_seed"][k]]) % NR] = set(o["trk_hits"][a:a + int(o["trk_nhits"][k])].tolist())
        out[mode] = ((sr[o["starts"]][order] % NR).tolist(), o["ran"][order].astype(int).tolist(),
                     o["n_hits"][order].tolist(), tracks, o)
    return out


def idx_of_rows(sr, rows):
    return set(np.nonzero(np.isin(sr % NR, list(rows)))[0].tolist())


def test_R17_clean_fragments(orc):
    """Three fragments of one straight track, gaps of 2 and 3 rows.  R17: the upper two wait (i); the first wave is
    the lowest alone (ii), its upward leg bridges both gaps and marks both upper start hits; nobody is left for
    the second wave (iii); the upper two are absorbed without ever running (iv).  One track with every cluster --
    in every mode (in mode 0 the three tracklets cover the same clusters and R20 keeps the lowest start index)."""
    A, B, C = line(range(10, 51), 10, 5.0, 50.0), line(range(53, 101), 10, 5.0, 50.0), line(range(104, 140), 10, 5.0, 50.0)
    y, z, sr = build([A, B, C])
    res = run_modes(orc, P1, y, z, sr)
    n = y.size
    assert res[2][0] == [11, 54, 105]
    assert res[2][1] == [1, 0, 0] and res[2][2] == [n, 0, 0]
    assert res[1][1] == [1, 1, 1] and res[1][2] == [n, 0, 0]
    assert res[0][1] == [1, 1, 1] and res[0][2] == [n, n, n]
    for mode in (0, 1, 2):
        assert list(res[mode][3].keys()) == [11] and len(res[mode][3][11]) == n


def test_R16_leg_bridges_max_gap_missing_rows_and_no_more(orc):
    """R16: a leg goes on over rows without a hit and stops after max_gap + 1 of them in a row -- max_gap is the longest
    hole that is bridged.  Mode 0 (every start hit followed in full, nothing absorbed), a straight line in two
    fragments: with exactly max_gap missing rows the lower tracklet's upward leg (and the upper one's downward leg)
    crosses the hole and both record every cluster; with max_gap + 1 both stop at the hole and each keeps its own
    fragment.  (The wave test has its own pin at the same boundary; this is the leg that does the bridging.)"""
    for g, bridged in ((MAX_GAP - 1, True), (MAX_GAP, True), (MAX_GAP + 1, False), (MAX_GAP + 2, False)):
        y, z, sr, r_up = two_fragments(g)
        n_lo, n_up = 41, 25
        assert y.size == n_lo + n_up
        rows, ran, n_hits, tracks, o = run_modes(orc, P1, y, z, sr)[orc.R17_NAIVE]
        assert rows == [11, r_up] and ran == [1, 1]
        assert n_hits == ([n_lo + n_up] * 2 if bridged else [n_lo, n_up]), f"{g} missing rows"
        if bridged:
            assert list(tracks.keys()) == [11] and len(tracks[11]) == n_lo + n_up
        else:
            assert tracks == {11: set(range(n_lo)), r_up: set(range(n_lo, n_lo + n_up))}


def stub_below(row_top, dy):
    """A 16-cluster chain whose top sits on row `row_top`, `dy` cm beside the default line through (row 60, 0, 100),
    and which runs off at a very different angle (slope + 0.6): a plausible-looking predecessor that is none."""
    yt = 0.0 + MY * (ROWX[row_top] - ROWX[60]) + dy
    zt = 100.0 + MZ * (ROWX[row_top] - ROWX[60])
    return line(range(row_top - 14, row_top + 2), row_top, yt, zt, MY + 0.6, MZ)


def test_R17_wrong_wait_runs_in_second_wave(orc):
    """The top of an unrelated chain lies 1.5 cm beside the backward line, 7 rows below the start hit of track U
    (tolerance there: 2.56 cm): U waits.  The stub's own upward leg extrapolates 0.6 * 7.4 cm = 4.4 cm further away
    and cannot attach U's clusters, so U is unmarked after the first wave and is followed in full in the second:
    the result is the one of mode 0 and mode 1."""
    U, S = line(range(60, 100), 60, 0.0, 100.0), stub_below(54, 1.5)
    y, z, sr = build([S, U])
    res = run_modes(orc, P1, y, z, sr)
    up, dn = orc.neighbours(P1, y, z, sr, "f64")
    up_c, _, starts = orc.links(up, dn)
    w = dict(zip((sr[starts] % NR).tolist(), orc.wave_test(P1, y, z, sr, up_c, starts, "f64").tolist()))
    assert w == {41: False, 61: True}
    assert res[2][1] == [1, 1] and res[2][2] == [16, 40]
    want = {41: idx_of_rows(sr, range(40, 56)) - idx_of_rows(sr, range(60, 100)), 61: set(range(16, 56))}
    for mode in (0, 1, 2):
        assert res[mode][3] == want, f"mode {mode}"


def test_R17_marks_of_the_second_wave_absorb(orc):
    """Stub S, then track fragments B and C (gap of 3 rows).  B waits because of S, C waits because of B.  First wave:
    S alone, marks nothing.  The second wave's list is fixed before it runs: B and C, both unmarked at that point,
    so BOTH run phase A; B's upward leg marks C's start hit during that wave, and (iv) looks at the marks after
    both waves: C is absorbed although it ran.  One track B + C."""
    S, B, C = stub_below(54, 1.5), line(range(60, 100), 60, 0.0, 100.0), line(range(103, 140), 60, 0.0, 100.0)
    y, z, sr = build([S, B, C])
    res = run_modes(orc, P1, y, z, sr)
    assert res[2][0] == [41, 61, 104]
    assert res[2][1] == [1, 1, 1], "C is on the second wave's list: B had not run when the list was made"
    assert res[2][2] == [16, 77, 0]
    assert res[2][3][61] == set(range(16, 16 + 77)) and 104 not in res[2][3]


def test_R17_ran_and_marked_in_the_same_wave(orc):
    """Track A B C.  Row 41 of A is missing and rows 42, 43 hold two linkless clusters, so A's chain top is on row 39,
    9 rows below B's start hit (row 48): out of the wave test's range, B does NOT wait -- but A's upward leg does
    reach it (misses on rows 41 and 44-46 only).  First wave = {A, B}: B runs phase A and marks C (C waited: B's top
    is 5 rows below it) whichever of the two is processed first, and B, marked by A in the same wave, is absorbed.
    C never runs.  One track with every cluster."""
    A = line([r for r in range(10, 44) if r != 41], 10, 5.0, 50.0)
    B, C = line(range(47, 80), 10, 5.0, 50.0), line(range(83, 120), 10, 5.0, 50.0)
    y, z, sr = build([A, B, C])
    res = run_modes(orc, P1, y, z, sr)
    n = y.size
    assert res[2][0] == [11, 48, 84]
    assert res[2][1] == [1, 1, 0] and res[2][2] == [n, 0, 0]
    assert list(res[2][3].keys()) == [11] and len(res[2][3][11]) == n


def kinked(with_C):
    """A: rows 10..50 on line L1.  B: rows 53..56 on L1, then bends by 0.3 in dy/dx at row 56 and continues to row
    100 on L2.  C (optional): rows 104..139 on L2.  A fit that has 40 clusters of L1 behind it cannot follow the bend
    (0.32 cm per row against sigma_y = 0.08: chi2 > 16 from the second row on); a fit that starts inside B can.
    (y = -12 cm at row 10 keeps L2 inside the sector up to the last row.)"""
    A = line(range(10, 51), 10, -12.0, 50.0)
    Bl = line(range(53, 57), 10, -12.0, 50.0)
    yk, zk = -12.0 + MY * (ROWX[56] - ROWX[10]), 50.0 + MZ * (ROWX[56] - ROWX[10])
    Bu = line(range(57, 101), 56, yk, zk, MY + 0.3, MZ)
    parts = [A, Bl, Bu] + ([line(range(104, 140), 56, yk, zk, MY + 0.3, MZ)] if with_C else [])
    return build(parts)


def test_R17_kinked_track_three_fragments(orc):
    """Whether B runs decides what happens to C.  R17 by hand:
    mode 2: B and C wait.  First wave = A: its upward leg attaches B's first clusters including B's start hit (row
      54, marked) and dies at the bend.  Second wave: B is marked -> does not run, so nobody marks C; C is unmarked ->
      runs.  B is absorbed; C's downward leg walks down L2 and collects B's upper part.  Two tracks: A + B's L1 part,
      C + B's L2 part.
    mode 1 (no waiting): all three run phase A; B's upward leg marks C, A's marks B; B and C are both absorbed and
      everything above the bend is lost: one track.
    mode 0: B is followed in full and owns B + C."""
    y, z, sr = kinked(True)
    res = run_modes(orc, P1, y, z, sr)
    # rows 55..57, next to the bend, are within chi2 < 16 of both lines: R20 gives them to the longer track
    A_rows, B_low, B_up, C_rows = range(10, 51), range(53, 55), range(58, 101), range(104, 140)
    assert res[2][0] == [11, 54, 105]
    assert res[2][1] == [1, 0, 1] and res[2][2][1] == 0
    t2 = res[2][3]
    assert set(t2.keys()) == {11, 105}
    assert idx_of_rows(sr, A_rows) | idx_of_rows(sr, B_low) <= t2[11]
    assert idx_of_rows(sr, C_rows) | idx_of_rows(sr, B_up) <= t2[105]
    assert len(t2[11] | t2[105]) == y.size and not (t2[11] & t2[105]), "every cluster in exactly one of the two"
    t1 = res[1][3]
    assert res[1][1] == [1, 1, 1] and res[1][2][1:] == [0, 0]
    assert set(t1.keys()) == {11} and not (t1[11] & (idx_of_rows(sr, C_rows) | idx_of_rows(sr, B_up)))
    t0 = res[0][3]
    assert idx_of_rows(sr, C_rows) | idx_of_rows(sr, B_up) <= t0[54] and idx_of_rows(sr, A_rows) <= t0[11]


def test_R17_failure_mode_picker_dies(orc):
    """The cost of absorption, stated: an upward leg that attaches another fragment's start hit and then dies takes
    that fragment out of the game.  Same kinked track without C: in modes 1 and 2 everything above the bend (44
    clusters) is in no track; mode 0 finds it.  test_R17_modes_physics bounds how often this happens."""
    y, z, sr = kinked(False)
    res = run_modes(orc, P1, y, z, sr)
    upper = idx_of_rows(sr, range(58, 101))
    assert upper <= res[0][3][54]
    for mode in (1, 2):
        assert set(res[mode][3].keys()) == {11}
        assert not (res[mode][3][11] & upper)
        assert int(np.count_nonzero(res[mode][4]["cluster_track"] < 0)) >= len(upper)


# ---------------------------------------------------------------------------------------------------------
# physics cost of the amended reading, measured (R17 quotes exactly these numbers)
# ---------------------------------------------------------------------------------------------------------
R17_EVENTS = {"c0": lambda: config0(), "c1_1500": lambda: config1(n_tracks=1500),
              "c3_2x800": lambda: config3(n_coll=2, n_tracks=800)}


@pytest.mark.parametrize("name", list(R17_EVENTS))
def test_R17_modes_physics(orc, name):
    ev = R17_EVENTS[name]()
    s, o = {}, {}
    for mode in (0, 1, 2):
        o[mode] = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True, r17_mode=mode)
        s[mode] = physics_summary(ev, o[mode])
        s[mode]["ran_A"] = int(o[mode]["ran"].sum())
        s[mode]["ran_B"] = int(np.count_nonzero(o[mode]["n_hits"] > 0))
    a0, a2 = o[0]["cluster_track"] >= 0, o[2]["cluster_track"] >= 0
    lost, gained = int(np.count_nonzero(a0 & ~a2)), int(np.count_nonzero(a2 & ~a0))
    print(f"\nR17 {name}: n = {ev.n}, start hits = {o[0]['starts'].size}, clusters lost / gained by mode 2 vs 0: {lost} / {gained}")
    for mode in (0, 1, 2):
        print(f"  mode {mode}: " + ", ".join(f"{k} {v:.5f}" if isinstance(v, float) else f"{k} {v}" for k, v in s[mode].items()))
    n_starts = o[0]["starts"].size
    # what the amended reading may cost: nothing visible in tracks, efficiency, attachment; no fakes
    assert abs(s[2]["tracks"] - s[0]["tracks"]) <= max(2, 0.001 * s[0]["tracks"])
    assert s[2]["found"] >= s[0]["found"] - max(1, round(0.001 * s[0]["findable"]))
    assert s[2]["attached"] >= s[0]["attached"] - 0.0025
    assert s[2]["fakes"] <= s[0]["fakes"] and s[2]["duplicates"] <= s[0]["duplicates"]
    assert lost <= 0.002 * int(a0.sum()), "clusters in a track in mode 0 and in none in mode 2 (failure mode above)"
    # what it buys: fewer than half of the start hits are followed at all (mode 0 follows every one of them twice over)
    assert s[0]["ran_A"] == s[0]["ran_B"] == n_starts and s[1]["ran_A"] == n_starts
    if name != "c0":
        assert s[2]["ran_A"] <= 0.5 * n_starts and s[2]["ran_B"] <= 0.5 * n_starts
    # the waves themselves (mode 2 vs mode 1) do not lose anything against plain phases
    assert s[2]["found"] >= s[1]["found"] and s[2]["assigned"] >= s[1]["assigned"] - 2


# ---------------------------------------------------------------------------------------------------------
# the stored summary of configs[0] (tests/golden/, written by make_config0_summary.py from the oracle alone)
# ---------------------------------------------------------------------------------------------------------
def test_config0_reproduces_golden_summary(orc):
    """A silent change of the oracle's arithmetic shows up here, on the CPU, not only in the GPU run that reads the
    same file (tests/test_gpu_parity.py::test_config0_golden_counts)."""
    ev = config0()
    o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)
    want = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "config0_oracle_summary.txt")) as f:
        for ln in f:
            if not ln.startswith("#") and ln.strip():
                k, v = ln.split()
                want[k] = v
    seeds = np.where(o["cluster_track"] >= 0, o["trk_seed"][np.maximum(o["cluster_track"], 0)], -1).astype(np.int32)
    got = {"n_clusters": str(ev.n), "n_start_hits": str(o["starts"].size), "n_tracks": str(o["trk_seed"].size),
           "n_assigned": str(int((o["cluster_track"] >= 0).sum())), "sum_trk_nhits": str(int(o["trk_nhits"].sum())),
           "sha256_cluster_seed": hashlib.sha256(seeds.tobytes()).hexdigest()}
    assert got == want
