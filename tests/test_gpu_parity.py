"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, same seeded inputs.

configs[0..3] of BASELINE.json whole; configs[4] (the bench workload) on sampled sectors in
test_gpu_config4.py.  Edge cases: empty input, one cluster, clusters outside the z range, capacity overflow,
determinism (two runs bit-identical).
"""
import numpy as np
import pytest

import parity
from paper_2106_03636_b200.synth import make_config, config0

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: -m gpu tests must run on the B200 box")
    return torch


def _dev(torch, ev):
    return (torch.from_numpy(ev.y).cuda(), torch.from_numpy(ev.z).cuda(), torch.from_numpy(ev.sector_row).cuda())


def _run_both(torch, orc, ev, stages=True):
    from paper_2106_03636_b200 import binding
    o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)
    trk = binding.Tracker(ev.params, ev.n)
    y, z, sr = _dev(torch, ev)
    res = trk.run(y, z, sr)
    torch.cuda.synchronize()
    assert res["status"] == 0, f"device status bits {res['status']}"
    if stages:
        sidx, bfirst = trk.grid_export()
        parity.compare_grid(o, sidx, bfirst)
        fe = trk.find_export()
        parity.compare_links(o, fe)
        nd, nt = parity.compare_tracklets(o, fe)
        assert nd == 0, f"{nd} of {nt} tracklets differ from the oracle's row_hit tables"
    st = parity.compare_tracks(o, res, ev.n)
    print(ev.name, st)
    return o, res, st


@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_config_matches_oracle(torch_cuda, orc, cfg):
    ev = make_config(cfg)
    o, res, st = _run_both(torch_cuda, orc, ev)
    parity.assert_contract(st, exact_count=True)
    # the CUDA arithmetic restates the oracle's rounding sequence: expect identity, not just tolerance
    assert st["assign_identical"] == ev.n
    assert st["tracks_same_hits"] == st["tracks_oracle"]
    assert st["par_bit_identical"] and st["cov_bit_identical"]


def test_fit_gather_path_is_bit_identical(torch_cuda):
    """tpc_fit_tracks with workspace = NULL (self-contained gather through y/z/sector_row, any hit lists) runs the
    same arithmetic as the cached-record path tpc_find_tracks feeds: every output bit-identical."""
    from paper_2106_03636_b200 import binding
    ev = make_config(3, n_coll=2, n_tracks=1000)
    trk = binding.Tracker(ev.params, ev.n)
    a = trk.run(*_dev(torch_cuda, ev))
    for t in (trk.par, trk.cov, trk.xref, trk.zref, trk.chi2):
        t.fill_(float("nan"))
    trk.ndf.fill_(-7)
    trk.fit_tracks(gather=True)
    b = trk.results()
    assert a["trk_seed"].size > 100
    for k in ("par", "cov", "xref", "zref", "chi2", "ndf"):
        assert np.array_equal(a[k], b[k]), k


def test_row_ordered_input_matches_oracle(torch_cuda, orc):
    """Inputs ordered by (sector, row) -- the order a clusterizer delivers -- put whole warps into one grid bucket
    (the warp-aggregated atomics of the grid build); the result must equal the oracle's on the same ordering."""
    from paper_2106_03636_b200 import binding
    ev = make_config(1, n_tracks=1500)
    order = np.argsort(ev.sector_row, kind="stable")
    y, z, sr = ev.y[order].copy(), ev.z[order].copy(), ev.sector_row[order].copy()
    o = orc.run(ev.params, y, z, sr, "f32", True)
    trk = binding.Tracker(ev.params, y.size)
    res = trk.run(torch_cuda.from_numpy(y).cuda(), torch_cuda.from_numpy(z).cuda(), torch_cuda.from_numpy(sr).cuda())
    sidx, bfirst = trk.grid_export()
    parity.compare_grid(o, sidx, bfirst)
    st = parity.compare_tracks(o, res, y.size)
    parity.assert_contract(st, exact_count=True)
    assert st["assign_identical"] == y.size and st["par_bit_identical"] and st["cov_bit_identical"]


def test_max_tracklets_limit_is_an_argument_error(torch_cuda):
    from paper_2106_03636_b200 import binding
    ev = config0()
    with pytest.raises(binding.TpcError):
        binding.workspace_bytes(ev.params, ev.n, binding.TPC_MAX_TRACKLETS + 1)


def test_config0_golden_counts(torch_cuda, orc):
    """tests/golden/config0_oracle_summary.txt (written from the oracle alone) against the CUDA path."""
    import os
    gold = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "config0_oracle_summary.txt")) as f:
        for line in f:
            if not line.startswith("#"):
                k, v = line.split()
                gold[k] = v
    from paper_2106_03636_b200 import binding
    ev = config0()
    trk = binding.Tracker(ev.params, ev.n)
    res = trk.run(*_dev(torch_cuda, ev))
    assert ev.n == int(gold["n_clusters"])
    assert int(res["counters"][binding.CNT_TRACKLETS]) == int(gold["n_start_hits"])
    assert res["trk_seed"].size == int(gold["n_tracks"])
    assert int(np.count_nonzero(res["cluster_track"] >= 0)) == int(gold["n_assigned"])
    import hashlib
    cs = parity.cluster_seed(res["cluster_track"], res["trk_seed"]).astype(np.int32)
    assert hashlib.sha256(cs.tobytes()).hexdigest() == gold["sha256_cluster_seed"]


def test_deterministic_two_runs(torch_cuda):
    from paper_2106_03636_b200 import binding
    ev = make_config(1)
    trk = binding.Tracker(ev.params, ev.n)
    d = _dev(torch_cuda, ev)
    a = trk.run(*d)
    ga = trk.grid_export()
    b = trk.run(*d)
    gb = trk.grid_export()
    assert np.array_equal(ga[0], gb[0]) and np.array_equal(ga[1], gb[1])
    for k in a:
        assert np.array_equal(a[k], b[k]), k


def test_empty_and_tiny_inputs(torch_cuda, orc):
    from paper_2106_03636_b200 import binding
    torch = torch_cuda
    p = config0().params
    # n = 0
    trk = binding.Tracker(p, 0)
    e = torch.empty(0, dtype=torch.float32, device="cuda")
    res = trk.run(e, e, torch.empty(0, dtype=torch.int32, device="cuda"))
    assert res["counters"][binding.CNT_TRACKS] == 0 and res["counters"][binding.CNT_TRACKLETS] == 0
    assert res["status"] == 0
    # n = 1, n = 2 on the same row
    for n in (1, 2):
        trk = binding.Tracker(p, n)
        y = torch.zeros(n, dtype=torch.float32, device="cuda")
        z = torch.full((n,), 10.0, dtype=torch.float32, device="cuda")
        sr = torch.full((n,), 70, dtype=torch.int32, device="cuda")
        res = trk.run(y, z, sr)
        assert res["counters"][binding.CNT_TRACKS] == 0
        assert np.all(res["cluster_track"] == -1)


def test_short_tracks_below_min_hits(torch_cuda, orc):
    """A 6-row stub (< min_hits) is followed but rejected; a 30-row track is kept: ragged tail of the track list."""
    from paper_2106_03636_b200 import binding
    from paper_2106_03636_b200.synth import single_helix
    ev = single_helix(0.8, np.radians(9.0), 0.3)
    keep = (ev.sector_row % 152 < 30)
    stub = (ev.sector_row % 152 >= 100) & (ev.sector_row % 152 < 106)
    sel = keep | stub
    y, z, sr = ev.y[sel], ev.z[sel], ev.sector_row[sel]
    o = orc.run(ev.params, y, z, sr, "f32", True)
    trk = binding.Tracker(ev.params, y.size)
    res = trk.run(torch_cuda.from_numpy(y).cuda(), torch_cuda.from_numpy(z).cuda(), torch_cuda.from_numpy(sr).cuda())
    st = parity.compare_tracks(o, res, y.size)
    parity.assert_contract(st, exact_count=True)
    assert st["tracks_cuda"] == 1 and res["counters"][binding.CNT_TRACKLETS] == 2


def test_clusters_outside_z_range_are_clamped_not_lost(torch_cuda, orc):
    """z_lo/z_hi tighter than the data: edge bins absorb the outliers (status bit set), results stay exact (R8)."""
    from paper_2106_03636_b200 import binding
    ev = config0()
    p = ev.params.with_(z_lo=20.0, z_hi=180.0)
    o = orc.run(p, ev.y, ev.z, ev.sector_row, "f32", True)
    trk = binding.Tracker(p, ev.n)
    res = trk.run(*_dev(torch_cuda, ev))
    assert res["status"] & binding.ST_Z_CLAMPED
    sidx, bfirst = trk.grid_export()
    parity.compare_grid(o, sidx, bfirst)
    st = parity.compare_tracks(o, res, ev.n)
    parity.assert_contract(st, exact_count=True)
    assert st["assign_identical"] == ev.n


def test_corrupt_sector_row_is_flagged_and_ignored(torch_cuda, orc):
    """A sector_row outside [0, n_sectors * n_rows) (negative or too large) names no grid bin: the status bit is set,
    nothing is written out of bounds, those clusters stay unassigned, and everything else is tracked exactly as if
    they were not there (oracle on the valid clusters alone)."""
    from paper_2106_03636_b200 import binding
    ev = make_config(1, n_tracks=300)
    p = ev.params
    rng = np.random.Generator(np.random.PCG64(3))
    sr = ev.sector_row.copy()
    bad = rng.choice(ev.n, 37, replace=False)
    sr[bad[:12]] = -1 - rng.integers(0, 1000, 12)
    sr[bad[12:24]] = int(p.n_sectors) * int(p.n_rows) + rng.integers(0, 5000, 12)
    sr[bad[24:]] = 2**31 - 1 - rng.integers(0, 100, 13)
    trk = binding.Tracker(p, ev.n)
    t = torch_cuda
    res = trk.run(t.from_numpy(ev.y).cuda(), t.from_numpy(ev.z).cuda(), t.from_numpy(sr).cuda())
    assert res["status"] & binding.ST_BAD_ROW
    assert np.all(res["cluster_track"][bad] == -1)
    good = np.setdiff1d(np.arange(ev.n), bad)                  # ascending: index tie-breaks are preserved
    o = orc.run(p, ev.y[good], ev.z[good], ev.sector_row[good], "f32", True)
    new_of_old = np.full(ev.n, -1, np.int64)
    new_of_old[good] = np.arange(good.size)
    sub = dict(res)
    sub["cluster_track"] = res["cluster_track"][good]
    sub["trk_seed"] = new_of_old[res["trk_seed"]].astype(np.int32)
    sub["trk_hits"] = new_of_old[res["trk_hits"]].astype(np.int32)
    assert sub["trk_hits"].min() >= 0 and sub["trk_seed"].min() >= 0
    st = parity.compare_tracks(o, sub, good.size)
    parity.assert_contract(st, exact_count=True)
    assert st["assign_identical"] == good.size and st["par_bit_identical"]
    sorted_idx, bin_first = trk.grid_export()
    assert bin_first[-1] == good.size and set(sorted_idx[good.size:].tolist()) == set(bad.tolist())


def test_find_twice_on_one_grid_with_other_cuts(torch_cuda, orc):
    """The grid stays valid until the next tpc_grid_build: a second tpc_find_tracks on it with other cuts (other links,
    other start hits) must give what a fresh build with those cuts gives -- no start bit of the first call survives."""
    from paper_2106_03636_b200 import binding
    ev = make_config(1, n_tracks=300)
    p2 = ev.params.with_(ca_cut=2.0, chi2_cut=9.0, max_gap=2)
    t = torch_cuda
    y, z, sr = t.from_numpy(ev.y).cuda(), t.from_numpy(ev.z).cuda(), t.from_numpy(ev.sector_row).cuda()
    trk = binding.Tracker(ev.params, ev.n)
    first = trk.run(y, z, sr)
    trk.params, trk.P = p2, binding.make_params(p2)           # same grid (cells unchanged), other cuts
    trk.find_tracks()
    trk.fit_tracks()
    again = trk.results()
    fresh = binding.Tracker(p2, ev.n).run(y, z, sr)
    assert not np.array_equal(first["cluster_track"], fresh["cluster_track"])      # the cuts do matter
    for k in fresh:
        assert np.array_equal(again[k], fresh[k]), k
    o = orc.run(p2, ev.y, ev.z, ev.sector_row, "f32", True)
    st = parity.compare_tracks(o, again, ev.n)
    assert st["assign_identical"] == ev.n and st["tracks_oracle"] == st["tracks_cuda"]


def test_capacity_overflow_is_flagged_and_bounded(torch_cuda):
    from paper_2106_03636_b200 import binding
    ev = config0()
    trk = binding.Tracker(ev.params, ev.n, max_tracklets=40, max_tracks=8)
    res = trk.run(*_dev(torch_cuda, ev))
    assert res["status"] & binding.ST_TRACKLET_OVERFLOW
    assert res["counters"][binding.CNT_TRACKLETS] == 40
    assert res["counters"][binding.CNT_STARTS_FOUND] > 40
    assert res["status"] & binding.ST_TRACK_OVERFLOW
    assert res["trk_seed"].size == 8 and res["trk_hits"].size == int(res["trk_nhits"].sum())
    assert np.all(res["cluster_track"] < 8)


@pytest.mark.parametrize("cell", [1.0, 3.25])
def test_grid_cell_independence(torch_cuda, orc, cell):
    """R8 / pin I4 on the CUDA side: another cell size changes the grid, not the tracks."""
    from paper_2106_03636_b200 import binding
    ev = make_config(1, n_tracks=600)
    p = ev.params.with_(cell_y=cell, cell_z=cell)
    o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)     # oracle at the default cell
    trk = binding.Tracker(p, ev.n)
    res = trk.run(*_dev(torch_cuda, ev))
    st = parity.compare_tracks(o, res, ev.n)
    parity.assert_contract(st, exact_count=True)
    assert st["assign_identical"] == ev.n


def test_host_buffer_entry_point(torch_cuda, orc):
    """tpc_track_host (the e2e call of bench.py) returns EVERY output, equal to the device-pointer calls; so does
    the enqueue-only pair tpc_track_host_async / tpc_track_host_fetch with two contexts in flight."""
    from paper_2106_03636_b200 import binding
    torch = torch_cuda
    ev = make_config(1, n_tracks=400)
    trk = binding.Tracker(ev.params, ev.n)
    ref = trk.run(*_dev(torch, ev))

    def same(t):
        got = t.host_results()
        assert set(got) == set(ref)
        for k in ref:
            assert np.array_equal(got[k], ref[k]), k

    trk2 = binding.Tracker(ev.params, ev.n)
    trk2.make_host_staging()
    hy, hz, hs = (torch.from_numpy(a).pin_memory() for a in (ev.y, ev.z, ev.sector_row))
    h2d, d2h = trk2.track_host(hy, hz, hs)
    assert h2d == 12 * ev.n
    K, H = ref["trk_seed"].size, ref["trk_hits"].size
    assert d2h == 4 * 16 + 4 * ev.n + K * (12 + 8 + 80 + 16) + 4 * H
    same(trk2)
    # enqueue-only variant on side streams, two contexts in flight (bench.py's e2e pipeline)
    trk3 = binding.Tracker(ev.params, ev.n)
    trk3.make_host_staging()
    ctx, streams = [trk2, trk3], [torch.cuda.Stream(), torch.cuda.Stream()]
    events = [torch.cuda.Event(), torch.cuda.Event()]
    for t in ctx:
        for v in t.host.values():
            v.zero_()
    fetched = 0
    for i in range(4):
        with torch.cuda.stream(streams[i % 2]):
            ctx[i % 2].track_host_async(hy, hz, hs)
            events[i % 2].record()
        if i > 0:
            events[(i - 1) % 2].synchronize()
            with torch.cuda.stream(streams[(i - 1) % 2]):
                fetched = ctx[(i - 1) % 2].track_host_fetch()
    events[1].synchronize()
    with torch.cuda.stream(streams[1]):
        ctx[1].track_host_fetch()
    for st in streams:
        st.synchronize()
    assert fetched + 4 * 16 + 4 * ev.n == d2h
    for t in ctx:
        same(t)
