"""-m gpu: the bench workload (BASELINE.json configs[4], one 128-orbit 50 kHz Pb-Pb Time Frame, ~1.4e8 clusters)
in the launch configuration bench.py times, checked two ways:

 1. properties that hold at any size on the WHOLE output (parity.check_output_invariants);
 2. element-by-element parity with the CPU oracle on EVERY sector (~3.8e6 clusters each; sectors are independent
    through the hot path, so the oracle run on a sector's clusters alone must reproduce the CUDA result restricted
    to it -- assignments, hit lists, fitted parameters and covariances, bit for bit).  The 36 oracle runs are dealt
    to the host cores (about a minute on 16 cores).
(bench.py's cpu_baseline leg runs the oracle on all 36 sectors and compares the track and assignment COUNTS of the
whole Time Frame with the GPU's in every bench run.)
"""
import numpy as np
import pytest

import parity

pytestmark = pytest.mark.gpu

SAMPLED_SECTORS = tuple(range(36))     # every sector of the Time Frame: the whole bench workload, element by element
KEEP = ("cluster_track", "trk_seed", "trk_nhits", "trk_first_hit", "trk_hits", "par", "cov", "xref", "zref", "chi2", "ndf")
_EV = None


@pytest.fixture(scope="module")
def c4_run():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: -m gpu tests must run on the B200 box")
    from bench import make_event                      # the same event bench.py times (seed 5, A7)
    from paper_2106_03636_b200 import binding
    ev = make_event(4, 0, 1)
    trk = binding.Tracker(ev.params, ev.n)
    y, z, sr = (torch.from_numpy(a).cuda() for a in (ev.y, ev.z, ev.sector_row))
    res = trk.run(y, z, sr)
    assert res["status"] == 0, f"device status bits {res['status']}"
    work = binding.work_counts(res["counters"])
    res["merge"] = trk.merge_tracks()                 # R26 on the whole Time Frame (invariants below)
    res["tags"] = trk.tag_clusters(qpt_max=10.0)      # R28c
    del trk, y, z, sr
    torch.cuda.empty_cache()
    return ev, res, work


def _oracle_sector(sector):
    from oracle import tpc_oracle as orc
    ev = _EV
    sel = np.nonzero(ev.sector_row // int(ev.params.n_rows) == sector)[0]
    o = orc.run(ev.params, ev.y[sel], ev.z[sel], ev.sector_row[sel], "f32", True)
    return sector, {k: o[k] for k in KEEP}


@pytest.fixture(scope="module")
def c4_oracle(c4_run, orc):
    """Oracle output of every sampled sector, computed by a pool of forked workers (they only touch numpy + the oracle)."""
    import multiprocessing as mp
    import os
    global _EV
    _EV = c4_run[0]
    with mp.get_context("fork").Pool(min(len(SAMPLED_SECTORS), os.cpu_count() or 1)) as pool:
        out = dict(pool.imap_unordered(_oracle_sector, SAMPLED_SECTORS, chunksize=1))
    _EV = None
    return out


def test_c4_size_and_whole_output_invariants(c4_run):
    ev, res, work = c4_run
    assert ev.n > 100_000_000, "configs[4] should hold > 1e8 clusters (DESIGN.md A8)"
    assert res["trk_seed"].size > 1_000_000
    parity.check_output_invariants(res, ev.sector_row, int(ev.params.n_rows), int(ev.params.min_hits))
    # the follower's work is what scales: every recorded update is preceded by a transport
    assert work["propagations"] >= work["updates"] - int(res["counters"][1]) > 0


def test_c4_merge_and_tags_invariants(c4_run):
    """tpc_merge_tracks / tpc_tag_clusters at the full size (the oracle cannot merge 1.8e6 tracks in test time; it is
    compared link for link on configs 0-3 in tests/test_gpu_merge.py): properties that hold at any size."""
    ev, res, _ = c4_run
    m, K = res["merge"], res["trk_seed"].size
    assert m["n_pairs_dropped"] == 0, "pair list full: links would be incomplete and not reproducible"
    assert m["n_links"] <= m["n_pairs"] <= 4 * K
    succ, pred = m["trk_succ"], m["trk_pred"]
    a = np.nonzero(succ >= 0)[0]
    assert np.array_equal(pred[succ[a]], a), "succ and pred must be inverse to one another"
    assert np.unique(succ[a]).size == a.size, "a track follows at most one track"
    assert (pred >= 0).sum() == a.size == m["n_links"] and m["n_global"] == K - a.size
    sec = res["trk_sector"]
    rel_ok = (sec[a] == sec[succ[a]]) | (np.abs(sec[a] % 18 - sec[succ[a]] % 18) % 16 <= 1)
    assert rel_ok.all(), "links only join a sector with itself, a neighbour or its mirror"
    assert int(m["g_nhits"].sum()) == int(res["trk_nhits"].sum()) and int(m["g_nseg"].sum()) == K
    assert np.array_equal(np.bincount(m["trk_global"], minlength=m["n_global"]), m["g_nseg"])
    assert np.all(np.diff(m["g_head"]) > 0) and np.all(pred[m["g_head"]] < 0)
    single = m["g_nseg"] == 1
    assert np.array_equal(m["gpar"][:, single], res["par"][:, m["g_head"][single]])
    merged_ok = (~single) & (m["gndf"] > 0)
    assert merged_ok.sum() > 0.9 * (~single).sum()
    assert 0.8 < np.median(m["gchi2"][merged_ok] / m["gndf"][merged_ok]) < 1.3
    assert a.size > 0.3 * K, "about half of the sector-local tracks of a Time Frame are pieces of longer ones"
    tags = res["tags"]
    assert np.array_equal(tags > 0, res["cluster_track"] >= 0) and np.all(tags <= 3)
    low = np.abs(res["par"][4]) > 10.0
    assert np.array_equal((tags & 2) > 0, (res["cluster_track"] >= 0) & (low | (res["ndf"] < 0))[np.maximum(res["cluster_track"], 0)])


@pytest.mark.parametrize("sector", SAMPLED_SECTORS)
def test_c4_sector_matches_oracle(c4_run, c4_oracle, sector):
    ev, res, _ = c4_run
    nrows = int(ev.params.n_rows)
    sel, rs = parity.restrict_to_sector(res, ev.sector_row, nrows, sector)
    assert sel.size > 1_000_000
    o = c4_oracle[sector]
    st = parity.compare_tracks(o, rs, sel.size)
    print(f"c4 sector {sector}: {st}")
    parity.assert_contract(st, exact_count=True)
    assert st["assign_identical"] == sel.size
    assert st["tracks_same_hits"] == st["tracks_oracle"]
    assert st["par_bit_identical"] and st["cov_bit_identical"]
