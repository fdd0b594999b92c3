"""R26 on the GPU: tpc_merge_tracks against the CPU oracle on the same events (-m gpu).

The sector-local tracks of the two sides are bit-identical (tests/test_gpu_parity.py), so the links -- integer
decisions taken from the same fp32 arithmetic -- and the merged fits must be too.  Tracks are matched by seed (the
order of the track list differs between the two), global tracks by the seed of their head piece."""
import numpy as np
import pytest

from paper_2106_03636_b200.synth import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: -m gpu tests must run on the B200 box")
    return torch


def compare_merge(orc, ev, res, gm, mp=None):
    o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)
    m = orc.merge(ev.params, ev.y, ev.z, ev.sector_row, o, mp, "f32")
    assert res["trk_seed"].size == o["trk_seed"].size
    g_of_seed = {int(s): i for i, s in enumerate(res["trk_seed"])}
    to_g = np.array([g_of_seed[int(s)] for s in o["trk_seed"]])            # oracle track -> cuda track

    def seed_or_none(idx, seeds):
        return np.where(idx >= 0, seeds[np.maximum(idx, 0)], -1)

    # links, as (seed, seed of successor / predecessor)
    for key in ("succ", "pred"):
        a = seed_or_none(m[key], o["trk_seed"])
        b = seed_or_none(gm["trk_" + key][to_g], res["trk_seed"])
        assert np.array_equal(a, b), f"{key}: {np.count_nonzero(a != b)} of {a.size} links differ"
    assert np.array_equal(m["succ_chi2"], gm["trk_succ_chi2"][to_g]), "chi2 of the best successor differs"
    assert gm["n_pairs_dropped"] == 0 and gm["n_pairs"] >= int((m["succ_chi2"] >= 0).sum())
    n_links = int((m["succ"] >= 0).sum())
    assert gm["n_links"] == n_links and gm["n_global"] == m["g_head"].size == o["trk_seed"].size - n_links
    # global tracks, matched by the seed of the head
    og = {int(o["trk_seed"][h]): i for i, h in enumerate(m["g_head"])}
    order = np.array([og[int(res["trk_seed"][h])] for h in gm["g_head"]])  # cuda global -> oracle global
    for key in ("g_nseg", "g_nhits", "gndf"):
        assert np.array_equal(m[key][order], gm[key]), key
    for key in ("gxref", "gzref", "gchi2"):
        assert np.array_equal(m[key][order], gm[key]), key
    assert np.array_equal(m["gpar"][:, order], gm["gpar"]) and np.array_equal(m["gcov"][:, order], gm["gcov"])
    # trk_global is consistent with the heads
    assert np.array_equal(order[gm["trk_global"][to_g]], m["trk_global"])
    return n_links, int((m["g_nseg"] > 1).sum())


@pytest.mark.parametrize("cfg,kw", [(1, {}), (2, {}), (3, dict(n_coll=2, n_tracks=2500))])
def test_merge_matches_oracle(torch_cuda, orc, cfg, kw):
    from paper_2106_03636_b200 import binding
    ev = make_config(cfg, **kw)
    t = torch_cuda
    trk = binding.Tracker(ev.params, ev.n)
    res = trk.run(t.from_numpy(ev.y).cuda(), t.from_numpy(ev.z).cuda(), t.from_numpy(ev.sector_row).cuda())
    gm = trk.merge_tracks()
    links, merged = compare_merge(orc, ev, res, gm)
    print(f"\nmerge c{cfg}: {res['trk_seed'].size} sector-local tracks, {links} links, {merged} merged global tracks of "
          f"{gm['n_global']}")
    assert links > 50


def test_merge_single_sector_has_nothing_to_link_but_gaps(torch_cuda, orc):
    """configs[0]: one sector -- only same-sector links (holes longer than max_gap) are possible."""
    from paper_2106_03636_b200 import binding
    ev = make_config(0)
    t = torch_cuda
    trk = binding.Tracker(ev.params, ev.n)
    res = trk.run(t.from_numpy(ev.y).cuda(), t.from_numpy(ev.z).cuda(), t.from_numpy(ev.sector_row).cuda())
    gm = trk.merge_tracks()
    compare_merge(orc, ev, res, gm)


def test_merge_argument_errors(torch_cuda):
    from paper_2106_03636_b200 import binding
    ev = make_config(0)
    t = torch_cuda
    trk = binding.Tracker(ev.params, ev.n)
    trk.run(t.from_numpy(ev.y).cuda(), t.from_numpy(ev.z).cuda(), t.from_numpy(ev.sector_row).cuda())
    with pytest.raises(binding.TpcError):
        trk.merge_tracks(chi2_cut=0.0)
    with pytest.raises(binding.TpcError):
        trk.merge_tracks(max_rows=0)


@pytest.mark.parametrize("passes", [1, 3])
def test_merge_refuses_tracks_fitted_with_an_odd_number_of_passes(torch_cuda, passes):
    """After an odd number of R22 passes the fitted state sits at the outermost hit; R26 needs it at the innermost one.
    find + fit run as usual, tpc_merge_tracks returns TPC_EINVAL instead of linking from the wrong end."""
    from paper_2106_03636_b200 import binding
    ev = make_config(0)
    t = torch_cuda
    p = ev.params.with_(n_fit_passes=passes)
    trk = binding.Tracker(p, ev.n)
    res = trk.run(t.from_numpy(ev.y).cuda(), t.from_numpy(ev.z).cuda(), t.from_numpy(ev.sector_row).cuda())
    assert res["trk_seed"].size > 50
    with pytest.raises(binding.TpcError, match="invalid argument"):
        trk.merge_tracks()



def test_merge_refits_chains_of_more_than_16_pieces(torch_cuda, orc):
    """Holes longer than max_gap inside one sector give one piece each, so the number of pieces of a chain is not
    bounded by the sector crossings.  A 400-particle collision with two of every six pad rows removed, max_gap = 1 and
    min_hits = 4 leaves pieces of four hits; with a wide chi2 cut they chain up to ~20 pieces, and every chain is refitted
    (the refit kernel used to give up beyond 16 pieces while the oracle went on)."""
    from types import SimpleNamespace
    from paper_2106_03636_b200 import binding
    full = make_config(1, n_tracks=400)
    keep = (full.sector_row % full.params.n_rows) % 6 < 4
    ev = SimpleNamespace(params=full.params.with_(max_gap=1, min_hits=4), y=full.y[keep], z=full.z[keep],
                         sector_row=full.sector_row[keep], n=int(keep.sum()))
    mp = dict(chi2_cut=500.0, dz_max=64.0, ce_tol=1.0, max_rows=12)
    t = torch_cuda
    dev = [t.from_numpy(a).cuda() for a in (ev.y, ev.z, ev.sector_row)]
    # ~8300 four-hit pieces with ~15 candidate pairs each under this cut: the pair list of the default capacity
    # (4 x max_tracks entries) overflows, and that is reported, not swallowed ...
    small = binding.Tracker(ev.params, ev.n)
    small.run(*dev)
    with pytest.raises(binding.TpcError, match="pair list"):
        small.merge_tracks(**mp)
    # ... and with room for every pair the result is the oracle's
    trk = binding.Tracker(ev.params, ev.n, max_tracklets=65536, max_tracks=262144)   # room for ~50 candidate pairs per piece
    res = trk.run(*dev)
    assert res["status"] == 0
    gm = trk.merge_tracks(**mp)
    compare_merge(orc, ev, res, gm, mp)
    long_chain = gm["g_nseg"] > 16
    assert long_chain.sum() >= 10 and (gm["gndf"][long_chain] > 0).sum() >= 10
