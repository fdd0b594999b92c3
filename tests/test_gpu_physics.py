"""R28 on the GPU: tpc_fit_tracks_physics and tpc_tag_clusters against the CPU oracle (-m gpu)."""
import numpy as np
import pytest

from paper_2106_03636_b200.synth import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.mark.parametrize("cfg,kw", [(0, {}), (1, dict(n_tracks=1500)), (3, dict(n_coll=1, n_tracks=1500))])
def test_physics_fit_and_tags_match_oracle(torch_cuda, orc, cfg, kw):
    from paper_2106_03636_b200 import binding
    t = torch_cuda
    ev = make_config(cfg, **kw)
    trk = binding.Tracker(ev.params, ev.n)
    res = trk.run(t.from_numpy(ev.y).cuda(), t.from_numpy(ev.z).cuda(), t.from_numpy(ev.sector_row).cuda())
    # defaults: the plain refit, bit for bit
    g0 = trk.fit_tracks_physics()
    for k in ("par", "cov", "xref", "zref", "chi2", "ndf"):
        assert np.array_equal(g0[k], res[k]), k
    assert not g0["hit_flag"].any()
    # material + outlier rejection against the oracle on the same hit lists
    g = trk.fit_tracks_physics(x0inv=2e-4, outlier_cut=12.0)
    o = orc.fit_physics(ev.params, ev.y, ev.z, ev.sector_row, res["trk_nhits"], res["trk_first_hit"], res["trk_hits"],
                        x0inv=2e-4, outlier_cut=12.0)
    for k in ("par", "cov", "xref", "zref", "chi2", "ndf", "hit_flag"):
        assert np.array_equal(g[k], o[k]), k
    assert g["hit_flag"].sum() > 0, "a cut of 12 rejects some hits on smeared data"
    # tags
    tag = trk.tag_clusters(qpt_max=4.0, use_physics_fit=True)
    want = orc.tag_clusters(res["cluster_track"], o["par"][4], o["ndf"], res["trk_nhits"], res["trk_first_hit"], res["trk_hits"],
                            o["hit_flag"], qpt_max=4.0)
    assert np.array_equal(tag, want)
    assert (tag & 2).any() and (tag & 4).any() and (tag == 0).any() == bool((res["cluster_track"] < 0).any())
    tag2 = trk.tag_clusters(qpt_max=4.0)
    want2 = orc.tag_clusters(res["cluster_track"], res["par"][4], res["ndf"], res["trk_nhits"], res["trk_first_hit"], res["trk_hits"],
                             None, qpt_max=4.0)
    assert np.array_equal(tag2, want2)
