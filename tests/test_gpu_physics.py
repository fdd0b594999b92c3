"""R28 on the GPU: tpc_fit_tracks_physics and tpc_tag_clusters against the CPU oracle (-m gpu)."""
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


OPT_DE = dict(x0inv=2e-4, outlier_cut=12.0, dedx=1.5e-4, eloss_sigma=0.4, err_ang_y=1.5, err_ang_z=0.8, err_drift_y=2e-4,
              err_drift_z=3e-4, v_drift=2.58, z_len=250.0)


@pytest.mark.parametrize("cfg,kw", [(0, {}), (2, dict(n_coll=40)), (4, dict(n_orbits=4))])
def test_energy_loss_and_cluster_errors_match_oracle(torch_cuda, orc, cfg, kw):
    """R28d/e: every option on, the drift length from tpc_track_time's own time offsets (both TPC sides in configs 2
    and 4: the sign of the shift), bit for bit; then without time offsets, and with a NaN among them."""
    from paper_2106_03636_b200 import binding
    t = torch_cuda
    ev = make_config(cfg, **kw)
    trk = binding.Tracker(ev.params, ev.n)
    res = trk.run(t.from_numpy(ev.y).cuda(), t.from_numpy(ev.z).cuda(), t.from_numpy(ev.sector_row).cuda())
    lists = (res["trk_nhits"], res["trk_first_hit"], res["trk_hits"])
    t0 = trk.track_time(2.58)["t0"]
    K = t0.size
    if cfg != 0:
        assert (res["trk_sector"] >= 18).any() and (res["trk_sector"] < 18).any()
    for case in ("t0", "none", "nan"):
        dev_t0 = None
        host_t0 = None
        if case != "none":
            dev_t0 = trk.trk_t0.clone()
            host_t0 = t0.copy()
            if case == "nan":
                dev_t0[: K : 3] = float("nan")
                host_t0[::3] = np.nan
        g = trk.fit_tracks_physics(trk_t0=dev_t0, **OPT_DE)
        o = orc.fit_physics(ev.params, ev.y, ev.z, ev.sector_row, *lists, trk_t0=host_t0, **OPT_DE)
        for k in ("par", "cov", "xref", "zref", "chi2", "ndf", "hit_flag"):
            assert np.array_equal(g[k], o[k], equal_nan=True), (case, k)
        if case == "t0":
            first = g
            # the self-contained gather path (no workspace) gives the same bits as the streamed hit records
            g2 = trk.fit_tracks_physics(trk_t0=dev_t0, use_workspace=False, **OPT_DE)
            for k in g:
                assert np.array_equal(g[k], g2[k], equal_nan=True), ("gather", k)
        elif case == "none":
            assert not np.array_equal(first["cov"], g["cov"]), "the drift terms must change the result"
    # each group of options alone, too
    for only in (dict(dedx=1.5e-4, eloss_sigma=0.4), dict(err_ang_y=1.5, err_ang_z=0.8),
                 dict(err_drift_y=2e-4, err_drift_z=3e-4, v_drift=2.58)):
        g = trk.fit_tracks_physics(trk_t0=trk.trk_t0, **only)
        o = orc.fit_physics(ev.params, ev.y, ev.z, ev.sector_row, *lists, trk_t0=t0, **only)
        for k in ("par", "cov", "chi2", "ndf"):
            assert np.array_equal(g[k], o[k], equal_nan=True), (tuple(only), k)
        assert not np.array_equal(g["par"], res["par"]), tuple(only)


def test_fit_options_argument_errors(torch_cuda):
    import ctypes as C
    from paper_2106_03636_b200 import binding
    ev = make_config(0)
    t = torch_cuda
    trk = binding.Tracker(ev.params, ev.n)
    trk.run(t.from_numpy(ev.y).cuda(), t.from_numpy(ev.z).cuda(), t.from_numpy(ev.sector_row).cuda())
    for bad in (dict(x0inv=-1.0), dict(dedx=float("nan")), dict(err_ang_y=float("inf")), dict(z_len=-1.0),
                dict(outlier_cut=float("nan"))):
        with pytest.raises(binding.TpcError):
            trk.fit_tracks_physics(**bad)
    with pytest.raises(ValueError):
        trk.fit_tracks_physics(trk_t0=t.zeros(trk.max_tracks, dtype=t.float64, device="cuda"))
