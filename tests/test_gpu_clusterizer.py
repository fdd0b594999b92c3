"""R27 on the GPU: tpc_clusterize against the CPU oracle on the same digits (-m gpu).  The output order of the CUDA
path is unspecified, so both cluster lists are ordered by peak cell (sector_row, time, pad) and then compared bit for
bit (integer sums; fp32 positions from the same operations)."""
import numpy as np
import pytest

from paper_2106_03636_b200.synth import config0, digitize, make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: -m gpu tests must run on the B200 box")
    return torch


def run_both(torch, orc, params, d, peak_min=6, **kw):
    from paper_2106_03636_b200 import binding
    dev = [torch.from_numpy(a).cuda() for a in (d.sector_row, d.pad, d.time, d.adc)]
    g = binding.clusterize(params, *dev, d.pad_width, d.time_width, peak_min, **kw)
    o = orc.clusterize(params, d.sector_row, d.pad, d.time, d.adc, d.pad_width, d.time_width, peak_min)
    return g, o


def ordered(c):
    k = np.lexsort((c["pad"], c["time"], c["sector_row"]))
    return {a: c[a][k] for a in ("y", "z", "q", "sector_row", "pad", "time")}


@pytest.mark.parametrize("cfg,kw", [(0, {}), (1, dict(n_tracks=2000)), (2, {})])
def test_clusterizer_matches_oracle(torch_cuda, orc, cfg, kw):
    ev = make_config(cfg, **kw)
    d = digitize(ev)
    g, o = run_both(torch_cuda, orc, ev.params, d)
    assert g["n_found"] == o["n_found"] > 0.9 * ev.n
    a, b = ordered(g), ordered(o)
    for k in b:
        assert np.array_equal(a[k], b[k]), k


def test_duplicates_invalid_digits_and_capacity(torch_cuda, orc):
    from paper_2106_03636_b200 import binding
    from paper_2106_03636_b200.synth.digitizer import Digits
    ev = config0(seed=7, n_tracks=30)
    d = digitize(ev)
    # every digit split into two of half the ADC (+ remainder): same clusters
    h = d.adc // 2
    d2 = Digits(np.r_[d.sector_row, d.sector_row], np.r_[d.pad, d.pad], np.r_[d.time, d.time], np.r_[h, d.adc - h].astype(np.int32),
                d.pad_width, d.time_width, d.n_deposits)
    g2, o = run_both(torch_cuda, orc, ev.params, d2)
    g1, _ = run_both(torch_cuda, orc, ev.params, d)
    a, b, c = ordered(g2), ordered(o), ordered(g1)
    for k in b:
        assert np.array_equal(a[k], b[k]) and np.array_equal(a[k], c[k]), k
    # digits that name no cell are ignored
    bad = Digits(np.r_[d.sector_row, [-3, 10 ** 6, 5]].astype(np.int32), np.r_[d.pad, [4, 4, 70000]].astype(np.int32),
                 np.r_[d.time, [4, 4, 4]].astype(np.int32), np.r_[d.adc, [99, 99, 99]].astype(np.int32), d.pad_width, d.time_width, 0)
    t = torch_cuda
    gb = binding.clusterize(ev.params, *[t.from_numpy(x).cuda() for x in (bad.sector_row, bad.pad, bad.time, bad.adc)],
                            d.pad_width, d.time_width)
    assert gb["n_found"] == g1["n_found"]
    # capacity: found is still counted, the arrays hold max_clusters
    gc, _ = run_both(torch_cuda, orc, ev.params, d, max_clusters=100)
    assert gc["n_found"] == g1["n_found"] and gc["y"].size == 100
    # empty input
    e = t.zeros(0, dtype=t.int32, device="cuda")
    assert binding.clusterize(ev.params, e, e, e, e, 0.5, 0.25)["n_found"] == 0


def test_digits_to_tracks_on_the_gpu(torch_cuda, orc):
    """The chain the paper runs: digits -> clusterizer -> tracker, all on the device; same tracks as the oracle chain."""
    from paper_2106_03636_b200 import binding
    t = torch_cuda
    ev = make_config(1, n_tracks=1500)
    d = digitize(ev)
    g, o = run_both(t, orc, ev.params, d)
    k = np.lexsort((g["pad"], g["time"], g["sector_row"]))          # fix an order so that index tie-breaks agree
    y, z, sr = g["y"][k], g["z"][k], g["sector_row"][k]
    trk = binding.Tracker(ev.params, y.size)
    res = trk.run(t.from_numpy(y).cuda(), t.from_numpy(z).cuda(), t.from_numpy(sr).cuda())
    oo = orc.run(ev.params, o["y"], o["z"], o["sector_row"], "f32", True)
    assert res["trk_seed"].size == oo["trk_seed"].size > 2000
    assert np.array_equal(np.sort(res["trk_seed"]), np.sort(oo["trk_seed"]))
