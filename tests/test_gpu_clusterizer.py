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
    """The chain the paper runs, digits -> clusterizer -> tracker, with both steps on the device.  tpc_clusterize writes
    its clusters in the order the peaks were found, which changes from run to run, and the tracker breaks exact ties by
    input index (include/tpc_b200.h); so between the two steps the clusters are put into the oracle's order -- ascending
    (sector_row, time, pad) of the peak cell -- on the host.  After that the chain must equal the oracle chain in
    everything: assignment of every cluster, hit lists, fitted parameters and covariances."""
    import parity
    from paper_2106_03636_b200 import binding
    t = torch_cuda
    ev = make_config(1, n_tracks=1500)
    d = digitize(ev)
    g, o = run_both(t, orc, ev.params, d)
    k = np.lexsort((g["pad"], g["time"], g["sector_row"]))
    y, z, sr = g["y"][k], g["z"][k], g["sector_row"][k]
    assert np.array_equal(y, o["y"]) and np.array_equal(z, o["z"]) and np.array_equal(sr, o["sector_row"])
    trk = binding.Tracker(ev.params, y.size)
    res = trk.run(t.from_numpy(y).cuda(), t.from_numpy(z).cuda(), t.from_numpy(sr).cuda())
    oo = orc.run(ev.params, o["y"], o["z"], o["sector_row"], "f32", True)
    assert res["status"] == 0 and res["trk_seed"].size == oo["trk_seed"].size > 2000
    st = parity.compare_tracks(oo, res, y.size)
    parity.assert_contract(st, exact_count=True)
    assert st["assign_identical"] == y.size and st["tracks_same_hits"] == st["tracks_matched"] == oo["trk_seed"].size
    assert st["par_bit_identical"]


def test_digits_without_charge_are_ignored_on_the_gpu(torch_cuda, orc):
    """R27: digits of ADC <= 0 change nothing -- same clusters as the oracle (which drops them) and as the run without
    them, and no NaN from a peak whose 3 x 3 sum would have been 0."""
    ev = make_config(0)
    d = digitize(ev)
    rng = np.random.default_rng(27)
    k = rng.integers(0, d.n, 5000)
    cat = lambda a, b: np.concatenate([a, b]).astype(np.int32)
    d2 = type(d)(sector_row=cat(d.sector_row, d.sector_row[k]),
                 pad=cat(d.pad, np.clip(d.pad[k] + rng.integers(-1, 2, k.size), 0, 65535)),
                 time=cat(d.time, np.clip(d.time[k] + rng.integers(-1, 2, k.size), 0, None)),
                 adc=cat(d.adc, rng.integers(-40, 1, k.size)), pad_width=d.pad_width, time_width=d.time_width,
                 n_deposits=d.n_deposits)
    g0, _ = run_both(torch_cuda, orc, ev.params, d)
    g2, o2 = run_both(torch_cuda, orc, ev.params, d2)
    assert g2["n_found"] == g0["n_found"] == o2["n_found"] > 1000
    k0, k2 = (np.lexsort((g["pad"], g["time"], g["sector_row"])) for g in (g0, g2))
    for key in ("y", "z", "q", "sector_row", "pad", "time"):
        assert np.array_equal(g2[key][k2], g0[key][k0]) and np.array_equal(g2[key][k2], o2[key]), key
    assert np.isfinite(g2["y"]).all() and np.isfinite(g2["z"]).all()
    # by hand: a peak of 6 between two digits of -3 (S would be 0)
    from paper_2106_03636_b200 import binding
    i32 = lambda *v: torch_cuda.tensor(v, dtype=torch_cuda.int32, device="cuda")
    c = binding.clusterize(ev.params, i32(5, 5, 5, 5), i32(10, 9, 11, 10), i32(20, 20, 20, 21), i32(6, -3, -3, 0), 0.5, 0.25)
    assert c["n_found"] == 1 and c["q"][0] == 6.0 and np.isfinite(c["y"][0]) and np.isfinite(c["z"][0])
