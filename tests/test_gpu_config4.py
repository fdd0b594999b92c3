"""-m gpu: the bench workload (BASELINE.json configs[4], one 128-orbit 50 kHz Pb-Pb Time Frame, ~1.4e8 clusters)
in the launch configuration bench.py times, checked two ways:

 1. properties that hold at any size on the WHOLE output (parity.check_output_invariants);
 2. element-by-element parity with the CPU oracle on sampled sectors: one A-side and one C-side sector, each
    whole (~3.8e6 clusters; sectors are independent through the hot path, so the oracle run on a sector's
    clusters alone must reproduce the CUDA result restricted to it -- assignments, hit lists, fitted
    parameters and covariances, bit for bit).
"""
import numpy as np
import pytest

import parity

pytestmark = pytest.mark.gpu

SAMPLED_SECTORS = (7, 29)     # alpha = 150 deg on side A; alpha = 230 deg on side C (mirrored drift axis)


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
    del trk, y, z, sr
    torch.cuda.empty_cache()
    return ev, res, work


def test_c4_size_and_whole_output_invariants(c4_run):
    ev, res, work = c4_run
    assert ev.n > 100_000_000, "configs[4] should hold > 1e8 clusters (DESIGN.md A8)"
    assert res["trk_seed"].size > 1_000_000
    parity.check_output_invariants(res, ev.sector_row, int(ev.params.n_rows), int(ev.params.min_hits))
    # the follower's work is what scales: every recorded update is preceded by a transport
    assert work["propagations"] >= work["updates"] - int(res["counters"][1]) > 0


@pytest.mark.parametrize("sector", SAMPLED_SECTORS)
def test_c4_sector_matches_oracle(c4_run, orc, sector):
    ev, res, _ = c4_run
    nrows = int(ev.params.n_rows)
    sel, rs = parity.restrict_to_sector(res, ev.sector_row, nrows, sector)
    assert sel.size > 1_000_000
    o = orc.run(ev.params, ev.y[sel], ev.z[sel], ev.sector_row[sel], "f32", True)
    st = parity.compare_tracks(o, rs, sel.size)
    print(f"c4 sector {sector}: {st}")
    parity.assert_contract(st, exact_count=True)
    assert st["assign_identical"] == sel.size
    assert st["tracks_same_hits"] == st["tracks_oracle"]
    assert st["par_bit_identical"] and st["cov_bit_identical"]
