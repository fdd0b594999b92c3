"""-m gpu: tpc_find_collisions (R25) against the oracle (integer work: bit-exact) and against the
generator's collision list on a short 50 kHz Pb-Pb slice (configs[4] recipe, 8 orbits)."""
import numpy as np
import pytest

from paper_2106_03636_b200.synth import V_DRIFT, make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def slice8():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: -m gpu tests must run on the B200 box")
    from paper_2106_03636_b200 import binding
    ev = make_config(4, n_orbits=8)
    trk = binding.Tracker(ev.params, ev.n)
    res = trk.run(torch.from_numpy(ev.y).cuda(), torch.from_numpy(ev.z).cuda(), torch.from_numpy(ev.sector_row).cuda())
    t_lo = float(np.floor(-ev.params.z_hi / V_DRIFT)) - 2.0
    t_hi = float(np.ceil(-ev.params.z_lo / V_DRIFT)) + 2.0
    g = {side: trk.find_collisions(t_lo, t_hi, V_DRIFT, side=side) for side in (0, 1, -1)}
    return ev, res, g, t_lo, t_hi


@pytest.mark.parametrize("side", [0, 1, -1])
def test_collisions_match_oracle_exactly(slice8, orc, side):
    ev, res, g, t_lo, t_hi = slice8
    g = g[side]
    o = orc.collisions(g["t0"], g["dca"], t_lo, t_hi, sector=res["trk_sector"], side=side)
    assert g["n_found"] == o["coll_time"].size > 10
    for k in ("coll_bin", "coll_ntracks", "trk_collision"):
        assert np.array_equal(g[k], o[k]), k
    assert np.array_equal(g["coll_time"], o["coll_time"])


@pytest.mark.parametrize("side", [1, -1])
def test_isolated_collisions_are_found_at_their_time(slice8, side):
    """A TPC side sees a collision at t - side * z_vertex / v_d (R5, R24): with the sides clustered separately every
    isolated collision with enough tracks is found within 1.5 us of that time, and its tracks are assigned to it."""
    ev, res, g, t_lo, t_hi = slice8
    g = g[side]
    t_true, idx = np.unique(ev.trk["t_us"], return_index=True)
    ntrk = np.array([np.count_nonzero(ev.trk["t_us"] == t) for t in t_true])
    vz = np.array([np.median(ev.trk["vz"][ev.trk["t_us"] == t]) for t in t_true])      # 85 % primaries share the vertex
    gap = np.minimum(np.diff(t_true, prepend=-1e9), np.diff(t_true, append=1e9))
    good = (gap > 12.0) & (ntrk >= 100)
    assert good.sum() >= 5
    first, nh = res["trk_first_hit"], res["trk_nhits"]
    tt = ev.true_track[res["trk_hits"][first + nh // 2]]
    on_side = (res["trk_sector"] < 18) == (side > 0)
    for t, z in zip(t_true[good], vz[good]):
        expect = t - side * z / V_DRIFT
        d = np.abs(g["coll_time"] - expect)
        assert d.min() < 1.5, f"collision at {t:.1f} us (side time {expect:.1f}) not found (nearest {g['coll_time'][d.argmin()]:.1f})"
        c = int(d.argmin())
        mine = (tt >= 0) & (nh >= 60) & (g["dca"] < 1.0) & on_side
        mine[mine] &= ev.trk["t_us"][tt[mine]] == t
        if mine.sum() > 20:
            assert np.mean(g["trk_collision"][mine] == c) > 0.9
    assert np.all(g["trk_collision"][~on_side] == -1)


def test_collisions_argument_errors():
    from paper_2106_03636_b200 import binding
    import ctypes as C
    L = binding.load()
    out = C.c_size_t(0)
    assert L.tpc_collisions_workspace_bytes(C.c_int64(0), C.c_int64(10), C.byref(out)) == -1
    assert L.tpc_collisions_workspace_bytes(C.c_int64(100), C.c_int64(10), C.byref(out)) == 0 and out.value > 0


def test_pair_sides_matches_oracle_and_truth(slice8, orc):
    """R29: tpc_pair_sides on the two per-side collision lists equals the oracle's pairing, and the paired (t, z_vertex)
    are the generator's for the collisions whose halves were both found (isolated ones)."""
    import torch
    from paper_2106_03636_b200 import binding
    ev, res, g, t_lo, t_hi = slice8
    trk = binding.Tracker(ev.params, ev.n)
    trk.run(torch.from_numpy(ev.y).cuda(), torch.from_numpy(ev.z).cuda(), torch.from_numpy(ev.sector_row).cuda())
    a = trk.find_collisions(t_lo, t_hi, V_DRIFT, side=1)
    c = trk.find_collisions(t_lo, t_hi, V_DRIFT, side=-1)
    p = trk.pair_sides()
    o = orc.pair_sides(a["coll_time"], a["coll_ntracks"], c["coll_time"], c["coll_ntracks"])
    for k in ("pair_of_a", "pair_of_c", "t", "z_vertex"):
        assert np.array_equal(p[k], o[k]), k
    assert p["t"].size >= 5
    # against the generator: every isolated, well-populated collision comes back as a pair at its time and vertex
    t_true = np.unique(ev.trk["t_us"])
    ntrk = np.array([np.count_nonzero(ev.trk["t_us"] == t) for t in t_true])
    vz = np.array([np.median(ev.trk["vz"][ev.trk["t_us"] == t]) for t in t_true])
    gap = np.minimum(np.diff(t_true, prepend=-1e9), np.diff(t_true, append=1e9))
    good = (gap > 25.0) & (ntrk >= 200)
    assert good.sum() >= 3
    for t, z in zip(t_true[good], vz[good]):
        d = np.abs(p["t"] - t)
        assert d.min() < 1.0, f"collision at {t:.1f} us has no pair (nearest {p['t'][d.argmin()]:.1f})"
        assert abs(p["z_vertex"][d.argmin()] - z) < 2.0


def test_pair_sides_reads_no_more_than_its_capacity(orc):
    """The per-side counts are read on the device.  A list longer than the max_collisions passed to tpc_pair_sides (the
    collision finder was given a larger capacity) is paired on its first max_collisions entries only and nothing is
    written beyond the capacity of the outputs or of the workspace."""
    import ctypes as C
    import torch
    from paper_2106_03636_b200 import binding
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: -m gpu tests must run on the B200 box")
    lib = binding.load()
    rng = np.random.default_rng(29)
    n, cap, guard = 600, 256, 64
    t_true = np.sort(rng.uniform(0.0, 12000.0, n))
    zv = rng.normal(0.0, 5.0, n)
    tA, tC = np.sort(t_true - zv / V_DRIFT).astype(np.float32), np.sort(t_true + zv / V_DRIFT).astype(np.float32)
    cA = rng.integers(10, 900, n).astype(np.int32)
    cC = np.maximum(1, cA + rng.integers(-8, 9, n)).astype(np.int32)
    dev = lambda a: torch.from_numpy(a).cuda()
    nn = torch.tensor([n, n], dtype=torch.int32, device="cuda")
    wsb = C.c_size_t(0)
    assert lib.tpc_pair_sides_workspace_bytes(C.c_int64(cap), C.byref(wsb)) == 0
    ws = torch.full((int(wsb.value) + 4 * guard,), 0x5A, dtype=torch.uint8, device="cuda")
    mk = lambda dt, v: torch.full((cap + guard,), v, dtype=dt, device="cuda")
    pa, pc, tt, zz = mk(torch.int32, -7), mk(torch.int32, -7), mk(torch.float32, -7.0), mk(torch.float32, -7.0)
    npairs = torch.zeros(1, dtype=torch.int32, device="cuda")
    p = lambda x: C.c_void_p(x.data_ptr())
    dA, dcA, dC, dcC = dev(tA), dev(cA), dev(tC), dev(cC)
    rc = lib.tpc_pair_sides(p(nn), p(dA), p(dcA), p(nn), p(dC), p(dcC), C.c_int64(cap), C.c_double(15.5), C.c_double(3.88),
                            C.c_double(V_DRIFT), p(ws), C.c_size_t(int(wsb.value)), p(pa), p(pc), p(tt), p(zz), p(npairs),
                            C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == 0
    torch.cuda.synchronize()
    o = orc.pair_sides(tA[:cap], cA[:cap], tC[:cap], cC[:cap], v_drift=V_DRIFT)
    k = int(npairs.item())
    assert k == o["t"].size > 200
    assert np.array_equal(pa[:cap].cpu().numpy(), o["pair_of_a"]) and np.array_equal(pc[:cap].cpu().numpy(), o["pair_of_c"])
    assert np.array_equal(tt[:k].cpu().numpy(), o["t"]) and np.array_equal(zz[:k].cpu().numpy(), o["z_vertex"])
    for out in (pa, pc, tt, zz):
        assert bool((out[cap:] == -7).all()), "written beyond max_collisions"
    assert bool((ws[int(wsb.value):] == 0x5A).all()), "workspace overrun"
