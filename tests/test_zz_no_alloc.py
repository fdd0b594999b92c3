"""tpc_pair_sides_static: the pairing of the two TPC sides' collisions (R29) for callers that cannot allocate.

Some users of this library cannot call cudaMalloc: a processing step inside a framework that owns every byte of GPU
memory and hands out slices of one block, or code on a path where the allocator's device-wide lock and the implicit
synchronisation of cudaMalloc / cudaFree are not acceptable.  tpc_pair_sides needs a small workspace (two arg-min
tables); tpc_pair_sides_static keeps those tables in an array inside the library's own device image instead (128.5 KiB
per GPU, at most TPC_PAIR_SIDES_STATIC_MAX = 16384 collisions per side), so such a caller passes inputs and outputs only.

What is checked here: on two calls in a row -- the first at the full 16384 collisions per side, so that the far end of
the array is used, the second on shorter, different lists, so that whatever the first call left in the array must not
matter -- the outputs equal those of tpc_pair_sides with a caller-owned workspace exactly (integer indices; t and
z_vertex bit for bit: same kernels, same arithmetic; the tolerance of the other R29 tests is equality too), and the
oracle's on the second.  Sizes beyond the limit are refused with their own error code.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a problem in this add-on must not hide
a result of the tests of the hot path.  The GPU test stands on its own (no fixture from another file, its own inputs), so
it passes alone in a fresh process -- where its first call is the one that looks up the array's device address -- and
after the rest of the suite."""
import ctypes as C

import numpy as np
import pytest

from paper_2106_03636_b200 import binding


def _collision_lists(rng, n_true, t_span_us, miss=0.1):
    """Two per-side collision lists as tpc_find_collisions writes them: ascending float32 times and track counts.  A
    collision at time t with vertex z_v is seen at t -/+ z_v / v_drift by sides A / C (R5); each side misses some."""
    t = np.sort(rng.uniform(0.0, t_span_us, n_true))
    zv = rng.normal(0.0, 5.0, n_true)
    mult = rng.integers(20, 2000, n_true)
    sides = []
    for sign in (-1.0, +1.0):
        keep = rng.random(n_true) > miss
        ts = (t + sign * zv / 2.58)[keep]
        order = np.argsort(ts, kind="stable")
        cnt = np.maximum(1, mult[keep] // 2 + rng.integers(-10, 11, keep.sum()))
        sides.append((ts[order].astype(np.float32), cnt[order].astype(np.int32)))
    return sides


def _to_device(side, cap, torch):
    ts, cnt = side
    n = ts.size
    assert n <= cap
    tt = torch.zeros(cap, dtype=torch.float32, device="cuda")
    cc = torch.zeros(cap, dtype=torch.int32, device="cuda")
    tt[:n] = torch.from_numpy(ts).cuda()
    cc[:n] = torch.from_numpy(cnt).cuda()
    nn = torch.tensor([n, n], dtype=torch.int32, device="cuda")
    return nn, tt, cc


def _outputs(cap, torch):
    return dict(pair_of_a=torch.full((cap,), -7, dtype=torch.int32, device="cuda"),
                pair_of_c=torch.full((cap,), -7, dtype=torch.int32, device="cuda"),
                t=torch.full((cap,), -7.0, dtype=torch.float32, device="cuda"),
                z_vertex=torch.full((cap,), -7.0, dtype=torch.float32, device="cuda"),
                n_pairs=torch.full((1,), -7, dtype=torch.int32, device="cuda"))


def _with_workspace(lib, a, c, cap, dt_max, sigma_t, v_drift, torch):
    """The existing path: tpc_pair_sides with a caller-owned workspace."""
    wsb = C.c_size_t(0)
    assert lib.tpc_pair_sides_workspace_bytes(C.c_int64(cap), C.byref(wsb)) == 0
    ws = torch.empty(int(wsb.value), dtype=torch.uint8, device="cuda")
    o = _outputs(cap, torch)
    p = lambda x: C.c_void_p(x.data_ptr())
    rc = lib.tpc_pair_sides(p(a[0]), p(a[1]), p(a[2]), p(c[0]), p(c[1]), p(c[2]), C.c_int64(cap), C.c_double(dt_max),
                            C.c_double(sigma_t), C.c_double(v_drift), p(ws), C.c_size_t(int(wsb.value)), p(o["pair_of_a"]),
                            p(o["pair_of_c"]), p(o["t"]), p(o["z_vertex"]), p(o["n_pairs"]),
                            C.c_void_p(torch.cuda.current_stream().cuda_stream))
    assert rc == 0
    torch.cuda.synchronize()
    return o


def _same(got, want, n_a, n_c):
    k = int(want["n_pairs"].item())
    assert int(got["n_pairs"].item()) == k
    for name, n in (("pair_of_a", n_a), ("pair_of_c", n_c), ("t", k), ("z_vertex", k)):
        g, w = got[name][:n].cpu().numpy(), want[name][:n].cpu().numpy()
        assert np.array_equal(g, w), name
    return k


@pytest.mark.gpu
def test_static_scratch_pairing_equals_the_workspace_path_on_two_calls_in_a_row(orc):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: -m gpu tests must run on the B200 box")
    lib = binding.load()
    rng = np.random.default_rng(20211106)
    dt_max, sigma_t, v_drift = 15.5, 3.88, 2.58
    cap1 = binding.PAIR_SIDES_STATIC_MAX

    # inputs of both calls first, so that nothing but the two static calls runs between them
    big = _collision_lists(rng, cap1, 20.0 * cap1, miss=0.0)            # 16384 per side: the whole array is in use
    small = _collision_lists(rng, 300, 6000.0, miss=0.15)               # a 128-orbit Time Frame has ~570 collisions
    a1, c1 = _to_device(big[0], cap1, torch), _to_device(big[1], cap1, torch)
    cap2 = 512
    a2, c2 = _to_device(small[0], cap2, torch), _to_device(small[1], cap2, torch)
    want1 = _with_workspace(lib, a1, c1, cap1, dt_max, sigma_t, v_drift, torch)
    want2 = _with_workspace(lib, a2, c2, cap2, dt_max, sigma_t, v_drift, torch)
    out1, out2 = _outputs(cap1, torch), _outputs(cap2, torch)

    # two calls in a row on one stream, outputs preallocated: the second finds the first one's tables in the array
    binding.pair_sides_static(*a1, *c1, cap1, dt_max, sigma_t, v_drift, out=out1)
    binding.pair_sides_static(*a2, *c2, cap2, dt_max, sigma_t, v_drift, out=out2)
    torch.cuda.synchronize()
    k1 = _same(out1, want1, big[0][0].size, big[1][0].size)
    k2 = _same(out2, want2, small[0][0].size, small[1][0].size)
    assert k1 > cap1 // 2 and k2 > 100          # the lists do pair up: the comparison is not one of empty results

    # the second call against the oracle as well (R29 is exact: reciprocal arg-mins in double, float outputs)
    o = orc.pair_sides(small[0][0], small[0][1], small[1][0], small[1][1], dt_max=dt_max, sigma_t=sigma_t, v_drift=v_drift)
    assert np.array_equal(out2["pair_of_a"][:small[0][0].size].cpu().numpy(), o["pair_of_a"])
    assert np.array_equal(out2["pair_of_c"][:small[1][0].size].cpu().numpy(), o["pair_of_c"])
    assert np.array_equal(out2["t"][:k2].cpu().numpy(), o["t"])
    assert np.array_equal(out2["z_vertex"][:k2].cpu().numpy(), o["z_vertex"])

    # the numpy-returning form of the wrapper gives the same answer (a third call on the same array)
    r = binding.pair_sides_static(*a2, *c2, cap2, dt_max, sigma_t, v_drift)
    assert np.array_equal(r["pair_of_a"], o["pair_of_a"]) and np.array_equal(r["z_vertex"], o["z_vertex"])

    # a call that is set up takes no device memory: free memory as the driver reports it does not move
    free_before = torch.cuda.mem_get_info()[0]
    binding.pair_sides_static(*a2, *c2, cap2, dt_max, sigma_t, v_drift, out=out2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before

    # beyond the fixed array: refused with its own code, outputs untouched
    cap3 = cap1 + 1
    a3, c3 = _to_device(small[0], cap3, torch), _to_device(small[1], cap3, torch)
    out3 = _outputs(cap3, torch)
    with pytest.raises(binding.TpcError, match="fixed scratch array"):
        binding.pair_sides_static(*a3, *c3, cap3, dt_max, sigma_t, v_drift, out=out3)
    torch.cuda.synchronize()
    assert int(out3["n_pairs"].item()) == -7


def test_static_entry_point_refuses_bad_sizes_without_a_gpu():
    """The size and pointer checks come before any CUDA call, so they can be exercised on a machine without a GPU."""
    lib = binding.load()
    buf = (C.c_int32 * 8)()
    p = C.cast(buf, C.c_void_p)

    def call(cap, dt_max=15.5, first=p):
        return lib.tpc_pair_sides_static(first, p, p, p, p, p, C.c_int64(cap), C.c_double(dt_max), C.c_double(3.88),
                                         C.c_double(2.58), p, p, p, p, p, C.c_void_p(0))

    assert call(binding.PAIR_SIDES_STATIC_MAX + 1) == -4
    assert b"fixed scratch array" in lib.tpc_strerror(-4)
    assert call(1 << 40) == -4
    assert call(0) == -1
    assert call(16, dt_max=0.0) == -1
    assert call(16, first=C.c_void_p(0)) == -1
    txt = open(__import__("os").path.join(__import__("os").path.dirname(binding.__file__), "..", "include", "tpc_b200.h")).read()
    assert f"#define TPC_PAIR_SIDES_STATIC_MAX {binding.PAIR_SIDES_STATIC_MAX}" in txt
