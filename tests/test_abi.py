"""CPU-side checks of the C-ABI boundary: the library builds, loads and exports every symbol that
include/tpc_b200.h declares; the host-only entry points (no GPU work) behave as documented."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2106_03636_b200 import binding
from paper_2106_03636_b200.synth import TpcParams, config0

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "tpc_b200.h")


def _declared_symbols():
    txt = open(HEADER).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(tpc_[a-z_0-9]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    lib = binding.load()
    names = _declared_symbols()
    assert len(names) >= 10
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/tpc_b200.h but not exported"
    assert sorted(binding.SYMBOLS) == names, "binding.SYMBOLS out of date with the header"


def test_params_struct_layout_matches_header():
    """Field order/count of the ctypes mirror == the header's typedef (sizes: all 4-byte scalars)."""
    txt = open(HEADER).read()
    body = re.search(r"typedef struct \{(.*?)\} tpc_params_t;", txt, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        _type, rest = decl.split(None, 1)
        for nm in rest.split(","):
            fields.append(re.sub(r"\[.*\]", "", nm).strip())
    assert fields == [f[0] for f in binding.tpc_params_t._fields_]
    assert C.sizeof(binding.tpc_params_t) == 4 * (2 + 152 + 16 + 3 + 5)


def test_strerror_and_version():
    lib = binding.load()
    assert lib.tpc_version().decode().count(".") == 2
    assert lib.tpc_strerror(0) == b"ok"
    assert b"workspace" in lib.tpc_strerror(-2)


def test_grid_bins_matches_formula_R7():
    """n_bins = n_sectors * sum_r max(1, ceil(2 X_r tan10 / cell_y)) * ceil((z_hi-z_lo)/cell_z), in fp32."""
    for p in (config0().params, TpcParams(), TpcParams(cell_y=3.25, cell_z=1.5, z_lo=-300.0, z_hi=251.0)):
        X = np.asarray(p.row_x, np.float32)
        ymax = X * np.float32(p.tan_half)
        ny = np.maximum(1, np.ceil((np.float32(2.0) * ymax) / np.float32(p.cell_y))).astype(np.int64)
        nz = int(np.ceil((np.float32(p.z_hi) - np.float32(p.z_lo)) / np.float32(p.cell_z)))
        assert binding.grid_bins(p) == int(p.n_sectors) * int(ny.sum()) * nz


def test_workspace_bytes_monotone_and_invalid_args():
    p = TpcParams()
    a = binding.workspace_bytes(p, 1000, 100)
    b = binding.workspace_bytes(p, 2000, 100)
    c = binding.workspace_bytes(p, 2000, 400)
    assert 0 < a < b < c
    assert a % 256 == 0
    with pytest.raises(binding.TpcError):
        binding.workspace_bytes(p, -1, 100)
    with pytest.raises(binding.TpcError):
        binding.workspace_bytes(p.with_(cell_y=0.0), 10, 10)
    with pytest.raises(binding.TpcError):
        binding.workspace_bytes(p.with_(n_rows=200), 10, 10)
    with pytest.raises(binding.TpcError):   # bins would overflow int32
        binding.workspace_bytes(p.with_(cell_y=0.01, cell_z=0.01, z_lo=-30000.0), 10, 10)


def test_compute_entry_points_reject_bad_arguments_without_a_gpu():
    """NULL workspace / too-small workspace are host-detected return codes; nothing is enqueued."""
    lib = binding.load()
    P = binding.make_params(TpcParams())
    null = C.c_void_p(0)
    rc = lib.tpc_grid_build(C.byref(P), C.c_int64(10), C.c_int64(10), null, null, null, null, null, null,
                            C.c_size_t(0), null)
    assert rc == -1
    fake = C.c_void_p(256 * 1000)       # aligned, never dereferenced: size check fails first
    rc = lib.tpc_grid_build(C.byref(P), C.c_int64(10), C.c_int64(10), null, null, null, null, null, fake,
                            C.c_size_t(1024), null)
    assert rc == -2


def test_binding_refuses_cpu_tensors():
    import torch
    with pytest.raises(binding.TpcError):
        binding._dp(torch.zeros(4))


@pytest.mark.parametrize("name,mirror", [("tpc_result_t", "tpc_result_t"), ("tpc_merge_params_t", "tpc_merge_params_t"),
                                         ("tpc_merged_t", "tpc_merged_t"), ("tpc_fit_options_t", "tpc_fit_options_t")])
def test_other_struct_layouts_match_header(name, mirror):
    """Field order of the ctypes mirrors == the header's typedefs (pointer structs: one pointer per member)."""
    txt = open(HEADER).read()
    body = re.search(r"typedef struct \{((?:(?!typedef struct).)*?)\} " + name + ";", txt, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if decl:
            fields += [piece.split()[-1].lstrip("*") for piece in decl.split(",")]
    cls = getattr(binding, mirror)
    assert fields == [f[0] for f in cls._fields_]
    if name == "tpc_merge_params_t":
        assert C.sizeof(cls) == 16
    elif name == "tpc_fit_options_t":
        assert C.sizeof(cls) == 4 * len(fields) and all(f[1] is C.c_float for f in cls._fields_)
    else:
        assert C.sizeof(cls) == 8 * len(fields)


def test_merge_refuses_an_odd_number_of_fit_passes_without_a_gpu():
    """R26 reads the fitted states at the innermost hit, where R22 leaves them after an even number of passes only.  With
    every other argument valid an odd n_fit_passes is TPC_EINVAL; the same call with an even one gets as far as the last
    host-side check (merge workspace too small: TPC_ENOMEM_WS).  Nothing is enqueued either way."""
    lib = binding.load()
    fake = 256 * 1000                       # aligned, never dereferenced
    dev = binding.tpc_result_t(*[C.c_void_p(fake)] * len(binding.tpc_result_t._fields_))
    out = binding.tpc_merged_t(*[C.c_void_p(fake)] * len(binding.tpc_merged_t._fields_))
    M = binding.tpc_merge_params_t(50.0, 64.0, 1.0, 12)

    def call(passes):
        P = binding.make_params(TpcParams(n_fit_passes=passes))
        return lib.tpc_merge_tracks(C.byref(P), C.byref(M), C.c_int64(10), C.c_int64(10), C.c_void_p(fake), C.c_size_t(1 << 40),
                                    C.c_void_p(fake), C.c_int64(100), C.byref(dev), C.c_void_p(fake), C.c_size_t(0), C.byref(out),
                                    C.c_void_p(0))

    assert call(2) == -2 and call(4) == -2
    assert call(1) == -1 and call(3) == -1
