"""Tracker parameters as plain values (no arithmetic of the method lives here).

`TpcParams` is the Python-side image of the host POD `tpc_params_t` declared in
`include/tpc_b200.h`; the CUDA binding and the CPU oracle each build
their own C struct from it, so the two never share a header.  Every field is an *input*
of the method: geometry (R1, R2), field constant (R4), measurement errors (R6), grid cell
(R7) and the cuts of R9-R22.  `row_x` is stored as float32 so both sides read bit-identical
pad-row positions.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np

N_ROWS = 152
SECTORS_PER_SIDE = 18
B_TESLA = 0.5
#: kB = 0.299792458e-2 * B[T]  (cm^-1 GeV), SURVEY.md R4
KB = 0.299792458e-2 * B_TESLA
#: drift velocity in cm/us (BASELINE.json configs[2])
V_DRIFT = 2.58


def default_row_x() -> np.ndarray:
    """X_r = 85 + r*160/151 cm, r = 0..151, rounded once to float32."""
    r = np.arange(N_ROWS, dtype=np.float64)
    return (85.0 + r * 160.0 / 151.0).astype(np.float32)


@dataclass(frozen=True)
class TpcParams:
    n_sectors: int = 36
    n_rows: int = N_ROWS
    row_x: np.ndarray = field(default_factory=default_row_x)
    tan_half: float = float(np.float32(math.tan(math.radians(10.0))))
    kB: float = float(np.float32(KB))
    sigma_y: float = float(np.float32(0.08))
    sigma_z: float = float(np.float32(0.10))
    z_lo: float = -1.0
    z_hi: float = 251.0
    cell_y: float = 2.0
    cell_z: float = 2.0
    ca_max_dydx: float = 2.0
    ca_max_dzdx: float = 2.5
    ca_cut: float = 20.0
    chi2_cut: float = 16.0
    chi2_chain_cut: float = 30.0
    win_max: float = 5.0
    max_sinphi: float = float(np.float32(0.95))
    edge_margin: float = 1.0
    max_gap: int = 4
    min_hits: int = 10
    n_fit_passes: int = 2
    cov0: tuple = (1.0, 1.0, 1.0, 10.0, 100.0)

    def with_(self, **kw) -> "TpcParams":
        return replace(self, **kw)
