"""Synthetic TPC digits (pad, time bin, ADC) from an Event's clusters: the input recipe of the clusterizer
(R27; the clusterizer is the step that feeds the tracker).

Every cluster deposits its charge q on the pads and time bins around it with a separable Gaussian response
(sigma_pad pads, sigma_time bins); the deposits of all clusters add up per (sector, row, pad, time bin); the ADC value
is the floor of the sum; values below `threshold` are suppressed (zero suppression).  The digit list is shuffled.
Coordinates: pad u = (y + ymax_row) / pad_width, time v = (zeta - z_lo) / time_width with zeta = side * z (R2) -- the
digit (p, t) covers u in [p, p+1), v in [t, t+1).  No tracker or clusterizer arithmetic lives here.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .params import N_ROWS, SECTORS_PER_SIDE


@dataclass
class Digits:
    sector_row: np.ndarray   # int32
    pad: np.ndarray          # int32
    time: np.ndarray         # int32
    adc: np.ndarray          # int32
    pad_width: float         # cm
    time_width: float        # cm of drift per time bin
    n_deposits: int

    @property
    def n(self) -> int:
        return int(self.adc.shape[0])


def digitize(ev, pad_width=0.5, time_width=0.25, sigma_pad=0.45, sigma_time=0.55, threshold=3, seed=0, window=2,
             shuffle=True) -> Digits:
    p = ev.params
    nrows = int(p.n_rows)
    rx = np.asarray(p.row_x, np.float64)
    sr = ev.sector_row.astype(np.int64)
    row = sr % nrows
    side = np.where(sr // nrows < SECTORS_PER_SIDE, 1.0, -1.0) if int(p.n_sectors) > 1 else np.ones(sr.size)
    u = (ev.y.astype(np.float64) + rx[row] * float(p.tan_half)) / pad_width
    v = (side * ev.z.astype(np.float64) - float(p.z_lo)) / time_width
    q = ev.q.astype(np.float64)
    p0, t0 = np.floor(u).astype(np.int64), np.floor(v).astype(np.int64)
    keys, vals = [], []
    for dp in range(-window, window + 1):
        wp = np.exp(-0.5 * ((p0 + dp + 0.5 - u) / sigma_pad) ** 2)
        for dt in range(-window, window + 1):
            wt = np.exp(-0.5 * ((t0 + dt + 0.5 - v) / sigma_time) ** 2)
            pp, tt_ = p0 + dp, t0 + dt
            ok = (pp >= 0) & (tt_ >= 0) & (pp < 65536)
            keys.append(((sr[ok] << 40) | (tt_[ok] << 16) | pp[ok]))
            vals.append((q * wp * wt)[ok] / (2.0 * np.pi * sigma_pad * sigma_time))
    keys = np.concatenate(keys); vals = np.concatenate(vals)
    order = np.argsort(keys, kind="stable")
    keys, vals = keys[order], vals[order]
    first = np.r_[True, keys[1:] != keys[:-1]]
    start = np.nonzero(first)[0]
    adc = np.floor(np.add.reduceat(vals, start)).astype(np.int64)
    k = keys[start]
    keep = adc >= threshold
    k, adc = k[keep], adc[keep]
    if shuffle:
        perm = np.random.Generator(np.random.PCG64(seed)).permutation(k.size)
        k, adc = k[perm], adc[perm]
    return Digits(sector_row=(k >> 40).astype(np.int32), pad=(k & 0xFFFF).astype(np.int32),
                  time=((k >> 16) & 0xFFFFFF).astype(np.int32), adc=adc.astype(np.int32), pad_width=float(pad_width),
                  time_width=float(time_width), n_deposits=int(sr.size))
