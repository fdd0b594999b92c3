"""Harness-side double-precision helix algebra, independent of the oracle.

Textbook closed forms of a circle of signed curvature kappa = -kB*q/pT in a sector-local frame:
    sin(phi)(X) = s0 + kappa (X - x0)
    y(X)        = y0 + (cos(phi0) - cos(phi(X))) / kappa
    z(X)        = z0 + tanl * (asin s(X) - asin s0) / kappa
They are NOT the chord/arc formulas the tracker uses (R12), which is what makes them a pin.
"""
import math

import numpy as np

from paper_2106_03636_b200.synth import KB, TpcParams

#: the tracker's field constant is the float32-rounded kB of tpc_params_t; the generator uses the exact double
KB_TRK = TpcParams().kB


def alpha_of(sector):
    return ((sector % 18) + 0.5) * math.radians(20.0)


def truth_state_local(qpt, phi, tanl, vx, vy, vz, sector, X):
    """Local state (y, z, sinphi, tanl, qpt) of the first outgoing crossing of x_local = X (A side)."""
    a = alpha_of(sector)
    kap = -KB * qpt
    vxl = vx * math.cos(a) + vy * math.sin(a)
    vyl = -vx * math.sin(a) + vy * math.cos(a)
    phil = phi - a
    S = math.sin(phil) + kap * (X - vxl)
    c2 = math.sqrt(1.0 - S * S)
    dphi = math.asin(S) - phil
    dphi = (math.fmod(dphi * np.sign(kap), 2 * math.pi) + 2 * math.pi) % (2 * math.pi) * np.sign(kap)
    s = dphi / kap
    y = vyl - (c2 - math.cos(phil)) / kap
    return np.array([y, vz + tanl * s, S, tanl, qpt])


def model_yz(theta, x0, X):
    """theta = (y0, z0, sinphi0, tanl, qpt) at x0 -> (y, z) at rows X (closed form, vectorised)."""
    y0, z0, s0, tl, q = theta
    kap = -KB_TRK * q
    s = s0 + kap * (X - x0)
    c0 = math.sqrt(1.0 - s0 * s0)
    c = np.sqrt(1.0 - s * s)
    if abs(kap) < 1e-12:
        return y0 + (X - x0) * s0 / c0, z0 + tl * (X - x0) / c0
    return y0 + (c0 - c) / kap, z0 + tl * (np.arcsin(s) - math.asin(s0)) / kap


def to_beamline(par, xref, zabs, sector):
    """R23: extrapolate a local state to the point of closest approach to the beam line.

    Returns (phi0_global, z0, dca).  par = (y, *, sinphi, tanl, qpt); zabs = absolute z at xref.
    """
    y, _, s, tl, q = par
    c = math.sqrt(1.0 - s * s)
    kap = -KB_TRK * q
    xc, yc = xref - s / kap, y + c / kap
    rc = math.hypot(xc, yc)
    R = 1.0 / abs(kap)
    px, py = xc * (1.0 - R / rc), yc * (1.0 - R / rc)
    phip = math.atan2(-(xc - px) * kap, (yc - py) * kap)
    dphi = math.asin(s) - phip
    dphi = (dphi + math.pi) % (2 * math.pi) - math.pi
    z0 = zabs - tl * dphi / kap
    return (phip + alpha_of(sector)) % (2 * math.pi), z0, abs(rc - R)
