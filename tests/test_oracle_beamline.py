"""Pins of the oracle's R24 (closest approach to the beam line, z there, time offset; R24) against what
geometry fixes -- none of them re-uses the oracle's own formula:
  * generator truth: a noiseless helix thrown from (0, 0, vz) at azimuth phi and collision time t is fitted by the
    oracle; R24 must return phi0 = phi, z0 = vz - v_d t, dca = 0, t0 = t (vz = 0) -- the generator is an independent
    global-frame circle tracer;
  * brute force: dense sampling of the circle through a random displaced state, arg-min of the distance to the origin;
  * straight-line closed form (q/pT = 0);
  * A/C mirror symmetry (R2, R5).
"""
import math

import numpy as np
import pytest

from paper_2106_03636_b200.synth import V_DRIFT, TpcParams, single_helix

from helix_ref import KB_TRK

PARAMS = TpcParams()


def _one(orc, y, dz, s, tl, q, xref, zref, sector):
    par = np.array([[y], [dz], [s], [tl], [q]], np.float32)
    o = orc.beamline(PARAMS, par, [xref], [zref], [sector], V_DRIFT)
    return {k: float(v[0]) for k, v in o.items()}


@pytest.mark.parametrize("qpt,phi_deg,tanl,vz,t_us", [(1.0, 10.0, 0.5, 0.0, 0.0), (-2.5, 3.0, 0.9, 3.0, 0.0),
                                                     (0.2, 12.0, 0.05, -4.0, 0.0), (3.0, 19.0, 0.3, 0.0, 40.0),
                                                     (-0.25, 4.0, 1.0, 0.0, 7.5), (-3.0, 1.0, 0.7, 0.0, 25.0)])
def test_R24_recovers_generating_vertex_direction_and_time(orc, qpt, phi_deg, tanl, vz, t_us):
    ev = single_helix(qpt, math.radians(phi_deg), tanl, vz=vz, t_us=t_us)
    o = orc.run(ev.params, ev.y, ev.z, ev.sector_row, "f32", True)
    assert o["trk_seed"].size == 1
    b = orc.beamline(ev.params, o["par"], o["xref"], o["zref"], np.zeros(1, np.int32), V_DRIFT)   # single-sector geometry: sector 0
    dphi = (float(b["phi0"][0]) - math.radians(phi_deg) + math.pi) % (2 * math.pi) - math.pi
    assert abs(dphi) < 2e-4                                  # fp32 fit of a noiseless helix
    assert float(b["dca"][0]) < 2e-2
    assert float(b["z0"][0]) == pytest.approx(vz - V_DRIFT * t_us, abs=2e-2)
    if vz == 0.0:
        assert float(b["t0"][0]) == pytest.approx(t_us, abs=1e-2)


def test_R24_equals_brute_force_closest_point_on_the_circle(orc):
    rng = np.random.default_rng(24)
    for _ in range(40):
        x = 85.0 + rng.uniform(0, 100)
        y, s, tl = rng.uniform(-25, 25), rng.uniform(-0.8, 0.8), rng.uniform(-1, 1)
        q = rng.choice([-1, 1]) * rng.uniform(0.1, 4.0)
        zref, dz = rng.uniform(-2e4, 2e4), rng.uniform(-1, 1)
        sector = int(rng.integers(0, 36))
        out = _one(orc, y, dz, s, tl, q, x, zref, sector)
        # independent parametrisation: walk the circle by turning angle w from the state (float32 inputs as the oracle saw them)
        y, dz, s, tl, q, x, zref = (float(np.float32(v)) for v in (y, dz, s, tl, q, x, zref))
        kap = -KB_TRK * q
        phi = math.asin(s)
        w = np.linspace(-math.pi, math.pi, 2_000_001)
        px = x + (np.sin(phi + w) - math.sin(phi)) / kap
        py = y - (np.cos(phi + w) - math.cos(phi)) / kap
        d = np.hypot(px, py)
        i = int(np.argmin(d))
        assert out["dca"] == pytest.approx(d[i], abs=2e-3 + 1e-6 * d[i])
        z_at = (zref + dz) + tl * w[i] / kap               # path length in the bending plane = w / kap
        assert out["z0"] == pytest.approx(z_at, abs=2e-3 + abs(tl / kap) * 4e-6 + 4e-3 * abs(zref) / 3e4)
        side = 1.0 if sector < 18 else -1.0
        assert out["t0"] == pytest.approx(-side * out["z0"] / V_DRIFT, rel=1e-6, abs=1e-6)
        alpha = ((sector % 18) + 0.5) * math.radians(20.0)
        dirn = (phi + w[i] + alpha) % (2 * math.pi)
        assert abs((out["phi0"] - dirn + math.pi) % (2 * math.pi) - math.pi) < 1e-5


def test_R24_straight_line_closed_form(orc):
    # q/pT = 0: the line through (x, y) with direction (cos, sin); closest point t* = -(x cos + y sin)
    x, y, s, tl, zabs = 120.0, 7.0, 0.3, -0.4, 55.0
    c = math.sqrt(1 - np.float32(s) ** 2)
    out = _one(orc, y, 0.0, s, tl, 0.0, x, zabs, 0)
    ts = -(x * c + y * float(np.float32(s)))
    assert out["dca"] == pytest.approx(abs(x * float(np.float32(s)) - y * c), rel=1e-6)
    assert out["z0"] == pytest.approx(zabs + float(np.float32(tl)) * ts, rel=1e-6)
    assert out["phi0"] == pytest.approx(math.asin(float(np.float32(s))) + math.radians(10.0), rel=1e-6)


def test_R24_mirror_A_to_C(orc):
    # R2/R5: the C side measures -z with the same drift direction: z -> -z, tanl -> -tanl, sector + 18
    a = _one(orc, 3.0, 0.5, 0.2, 0.7, -1.5, 100.0, 40.0, 4)
    c = _one(orc, 3.0, -0.5, 0.2, -0.7, -1.5, 100.0, -40.0, 22)
    assert c["z0"] == pytest.approx(-a["z0"], rel=1e-6)
    assert c["t0"] == pytest.approx(a["t0"], rel=1e-6)
    assert c["dca"] == a["dca"] and c["phi0"] == a["phi0"]
