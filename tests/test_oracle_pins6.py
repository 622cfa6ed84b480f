"""Pins of the oracle's NEXT-3 variants: quadratic Bezier plane interpolation
 and deterministic weighted-grid initialisation (L314).  CPU only."""
import math

import numpy as np
import pytest

import oracle as orc
from paper_2506_15812_b200 import workloads as wl

QM = wl.E_CHARGE / wl.MASS_LI7
V0 = math.sqrt(2 * 60e3 * wl.E_CHARGE / wl.MASS_LI7)


# ---- P18: quadratic Bezier interpolation to the plane (reading Z1) -------------------------
def test_p18_bezier_exact_for_uniform_acceleration():
    """B = 0, uniform E: the trajectory is a parabola, which a quadratic Bezier curve through
    (r_n, r_n+1) with control point r_n + v_n dt/2 = r_n+1 - v_n+1 dt/2 reproduces exactly: the hit
    equals the closed form for ANY dt, while the linear chord is off by ~a dt^2/8."""
    grid, nodal = wl.nodal_field_2d(33, 65)
    E = (2e7, 0.0, 5e6)
    f = orc.OracleField(grid, [0.0 * c for c in nodal], E=E)
    state = [np.array([0.6]), np.array([0.0]), np.array([0.0]), np.array([1e5]), np.array([2e4]), np.array([-3e4])]
    det = wl.uniform_detector(0.0, 0.0, 8, 2.5e-3)
    a = QM * np.array(E)
    t = (-1e5 + math.sqrt(1e10 + 2 * a[0] * 0.22)) / a[0]          # 0.6 + 1e5 t + a_x t^2/2 = 0.82
    ye, ze = 2e4 * t, -3e4 * t + 0.5 * a[2] * t * t
    for dt in (1e-8, 3.3e-9):
        r1 = orc.trace(f, QM, state, None, dt, 100000, det, interp=1)
        r0 = orc.trace(f, QM, state, None, dt, 100000, det, interp=0)
        assert abs(r1["u"][0] - ye) < 1e-15 and abs(r1["w"][0] - ze) < 1e-15
        assert abs(r0["w"][0] - ze) > 1e-8
        assert r1["steps"][0] == r0["steps"][0] and r1["status"][0] == 0


def test_p18_bezier_equals_linear_on_straight_lines():
    grid, nodal = wl.nodal_field_2d(33, 65)
    f = orc.OracleField(grid, [0.0 * c for c in nodal])
    state = [np.array([0.6, 0.7]), np.zeros(2), np.array([0.01, -0.02]), np.full(2, V0), np.array([3e4, -1e4]), np.array([1e4, 2e4])]
    det = wl.uniform_detector(0.0, 0.0, 8, 2.5e-3)
    r1 = orc.trace(f, QM, state, None, 1e-9, 100000, det, interp=1)
    r0 = orc.trace(f, QM, state, None, 1e-9, 100000, det, interp=0)
    assert np.abs(r1["u"] - r0["u"]).max() < 1e-16 and np.abs(r1["w"] - r0["w"]).max() < 1e-16


def test_p18_bezier_third_order_in_the_tokamak_field():
    """'The difference is negligible if we choose the right time step value' (L338): with RKN the
    linear hit converges at order 2 (3.7 um at dt = 1e-9 s), the Bezier hit at order 3 (0.2 nm)."""
    cfg = wl.config(1, n_override=8)
    grid, nodal = cfg.field_builder()
    f = orc.OracleField(grid, nodal)
    g = cfg.groups[0]
    st = orc.seed(g.beam, wl.depth_cdf(), wl.normal_cdf(), cfg.seed, 0, 8)
    ref = orc.trace(f, QM, st, None, 2e-11, 250000, cfg.detector, interp=1)
    ok = ref["status"] == 0
    assert ok.sum() >= 6
    for interp, order, e1 in ((0, 2.0, 3.7e-6), (1, 3.0, 1.7e-10)):
        e = []
        for dt in (2e-9, 1e-9, 5e-10):
            r = orc.trace(f, QM, st, None, dt, int(5e-6 / dt), cfg.detector, interp=interp)
            e.append(np.hypot(r["u"][ok] - ref["u"][ok], r["w"][ok] - ref["w"][ok]).max())
        assert abs(math.log2(e[0] / e[2]) / 2 - order) < 0.35, (interp, e)
        assert 0.5 < e[1] / e1 < 2.0, (interp, e)
