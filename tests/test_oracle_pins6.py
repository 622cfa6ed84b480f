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


# ---- P19: deterministic weighted-grid initialisation (L314, reading D1) ----------------------
def _li_beam():
    return wl.config(1).groups[0].beam


def test_p19_grid_weights_sum_to_one_and_marginals_are_cdf_increments():
    beam = _li_beam()
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    nd, nT, nZ = 50, 7, 9
    st, w0 = orc.seed_grid(beam, cd, cn, nd, nT, nZ, beam.z_max, 0, nd * nT * nZ)
    assert abs(w0.sum() - 1.0) < 1e-13 and np.all(w0 >= 0)
    W = w0.reshape(nd, nT, nZ)
    # depth marginal = increments of the tabulated CDF at the cell edges (linear between table points)
    edges = np.linspace(0.0, beam.depth_max, nd + 1)
    F = np.interp(edges, np.linspace(0.0, beam.depth_max, len(cd)), cd)
    assert np.abs(W.sum(axis=(1, 2)) - np.diff(F)).max() < 1e-15
    zc = np.linspace(-beam.z_max, beam.z_max, len(cn))
    PhiT = np.interp(np.linspace(-beam.z_max, beam.z_max, nT + 1), zc, cn)
    assert np.abs(W.sum(axis=(0, 2)) - np.diff(PhiT)).max() < 1e-15
    # truncated exponential with lambda = 2 cm: the first cell holds (1 - e^{-dd/lam}) / (1 - e^{-dmax/lam})
    dd = beam.depth_max / nd
    assert abs(W.sum(axis=(1, 2))[0] - (1 - math.exp(-dd / 0.02)) / (1 - math.exp(-beam.depth_max / 0.02))) < 1e-6   # linear interpolation of the table between its points
    # positions: cell centres on the beam frame; velocities along the axis; index i = (k nT + a) nZ + b
    x, y, z, vx, vy, vz = st
    k, a, b = 17, 3, 5
    i = (k * nT + a) * nZ + b
    assert abs(x[i] - (0.78 - (k + 0.5) * dd)) < 1e-15
    assert abs(y[i] - beam.sigma_pos_m * ((a + 0.5) * 2 * beam.z_max / nT - beam.z_max)) < 1e-16
    assert abs(z[i] - beam.sigma_pos_m * ((b + 0.5) * 2 * beam.z_max / nZ - beam.z_max)) < 1e-16
    assert np.all(vx == -V0) and np.all(vy == 0) and np.all(vz == 0)
    # sharding: a sub-range reproduces the same ions
    st2, w2 = orc.seed_grid(beam, cd, cn, nd, nT, nZ, beam.z_max, 1000, 77)
    assert np.array_equal(w2, w0[1000:1077]) and np.array_equal(st2[2], z[1000:1077])


def test_p19_weighted_grid_image_agrees_with_the_stochastic_one():
    """Both initialisations sample the same ionisation density (L314), so the weighted detector
    image of the grid run agrees with the image of the stochastic run within sampling error."""
    cfg = wl.config(1)
    grid, nodal = cfg.field_builder()
    f = orc.OracleField(grid, nodal)
    g = cfg.groups[0]
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    n = 40000
    st = orc.seed(g.beam, cd, cn, 123, 0, n)
    rs = orc.trace(f, QM, st, None, cfg.dt, cfg.max_steps, cfg.detector)
    cs = rs["status"] == 0
    nd, nT, nZ = 200, 15, 15
    sg, w0 = orc.seed_grid(g.beam, cd, cn, nd, nT, nZ, 4.0, 0, nd * nT * nZ)
    rg = orc.trace(f, QM, sg, None, cfg.dt, cfg.max_steps, cfg.detector)
    cg = rg["status"] == 0
    W = w0[cg].sum()
    # crossing fraction
    p_s, p_g = cs.mean(), W / w0.sum()
    assert abs(p_s - p_g) < 4 * math.sqrt(p_s * (1 - p_s) / n) + 2e-3
    # first and second moments of the hit distribution on the plane
    for key in ("u", "w"):
        m_s, s_s = rs[key][cs].mean(), rs[key][cs].std()
        m_g = (w0[cg] * rg[key][cg]).sum() / W
        s_g = math.sqrt((w0[cg] * (rg[key][cg] - m_g) ** 2).sum() / W)
        assert abs(m_s - m_g) < 4 * s_s / math.sqrt(cs.sum()) + 0.02 * s_s, (key, m_s, m_g)
        assert abs(s_s / s_g - 1) < 0.05, (key, s_s, s_g)
