"""P23: gridded electric field E(R, Z) of Eq. 3 (E(r); L177: the coordinates "are mapped to a poloidal
cross-section plane in each iteration step.  That is how the local magnetic and electric field is given"; L175: "we can
use parametric modeling for it"; reading E1 in DESIGN.md: E_R, E_Z, E_phi tabulated on the (R, Z) grid like B).  Pinned
against closed forms that do not involve the oracle's arithmetic.  CPU only.

A field that is LINEAR in the coordinates, E_R = kappa R, E_Z = gamma Z, is reproduced exactly by the cubic spline
(cubic precision, P9), has Cartesian components E_X = kappa X, E_Y = kappa Y, and with B = 0 makes every coordinate a
harmonic oscillator (kappa, gamma < 0):  x(t) = x0 cos(w t) + (v0 / w) sin(w t),  w^2 = -(q/m) kappa.  A sign error, a
transposed rotation, a missing q/m or a stage evaluated at the wrong position all break the fourth-order convergence.
"""
import math

import numpy as np
import pytest

import oracle as orc
from paper_2506_15812_b200 import workloads as wl

QM = wl.E_CHARGE / wl.MASS_LI7
W_R, W_Z = 1.0e7, 0.6e7                     # rad/s
KAPPA, GAMMA = -W_R ** 2 / QM, -W_Z ** 2 / QM


def _grid(nR=17, nZ=33):
    grid, _ = wl.nodal_field_2d(nR, nZ)
    R = np.linspace(grid.Rmin, grid.Rmax, grid.nR)[:, None] * np.ones((1, grid.nZ))
    Z = np.ones((grid.nR, 1)) * np.linspace(grid.Zmin, grid.Zmax, grid.nZ)[None, :]
    return grid, R, Z


def _harmonic_field(E_uniform=(0.0, 0.0, 0.0), e_phi=0.0):
    grid, R, Z = _grid()
    return orc.OracleField(kind=10, par=(0.0, 0.0, 0.0), E=E_uniform, E_nodal=(KAPPA * R, GAMMA * Z, e_phi + 0.0 * R), E_grid=grid)


def _exact(r0, v0, t):
    w = np.array([W_R, W_R, W_Z])
    r0, v0 = np.asarray(r0), np.asarray(v0)
    return r0 * np.cos(w * t) + v0 / w * np.sin(w * t), -r0 * w * np.sin(w * t) + v0 * np.cos(w * t)


def test_p23_linear_grid_is_reproduced_exactly_and_rotated_like_B():
    f = _harmonic_field(E_uniform=(3.0, -2.0, 5.0), e_phi=7.0e3)
    rng = np.random.default_rng(5)
    for _ in range(50):
        r = np.array([rng.uniform(0.3, 0.8) * math.cos(a := rng.uniform(-3.0, 3.0)), 0.0, rng.uniform(-0.5, 0.5)])
        Rr = abs(r[0] / math.cos(a)) if abs(math.cos(a)) > 1e-3 else 0.5
        r = np.array([Rr * math.cos(a), Rr * math.sin(a), r[2]])
        e = f.E(r)
        # E_X = E_R c - E_phi s, E_Y = E_R s + E_phi c (O0), plus the uniform vector
        want = np.array([3.0 + KAPPA * r[0] - 7.0e3 * math.sin(a), -2.0 + KAPPA * r[1] + 7.0e3 * math.cos(a), 5.0 + GAMMA * r[2]])
        assert np.allclose(e, want, rtol=0, atol=1e-9 * abs(KAPPA)), (r, e, want)


@pytest.mark.parametrize("solver,order", [(0, 4), (1, 3), (2, 4), (3, 2)])
def test_p23_harmonic_motion_converges_to_the_closed_form(solver, order):
    f = _harmonic_field()
    r0, v0, T = [0.55, 0.02, 0.03], [-2.0e5, 1.0e5, 0.5e5], 4.0e-7          # ~0.6 periods
    errs = []
    for n in (200, 400):
        r, v, _ = orc.rkn_advance(f, QM, r0, v0, 0.0, T / n, n, solver)
        re, ve = _exact(r0, v0, T)
        # Boris (solver 3) carries its velocity at half steps: compare positions only; printed k3 (solver 1): order 3 (P7)
        errs.append(np.abs(r - re).max() if solver == 3 else max(np.abs(r - re).max(), np.abs(v - ve).max() / W_R))
    assert errs[0] < {4: 5e-9, 3: 5e-7, 2: 5e-5}[order], errs
    assert 0.8 * 2 ** order < errs[0] / errs[1] < 1.25 * 2 ** order, (solver, errs)


def test_p23_constant_grid_equals_the_uniform_field():
    """nodal (0, E_Z, 0) constant: the spline reproduces it, so the gridded field IS the uniform field (0, 0, E_Z), whose
    parabola is pinned by P4; trajectories agree to rounding."""
    grid, R, Z = _grid()
    Ez = 2.5e4
    fg = orc.OracleField(kind=10, par=(0.0, 0.0, 1.0), E_nodal=(0.0 * R, Ez + 0.0 * R, 0.0 * R), E_grid=grid)
    fu = orc.OracleField(kind=10, par=(0.0, 0.0, 1.0), E=(0.0, 0.0, Ez))
    for solver in (0, 2, 3, 4):
        a = orc.rkn_advance(fg, QM, [0.6, 0.0, 0.0], [1e5, 2e4, 3e3], 0.0, 1e-9, 500, solver)
        b = orc.rkn_advance(fu, QM, [0.6, 0.0, 0.0], [1e5, 2e4, 3e3], 0.0, 1e-9, 500, solver)
        assert np.abs(a[0] - b[0]).max() < 1e-13 and np.abs(a[1] - b[1]).max() < 1e-7, solver


def test_p23_central_force_conserves_angular_momentum_and_energy():
    """E_R = E0 R0 / R, E_phi = 0 (a line charge): no torque, so L_z = X v_Y - Y v_X is constant, and
    v^2/2 - (q/m) E0 R0 ln R is constant up to the spline error of 1/R, which falls 16 x per grid refinement (h^4, P9)."""
    E0, R0 = -2.0e4, 0.56
    r0, v0 = np.array([0.7, 0.0, 0.0]), np.array([-3.0e5, 2.0e5, 1.0e4])
    dW = []
    for nR, nZ in ((17, 33), (33, 65), (65, 129)):
        grid, R, Z = _grid(nR, nZ)
        f = orc.OracleField(kind=10, par=(0.0, 0.0, 0.0), E_nodal=(E0 * R0 / R, 0.0 * R, 0.0 * R), E_grid=grid)
        r, v, _ = orc.rkn_advance(f, QM, r0, v0, 0.0, 1e-9, 800, 0)
        Lz0, Lz = r0[0] * v0[1] - r0[1] * v0[0], r[0] * v[1] - r[1] * v[0]
        W0 = 0.5 * v0 @ v0 - QM * E0 * R0 * math.log(math.hypot(r0[0], r0[1]))
        W = 0.5 * v @ v - QM * E0 * R0 * math.log(math.hypot(r[0], r[1]))
        assert abs(Lz / Lz0 - 1) < 1e-11, Lz / Lz0 - 1
        dW.append(abs(W - W0) / (0.5 * v0 @ v0))
        assert abs(0.5 * v @ v / (0.5 * v0 @ v0) - 1) > 0.02                          # the field did work on the ion
        assert 0.3 < math.hypot(r[0], r[1]) < 0.85 and np.abs(r - r0).max() > 0.1    # it moved, inside the grid
    assert dW[0] < 5e-6 and dW[2] < 3e-8, dW
    assert dW[0] / dW[1] > 8 and dW[1] / dW[2] > 8, dW


# ---- P24: loss integral with the Bezier plane interpolation (reading L2') -----------------------------------
def test_p24_bezier_fraction_of_the_crossing_step_is_the_exact_time_fraction_on_a_parabola():
    """Uniform E, B = 0: the trajectory is a parabola, which the quadratic Bezier curve through (r_n, v_n), (r_n+1, v_n+1)
    reproduces with tau = (t - t_n)/dt exactly.  With a constant rate every trapezoid is exact, so with the Bezier
    interpolation weight = exp(-nu t_hit) for the EXACT crossing time at any dt, while the linear interpolation's fraction
    lam is off by O(dt^2 a / v) and shows it."""
    grid, nodal = wl.nodal_field_2d(33, 65)
    Ex = 4.0e6                                                   # strong enough to bend the parabola within a step
    f = orc.OracleField(grid, [0.0 * c for c in nodal], E=(Ex, 0.0, 0.0))
    nu0 = 2.5e6
    L = orc.OracleLoss(grid, wl.nodal_psi(grid), 0.0, 1e-3, np.full(5, nu0))
    V0 = math.sqrt(2 * 60e3 * wl.E_CHARGE / wl.MASS_LI7)
    x0 = np.array([0.70, 0.61, 0.8123])
    state = [x0, np.zeros(3), np.array([0.0, 0.01, -0.02]), np.full(3, 0.2 * V0), np.zeros(3), np.zeros(3)]
    det = wl.uniform_detector(0.0, 0.0, 8, 2.5e-3, x_plane=0.82)
    a = QM * Ex
    v0 = 0.2 * V0
    t_hit = (-v0 + np.sqrt(v0 * v0 + 2.0 * a * (0.82 - x0))) / a          # x0 + v0 t + a t^2 / 2 = 0.82
    dev_lin = []
    for dt in (4e-9, 1.3e-9):
        rb = orc.trace_loss(f, L, QM, state, None, dt, 100000, det, interp=1)
        rl = orc.trace_loss(f, L, QM, state, None, dt, 100000, det, interp=0)
        assert np.all(rb["status"] == 0) and np.array_equal(rb["steps"], rl["steps"])
        assert np.abs(rb["weight"] / np.exp(-nu0 * t_hit) - 1).max() < 2e-13
        dev_lin.append(np.abs(rl["weight"] / np.exp(-nu0 * t_hit) - 1).max())
    assert dev_lin[0] > 1e-7 and dev_lin[0] > 4 * dev_lin[1] > 0, dev_lin
