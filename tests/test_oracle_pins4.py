"""Pins of the oracle's additional solvers: linearised RK4 (PAPER.md
Eq. 4), Boris-Verlet (Eq. 7-8) and the uniform "parametric" electric field
of Eq. 3 (L172-175).  CPU only.  Solver codes: 0 RKN, 2 RK4, 3 Boris-Verlet (reading R2), 4 Boris
with Eq. 8 as printed."""
import math

import numpy as np
import pytest

import oracle as orc
from paper_2506_15812_b200 import workloads as wl

QM = wl.E_CHARGE / wl.MASS_LI7
V0 = math.sqrt(2 * 60e3 * wl.E_CHARGE / wl.MASS_LI7)
SOLOVEV = (wl.PSI_A, wl.R0, wl.A_MINOR, wl.KAPPA, wl.B_T)


def uniform(B, E=(0, 0, 0)):
    return orc.OracleField(kind=orc.KIND_UNIFORM, par=B, E=E)


def solovev(E=(0, 0, 0)):
    return orc.OracleField(kind=orc.KIND_SOLOVEV, par=SOLOVEV, E=E)


def angle(a, b):
    """signed angle from a to b in the x-y plane"""
    return math.atan2(a[0] * b[1] - a[1] * b[0], a[0] * b[0] + a[1] * b[1])


# ---- P13: linearised RK4 (Eq. 4) ---------------------------------------------------------
@pytest.mark.parametrize("dt", [1e-9, 5e-9])
def test_p13_rk4_one_step_closed_form_uniform_B(dt):
    """Uniform B = B z: w = vx + i vy obeys dw/dt = -i Omega w, so one RK4 step multiplies w by
    1 + L + L^2/2 + L^3/6 + L^4/24 (L = -i Omega dt) and moves the position by
    w dt (1 + L/2 + L^2/6 + L^3/24) -- the Taylor polynomials of exp(L) and (exp(L)-1)/L."""
    B = 1.15
    f = uniform((0, 0, B))
    L = -1j * QM * B * dt
    v0, r0 = np.array([3e5, -4e5, 1.7e5]), np.array([0.7, 0.0, 0.0])
    r, v, _ = orc.rkn_advance(f, QM, r0, v0, 0.0, dt, 1, 2)
    w0 = v0[0] + 1j * v0[1]
    w1 = w0 * (1 + L + L ** 2 / 2 + L ** 3 / 6 + L ** 4 / 24)
    d = w0 * dt * (1 + L / 2 + L ** 2 / 6 + L ** 3 / 24)
    assert abs(v[0] - w1.real) < 2e-10 and abs(v[1] - w1.imag) < 2e-10       # |v| ~ 5e5: 4e-16 rel
    assert abs(r[0] - r0[0] - d.real) < 3e-16 and abs(r[1] - r0[1] - d.imag) < 3e-16
    assert v[2] == v0[2] and r[2] == r0[2] + v0[2] * dt
    z = QM * B * dt
    amp2 = (v[0] ** 2 + v[1] ** 2) / (v0[0] ** 2 + v0[1] ** 2)
    assert abs(amp2 - (1 - z ** 6 / 72 + z ** 8 / 576)) < 8e-16


def test_p13_rk4_uniform_E_parabola_exact():
    """B = 0, uniform E (paper scenario 2, L279): every stage sees the same acceleration, so RK4
    reproduces r0 + v0 t + a t^2/2 to rounding."""
    E = (10.0, -20.0, 1e3)
    f = uniform((0, 0, 0), E)
    r0, v0 = np.array([0.1, 0.2, 0.3]), np.array([1e3, 2e3, -5e2])
    n, dt = 200, 1e-8
    r, v, t = orc.rkn_advance(f, QM, r0, v0, 0.0, dt, n, 2)
    a = QM * np.array(E)
    T = n * dt
    assert np.abs(r - (r0 + v0 * T + 0.5 * a * T * T)).max() < 1e-13
    assert np.abs(v - (v0 + a * T)).max() < 1e-9


def test_p13_rk4_order_four_and_agrees_with_rkn():
    """Step halving in the analytic Solov'ev field: state error falls 16x per halving (4th order,
    L210), and RK4 and RKN differ by O(dt^4) only (both consistent to 4th order)."""
    f = solovev()
    T = 2e-7
    r_ref, _, _ = orc.rkn_advance(f, QM, [0.72, 0.003, 0.01], [-V0, 0, 0], 0.0, T / 200000, 200000, 0)
    err = []
    for n in (200, 400, 800):
        r, _, _ = orc.rkn_advance(f, QM, [0.72, 0.003, 0.01], [-V0, 0, 0], 0.0, T / n, n, 2)
        err.append(np.linalg.norm(r - r_ref))
    for a, b in zip(err, err[1:]):
        assert 3.9 < math.log2(a / b) < 4.15
    assert err[0] < 1e-10                                  # 8.1e-11 m at dt = 1e-9
    r_n, _, _ = orc.rkn_advance(f, QM, [0.72, 0.003, 0.01], [-V0, 0, 0], 0.0, T / 200, 200, 0)
    r_k, _, _ = orc.rkn_advance(f, QM, [0.72, 0.003, 0.01], [-V0, 0, 0], 0.0, T / 200, 200, 2)
    assert 1e-12 < np.linalg.norm(r_n - r_k) < 3e-10       # different schemes, same order


# ---- P14: Boris (Eq. 7-8) ----------------------------------------------------------------
@pytest.mark.parametrize("dt", [1e-9, 2e-8])
def test_p14_boris_rotation_exact_in_uniform_B(dt):
    """Eq. 7 in uniform B is an exact rotation of v_perp by 2 atan(Omega dt / 2) for ANY dt
    ("ensures the conservation of kinetic energy at every time step", L262), v_par untouched;
    the printed position update is r0 + v(t0) dt, the Verlet one r0 + v' dt (reading R2)."""
    B = 1.15
    f = uniform((0, 0, B))
    z = QM * B * dt
    v0, r0 = np.array([3e5, -4e5, 1.7e5]), np.array([0.7, 0.0, 0.0])
    r, v, _ = orc.rkn_advance(f, QM, r0, v0, 0.0, dt, 1, 4)
    assert abs((v @ v) / (v0 @ v0) - 1) < 5e-16
    assert abs(-angle(v0, v) - 2 * math.atan(z / 2)) < 1e-15
    assert v[2] == v0[2]
    assert np.abs(r - (r0 + v0 * dt)).max() < 2e-16
    # solver 3: leap-frog start = push over -dt/2, then one push over dt
    r3, v3, _ = orc.rkn_advance(f, QM, r0, v0, 0.0, dt, 1, 3)
    assert abs(-angle(v0, v3) - (2 * math.atan(z / 2) - 2 * math.atan(z / 4))) < 1e-15
    assert np.abs(r3 - (r0 + v3 * dt)).max() < 2e-16
    assert abs((v3 @ v3) / (v0 @ v0) - 1) < 5e-16


def test_p14_boris_conserves_speed_in_tokamak_field():
    """Pure B, non-uniform (analytic Solov'ev): |v| changes only by rounding, a few ulp per step
    -- against the RK solvers' (Omega dt)^6/72 per step (pin P5)."""
    f = solovev()
    for solver in (3, 4):
        r, v, _ = orc.rkn_advance(f, QM, [0.72, 0.003, 0.01], [-V0, 0, 0], 0.0, 1e-9, 5000, solver)
        assert abs(math.sqrt(v @ v) / V0 - 1) < 5000 * 4 * 2.3e-16


def test_p14_boris_parallel_E_and_ExB_drift():
    """Paper scenario 5 (L282): B = (0,0,B), E = (0,0,Ez): v_z gains (q/m) Ez dt per step exactly.
    E = (Ex,0,0) perpendicular to B: the gyro-averaged drift is E x B / B^2 = -(Ex/B) y; the
    Boris push reproduces it for any dt (known property of the scheme)."""
    B, Ez = 1.0, 0.1
    f = uniform((0, 0, B), (0, 0, Ez))
    n, dt = 300, 1e-9
    r, v, _ = orc.rkn_advance(f, QM, [0, 0, 0], [1e5, 0, 2e3], 0.0, dt, n, 4)
    assert abs(v[2] - (2e3 + QM * Ez * n * dt)) < 1e-9
    Ex = 2e4
    f = uniform((0, 0, B), (Ex, 0, 0))
    period = 2 * math.pi / (QM * B)
    dt = period / 64
    n = 64 * 50                                                 # 50 numerical gyrations (phase error aside)
    r, v, _ = orc.rkn_advance(f, QM, [0, 0, 0], [1e5, 0, 0], 0.0, dt, n, 3)
    # drift over many periods; residual = at most one gyro-diameter of the drift-frame orbit
    rho = (1e5 + Ex / B) / (QM * B)
    assert abs(r[1] - (-(Ex / B) * n * dt)) < 2.2 * rho
    assert abs(r[1]) > 20 * rho


def test_p14_boris_orders_second_vs_first():
    """Reading R2: Verlet form with the leap-frog start is 2nd order ("a second-order Verlet
    solver", L249); Eq. 8 exactly as printed (old velocity) is 1st order, 1.3 mm off after 200 ns
    at dt = 1e-9 s."""
    f = solovev()
    T = 2e-7
    r_ref, _, _ = orc.rkn_advance(f, QM, [0.72, 0.003, 0.01], [-V0, 0, 0], 0.0, T / 200000, 200000, 0)
    for solver, order, e0 in ((3, 2.0, 4.8e-6), (4, 1.0, 1.3e-3)):
        err = []
        for n in (200, 400, 800):
            r, _, _ = orc.rkn_advance(f, QM, [0.72, 0.003, 0.01], [-V0, 0, 0], 0.0, T / n, n, solver)
            err.append(np.linalg.norm(r - r_ref))
        for a, b in zip(err, err[1:]):
            assert abs(math.log2(a / b) - order) < 0.05
        assert abs(err[0] / e0 - 1) < 0.05


# ---- P15: the solvers agree as dt -> 0 --------------------------------------
def test_p15_solvers_agree_at_small_dt_on_detector_hit():
    """'the results of the solvers differ only in the eighth decimal position' at the smallest
    step (L294): traced to the detector plane in the spline field of config 1, the hit of RKN,
    RK4 and Boris-Verlet converges to the same point; differences shrink with dt at each
    solver's order."""
    cfg = wl.config(1, n_override=8)
    grid, nodal = cfg.field_builder()
    f = orc.OracleField(grid, nodal)
    g = cfg.groups[0]
    st = orc.seed(g.beam, wl.depth_cdf(), wl.normal_cdf(), cfg.seed, 0, 8)
    qm = g.beam.charge_C / g.beam.mass_kg
    hits = {}
    for solver in (0, 2, 3):
        for dt in (1e-9, 1e-10, 1e-11):
            res = orc.trace(f, qm, st, None, dt, int(5e-6 / dt), cfg.detector, solver)
            hits[solver, dt] = (res["status"].copy(), res["u"].copy(), res["w"].copy())
    ok = np.ones(8, bool)
    for k, (s, u, w) in hits.items():
        ok &= s == 0
    assert ok.sum() >= 6
    def dist(a, b):
        return np.hypot(hits[a][1][ok] - hits[b][1][ok], hits[a][2][ok] - hits[b][2][ok]).max()
    assert dist((0, 1e-11), (2, 1e-11)) < 1e-9             # RKN vs RK4: both limited by the O(dt^2) plane interpolation
    assert dist((0, 1e-11), (3, 1e-11)) < 2e-9
    assert dist((0, 1e-9), (3, 1e-9)) > 100 * dist((0, 1e-11), (3, 1e-11)) * 0.5
    assert dist((0, 1e-9), (0, 1e-11)) < 5e-6               # RKN at the production step: micrometres (L296-306)
