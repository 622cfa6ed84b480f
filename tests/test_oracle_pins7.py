"""Pins of what round 1 left unpinned: the stage-time arguments of the integrators in a
time-dependent field (reading A3: t, t+dt/2, t+dt/2, t+dt and t <- t+dt; PAPER.md L227-233 prints t0 in every
stage) and the treatment of invalid weights in the fixed-point counters (reading L3).  CPU only.

P20.  A kind-1 table made of two slices of spatially UNIFORM B_Z: the spline reproduces constants exactly and
the time blend is linear, so B_Z(t) = B0 + (B1 - B0) (t - s0)/ds exactly, everywhere.  Then dv/dt = (q/m) v x B
rotates v about Z by the closed-form angle  theta(T) = -(q/m) (B0 T + (B1 - B0) T^2 / (2 ds))  (|v| constant),
with no reference to the oracle's own arithmetic.  A fourth-order scheme with the right stage times converges
at order 4; evaluating every stage at t (or not advancing t) leaves an O(dt) error in theta.
"""
import math

import numpy as np
import pytest

import oracle as orc
from paper_2506_15812_b200 import workloads as wl

QM = wl.E_CHARGE / wl.MASS_LI7
V0 = math.sqrt(2 * 60e3 * wl.E_CHARGE / wl.MASS_LI7)
B0, B1, DS = 1.0, 2.0, 1e-6


def _field():
    grid, nodal = wl.nodal_field_time_slices(9, 17, 2)
    grid.s0, grid.ds = 0.0, DS
    nod = [np.zeros_like(nodal[0]), np.zeros_like(nodal[1]), np.zeros_like(nodal[2])]
    nod[1][0], nod[1][1] = B0, B1                       # B_Z of slice 0 and of slice 1
    return orc.OracleField(grid, nod)


def _theta(t_a, t_b):
    """closed form: - (q/m) integral of B_Z(t) dt over [t_a, t_b]"""
    F = lambda t: B0 * t + (B1 - B0) * t * t / (2.0 * DS)
    return -QM * (F(t_b) - F(t_a))


def test_p20_field_is_exactly_linear_in_time_and_uniform_in_space():
    f = _field()
    rng = np.random.default_rng(0)
    for _ in range(50):
        R, Z, t = rng.uniform(0.3, 0.85), rng.uniform(-0.6, 0.6), rng.uniform(0.0, DS)
        b = f.cyl(R, Z, t)
        assert b[0] == 0.0 and b[2] == 0.0
        assert abs(b[1] - (B0 + (B1 - B0) * t / DS)) < 4e-16


@pytest.mark.parametrize("solver", [0, 1, 2])
def test_p20_rotation_angle_converges_at_order_four_only_with_the_right_stage_times(solver):
    """RKN (both k3 readings: B does not depend on position here, so they coincide) and RK4 (Eq. 4)."""
    f = _field()
    t_a, T = 1.0e-7, 4.0e-7                                     # a start time other than the slice origin
    r0, v0 = (0.55, 0.0, 0.0), (V0 * math.cos(0.3), V0 * math.sin(0.3), 2.0e4)
    th = _theta(t_a, t_a + T)
    errs = []
    for n in (100, 200, 400):
        r, v, t = orc.rkn_advance(f, QM, r0, v0, t_a, T / n, n, variant=solver)
        assert abs(t - (t_a + T)) < 1e-18
        ang = math.atan2(v[1], v[0]) - 0.3
        d = (ang - th + math.pi) % (2 * math.pi) - math.pi      # angle error
        errs.append(abs(d))
        z = QM * (B0 + (B1 - B0) * (t_a + T) / DS) * (T / n)    # RK4 in a uniform field damps |v| by 1 - z^6/72 per step (pin P2)
        assert abs(math.hypot(v[0], v[1]) / V0 - 1.0) < n * z ** 6 / 72 + 1e-12 and v[2] == 2.0e4
    # order 4 (ratio 16 per halving).  With `t` in every stage the error is first order:
    # d(theta) ~ (q/m)(B1-B0)/ds * dt * T / 2 = 1.1e-2 rad at n = 100 -- four orders above what is allowed here.
    assert errs[0] < 2e-6, errs
    for a, b in zip(errs, errs[1:]):
        assert 12.0 < a / b < 20.0, errs


def test_p20_wrong_stage_times_would_be_first_order():
    """The size of the effect the pin guards against, from the closed form alone: a scheme that freezes B at the
    start of each step accumulates theta_frozen = -(q/m) sum B(t_n) dt, off by (q/m)(B1-B0) T dt / (2 ds)."""
    t_a, T, n = 1.0e-7, 4.0e-7, 100
    dt = T / n
    frozen = -QM * sum((B0 + (B1 - B0) * (t_a + k * dt) / DS) * dt for k in range(n))
    assert abs((frozen - _theta(t_a, t_a + T)) - QM * (B1 - B0) * T * dt / (2 * DS)) < 1e-9
    assert abs(frozen - _theta(t_a, t_a + T)) > 1e-2


@pytest.mark.parametrize("solver", [3, 4])
def test_p20_boris_takes_B_at_the_start_of_the_step(solver):
    """Eq. 7-8 (reading R2: B at r(t0), t0).  A Boris push in a field along Z rotates v by EXACTLY
    2 atan((q/m) B h / 2), so the angle after n steps is a closed-form sum over B(t_n): solver 3 (leap-frog start
    over -dt/2 at t0, then n pushes), solver 4 (n pushes).  B(t_n + dt/2) or B(t_n + dt) would differ at O(dt)."""
    f = _field()
    t_a, n, dt = 2.0e-7, 300, 1.0e-9
    r0, v0 = (0.55, 0.0, 0.0), (V0, 0.0, 0.0)
    r, v, t = orc.rkn_advance(f, QM, r0, v0, t_a, dt, n, variant=solver)
    Bt = lambda tt: B0 + (B1 - B0) * tt / DS
    th = sum(-2.0 * math.atan(QM * Bt(t_a + k * dt) * dt / 2.0) for k in range(n))
    if solver == 3:
        th += -2.0 * math.atan(QM * Bt(t_a) * (-dt / 2.0) / 2.0)
    d = (math.atan2(v[1], v[0]) - th + math.pi) % (2 * math.pi) - math.pi
    assert abs(d) < 1e-11, d
    th_mid = sum(-2.0 * math.atan(QM * Bt(t_a + (k + 0.5) * dt) * dt / 2.0) for k in range(n))
    assert abs(th_mid - th) > 1e-3                              # the alternative reading is far outside the bound


def test_p20_trace_hit_matches_an_independent_ode_solution():
    """End to end (orc_trace: t0 per ion, t advanced every step, plane interpolation): the hit of an ion that
    makes more than half a gyration in the time-linear field equals the crossing point of a scipy DOP853 solution of
    the analytic equations of motion (rtol 1e-13).  Freezing t would move the hit by ~1e-4 m."""
    from scipy.integrate import solve_ivp
    f = _field()
    det = wl.Detector((0.50, 0.0, 0.0), (-1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0),
                      np.array([-1.0]), np.array([1.0]), np.array([-1.0]), np.array([1.0]))
    t0s = np.array([0.0, 1.0e-7, 3.0e-7])
    n = len(t0s)
    state = [np.full(n, 0.55), np.zeros(n), np.zeros(n), np.full(n, V0), np.zeros(n), np.full(n, 3.0e4)]
    dt = 2.5e-10
    res = orc.trace(f, QM, state, t0s, dt, 20000, det)
    assert np.all(res["status"] == 0)
    for i in range(n):
        def rhs(t, y):
            bz = B0 + (B1 - B0) * t / DS
            return [y[3], y[4], y[5], QM * y[4] * bz, -QM * y[3] * bz, 0.0]
        ev = lambda t, y: 0.50 - y[0]                           # s = -(X - 0.50): crossing from s < 0 to s >= 0
        ev.terminal, ev.direction = True, 1.0
        sol = solve_ivp(rhs, (t0s[i], t0s[i] + 2e-6), [0.55, 0.0, 0.0, V0, 0.0, 3.0e4], method="DOP853",
                        rtol=1e-13, atol=1e-16, events=ev)
        assert len(sol.t_events[0]) == 1
        ye = sol.y_events[0][0]
        th = sol.t_events[0][0] - t0s[i]
        assert 150e-9 < th < 400e-9
        assert res["steps"][i] == math.ceil(th / dt - 1e-9)
        # linear plane interpolation: chord error <= (v dt)^2 / (8 rho) ~ 2e-7 m here
        assert abs(res["u"][i] - ye[1]) < 5e-7 and abs(res["w"][i] - ye[2]) < 5e-7, (i, res["u"][i] - ye[1])


# ---- P21: invalid weights in the 32.32 fixed-point counters (reading L3') --------------------------------------
def test_p21_weight_domain_of_the_fixed_point_counters():
    """weight = w0 exp(-Lambda) with w0 a probability mass (<= 1) or a count: the counters accept [0, 2^20].
    Typed values: a negative or NaN weight counts as 0, anything above 2^20 as 2^20 (so that q < 2^53 stays exact in
    fp64 and 2^11 ions of maximum weight cannot overflow the 64-bit sum), 1 -> 2^32, 0.5 ulp rounds half up."""
    det = wl.uniform_detector(0.0, 0.0, 4, 1e-3)
    cell = np.array([0, 0, 0, 0, 0, 0], dtype=np.int32)
    w = np.array([-1.0, np.nan, 2.0 ** 21, 1.0, 2.0 ** -33, 2.0 ** -34])
    res = dict(cell=cell, weight=w)
    wc, ws = orc.histogram_weighted(res, np.zeros(6, np.uint16), det, 1)
    assert int(wc[0].reshape(-1)[0]) == 0 + 0 + (1 << 52) + (1 << 32) + 1 + 0
    assert int(ws[0, 3]) == 6 and int(ws[0, 1]) == 0
    for k, expect in enumerate((0, 0, 1 << 52, 1 << 32, 1, 0)):
        wc1, _ = orc.histogram_weighted(dict(cell=cell[k:k + 1], weight=w[k:k + 1]), np.zeros(1, np.uint16), det, 1)
        assert int(wc1.sum()) == expect, (k, w[k])
