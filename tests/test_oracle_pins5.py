"""Pins of the oracle's secondary-ionisation loss: PAPER.md Eq. 2
(L142, McWhirter's rate), L177 ("numerically integrated with every step using the one-dimensional
secondary ionization profile"), L350 (counters weighted by the loss).  CPU only."""
import math

import numpy as np
import pytest

import oracle as orc
from paper_2506_15812_b200 import workloads as wl

QM = wl.E_CHARGE / wl.MASS_LI7
V0 = math.sqrt(2 * 60e3 * wl.E_CHARGE / wl.MASS_LI7)


# ---- P16: Eq. 2 ---------------------------------------------------------------------------
def test_p16_mcwhirter_values_typed_from_the_formula():
    """nu = n_e sqrt(t) exp(-1/t) / (E12^1.5 (6+t)) 1e-11, t = T_e/E12; numbers worked by hand:
    t=1, E12=100: 1e19 * e^-1 / (1000 * 7) * 1e-11;  t=4, E12=25: 2e19 * 2 e^-1/4 / (125 * 10) * 1e-11."""
    assert abs(orc.mcwhirter_rate(1e19, 100.0, 100.0) / 5255.420588163462 - 1) < 1e-14
    assert abs(orc.mcwhirter_rate(2e19, 100.0, 25.0) / 249216.25058284955 - 1) < 1e-14
    assert orc.mcwhirter_rate(1e19, 0.0, 75.64) == 0.0
    # linear in n_e; strongly suppressed for T_e << E12 (exp(-1/t)); paper validity 0.02 <= t <= 100
    assert abs(orc.mcwhirter_rate(3e19, 50.0, 75.64) / orc.mcwhirter_rate(1e19, 50.0, 75.64) - 3) < 1e-14
    assert orc.mcwhirter_rate(1e19, 0.02 * 75.64, 75.64) < 1e-15 * orc.mcwhirter_rate(1e19, 75.64, 75.64)
    # Na+ (47.3 eV) is ionised more readily than Li+ (75.6 eV): Table 1's ordering (L147-158)
    assert orc.mcwhirter_rate(1e19, 300.0, wl.E12_NA) > 1.5 * orc.mcwhirter_rate(1e19, 300.0, wl.E12_LI)


# ---- P17: loss integral ---------------------------------------------------------------------
def zero_field(nR=33, nZ=65):
    grid, nodal = wl.nodal_field_2d(nR, nZ)
    return grid, orc.OracleField(grid, [0.0 * c for c in nodal])


def det_plane(x=0.82):
    return wl.uniform_detector(0.0, 0.0, 8, 2.5e-3, x_plane=x)


def test_p17_constant_rate_straight_line_exact():
    """B = 0: the ion flies straight, t_hit = distance / v.  A constant rate makes every
    trapezoid exact, including the fractional last step, so weight = exp(-nu t_hit)."""
    grid, f = zero_field()
    nu0 = 2.5e6
    L = orc.OracleLoss(grid, wl.nodal_psi(grid), 0.0, 1e-3, np.full(5, nu0))
    x0 = np.array([0.70, 0.61, 0.8123])
    state = [x0, np.zeros(3), np.array([0.0, 0.01, -0.02]), np.full(3, V0), np.zeros(3), np.zeros(3)]
    for dt in (1e-9, 3.7e-10):
        res = orc.trace_loss(f, L, QM, state, None, dt, 100000, det_plane())
        assert np.all(res["status"] == 0)
        t_hit = (0.82 - x0) / V0
        assert np.abs(res["weight"] / np.exp(-nu0 * t_hit) - 1).max() < 1e-13
        assert np.all(res["steps"] == np.ceil(t_hit / dt - 1e-9))


def test_p17_profile_quadrature_order_two():
    """nu linear in psi along a straight chord through the Solov'ev flux: the trapezoid sum
    converges at order 2 to the independent quadrature of nu(psi(x(t))) (scipy quad on the
    ANALYTIC psi; the spline's own error is ~1e-9 relative)."""
    from scipy.integrate import quad
    grid, f = zero_field(65, 129)
    psi0, dpsi, n = 0.0, wl.PSI_A * 3.0 / 64, 65            # covers the chord: psi <= 2.6 PSI_A
    rate = 1e5 + 4e6 * np.arange(n) / (n - 1)                    # linear in psi: exact under linear interpolation
    L = orc.OracleLoss(grid, wl.nodal_psi(grid), psi0, dpsi, rate)
    z0, y0, x0 = 0.03, 0.0, 0.45
    state = [np.array([x0]), np.array([y0]), np.array([z0]), np.array([V0]), np.array([0.0]), np.array([0.0])]

    def nu_of_t(t):
        psi = float(wl.solovev_psi(x0 + V0 * t, z0))
        return 1e5 + 4e6 * (psi - psi0) / (dpsi * (n - 1))
    T = (0.82 - x0) / V0
    exact = math.exp(-quad(nu_of_t, 0.0, T, epsabs=1e-14, epsrel=1e-13)[0])
    err, val = [], []
    for dt in (4e-9, 2e-9, 1e-9):
        res = orc.trace_loss(f, L, QM, state, None, dt, 100000, det_plane())
        val.append(res["weight"][0])
        err.append(abs(val[-1] - exact))
    assert 1.9 < math.log2(err[0] / err[1]) < 2.1 and 1.9 < math.log2(err[1] / err[2]) < 2.1
    assert err[2] < 1e-5 and 0.3 < exact < 0.9
    assert abs((4.0 * val[2] - val[1]) / 3.0 - exact) < 2e-8        # Richardson: the dt^2 term cancels


def test_p17_rate_scaling_and_bounds_in_the_tokamak_field():
    """Config-1 field and ions: doubling a constant rate squares the weight; the weight lies
    between exp(-nu steps dt) and exp(-nu (steps-1) dt); trapped ions integrate all max_steps;
    bad starts keep weight 1."""
    cfg = wl.config(1, n_override=256)
    grid, nodal = cfg.field_builder()
    f = orc.OracleField(grid, nodal)
    g = cfg.groups[0]
    st = orc.seed(g.beam, wl.depth_cdf(), wl.normal_cdf(), cfg.seed, 0, 256)
    nu0 = 1.0e5
    out = []
    for k in (1.0, 2.0):
        L = orc.OracleLoss(grid, wl.nodal_psi(grid), 0.0, 1e-3, np.full(3, k * nu0))
        out.append(orc.trace_loss(f, L, QM, st, None, cfg.dt, cfg.max_steps, cfg.detector))
    a, b = out
    assert np.array_equal(a["steps"], b["steps"]) and np.array_equal(a["u"], b["u"])
    assert np.abs(b["weight"] / a["weight"] ** 2 - 1).max() < 1e-13
    cr = a["status"] == 0
    n = a["steps"].astype(np.float64)
    assert np.all(a["weight"][cr] <= np.exp(-nu0 * (n[cr] - 1) * cfg.dt) * (1 + 1e-14))
    assert np.all(a["weight"][cr] >= np.exp(-nu0 * n[cr] * cfg.dt) * (1 - 1e-14))
    tr = a["status"] == -2
    assert tr.any() and np.abs(a["weight"][tr] / math.exp(-nu0 * cfg.max_steps * cfg.dt) - 1).max() < 1e-12
    # same trajectories as the plain tracer
    ref = orc.trace(f, QM, st, None, cfg.dt, cfg.max_steps, cfg.detector)
    assert np.array_equal(ref["steps"], a["steps"]) and np.array_equal(ref["w"], a["w"])
    bad = orc.trace_loss(f, L, QM, [np.array([0.83]), np.zeros(1), np.zeros(1), np.array([-V0]), np.zeros(1), np.zeros(1)],
                         None, cfg.dt, 10, cfg.detector)
    assert bad["status"][0] == -4 and bad["weight"][0] == 1.0


def test_p17_synthetic_profile_loss_is_percent_level_and_deeper_is_larger():
    """The synthetic H-mode-like profiles give a Li+ loss of the order of Table 1 (percent level;
    L147-158 quotes 4.3-5.0 % on COMPASS profiles) that grows with the ionisation depth (L160:
    'the secondary ionization rate depends on the primary ionization's radial position')."""
    cfg = wl.config(1, n_override=1024)
    grid, nodal = cfg.field_builder()
    f = orc.OracleField(grid, nodal)
    psi0, dpsi, ne, te = wl.loss_profile_inputs()
    L = orc.OracleLoss(grid, wl.nodal_psi(grid), psi0, dpsi, orc.mcwhirter_rate(ne, te, wl.E12_LI))
    g = cfg.groups[0]
    st = orc.seed(g.beam, wl.depth_cdf(), wl.normal_cdf(), cfg.seed, 0, 1024)
    res = orc.trace_loss(f, L, QM, st, None, cfg.dt, cfg.max_steps, cfg.detector)
    cr = res["status"] == 0
    loss = 1.0 - res["weight"][cr]
    assert 0.003 < loss.mean() < 0.05
    depth = 0.78 - st[0][cr]
    assert np.corrcoef(depth, loss)[0, 1] > 0.8


def test_p17_fixed_point_counters():
    """32.32 fixed point: sums are exact integers, independent of the accumulation order."""
    rng = np.random.default_rng(5)
    n, n_hist = 5000, 3
    det = wl.uniform_detector(0.0, 0.0, 4, 1e-3)
    cell = rng.integers(-4, 16, n).astype(np.int32)
    w = rng.uniform(0.0, 1.0, n)
    w[:3] = (1.0, 0.0, 0.5)
    grp = rng.integers(0, n_hist + 1, n).astype(np.uint16)
    res = dict(cell=cell, weight=w)
    wc, ws = orc.histogram_weighted(res, grp, det, n_hist)
    q = [int(math.floor(float(x) * 4294967296.0 + 0.5)) for x in w]
    for h in range(n_hist):
        sel = [i for i in range(n) if grp[i] == h and cell[i] >= -1]
        assert int(ws[h, 0]) == sum(q[i] for i in sel if cell[i] >= 0)
        assert int(ws[h, 1]) == sum(q[i] for i in sel if cell[i] == -1)
        assert int(ws[h, 2]) == sum((q[i] * q[i]) >> 32 for i in sel)
        assert int(ws[h, 3]) == len(sel)
        for c in range(16):
            assert int(wc[h].reshape(-1)[c]) == sum(q[i] for i in sel if cell[i] == c)
    perm = rng.permutation(n)
    wc2, ws2 = orc.histogram_weighted(dict(cell=cell[perm], weight=w[perm]), grp[perm], det, n_hist)
    assert np.array_equal(wc, wc2) and np.array_equal(ws, ws2)
