"""Pins of the CPU oracle against what the paper and the mathematics fix (P1-P8).
CPU only (-m "not gpu").  Each pin cites the passage / closed form it checks."""
import math
import os

import numpy as np
import pytest

import oracle as orc
from paper_2506_15812_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
QM_LI = wl.E_CHARGE / wl.MASS_LI7
V0_60 = math.sqrt(2 * 60e3 * wl.E_CHARGE / wl.MASS_LI7)


def uniform_field(B, E=(0, 0, 0)):
    return orc.OracleField(kind=orc.KIND_UNIFORM, par=B, E=E)


# ---- P1 ---------------------------------------------------------------------------------
def test_p1_philox_known_answers():
    rows = [l.split() for l in open(os.path.join(GOLD, "philox4x32_10_kat.txt")) if l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert orc.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_p1_uniform_construction():
    # O2.1: U_k = ((w_2k>>6)*2^26 + (w_2k+1>>6) + 0.5) * 2^-52, counter=(i_lo,i_hi,j,0)
    seed, idx = 0x123456789ABCDEF0, (5 << 32) + 77
    w = []
    for j in range(3):
        w += orc.philox4x32_10([idx & 0xFFFFFFFF, idx >> 32, j, 0], [seed & 0xFFFFFFFF, seed >> 32])
    U = orc.uniforms(seed, idx)
    for k in range(5):
        n = ((w[2 * k] >> 6) << 26) + (w[2 * k + 1] >> 6)
        assert U[k] == (2 * n + 1) / 2.0 ** 53
        assert 0.0 < U[k] < 1.0


def test_constants_against_golden():
    vals = {"li7_q_over_m": QM_LI, "li7_v0_60keV": V0_60,
            "li7_omega_c_1p15T": QM_LI * 1.15, "li7_rL_1p15T_m": V0_60 / (QM_LI * 1.15),
            "li7_T_1p15T_s": 2 * math.pi / (QM_LI * 1.15), "li7_rL_1T_m": V0_60 / QM_LI,
            "li7_T_1T_s": 2 * math.pi / QM_LI,
            "na23_v0_40keV": math.sqrt(2 * 40e3 * wl.E_CHARGE / wl.MASS_NA23)}
    for l in open(os.path.join(GOLD, "physical_constants.txt")):
        if l[0] == "#":
            continue
        k, v, tol = l.split()
        assert abs(vals[k] / float(v) - 1) < float(tol), k


# ---- P2: RKN velocity update in uniform B is exactly RK4 on v' = Omega v x b ------------------
@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("dt", [1e-9, 5e-9, 2e-8])
def test_p2_rk4_amplification_factor(variant, dt):
    f = uniform_field((0, 0, 1.15))
    z = QM_LI * 1.15 * dt
    v0 = np.array([3e5, -4e5, 1.7e5])
    r, v, _ = orc.rkn_advance(f, QM_LI, [0.7, 0, 0], v0, 0.0, dt, 1, variant)
    amp2 = (v[0] ** 2 + v[1] ** 2) / (v0[0] ** 2 + v0[1] ** 2)
    assert abs(amp2 - (1 - z ** 6 / 72 + z ** 8 / 576)) < 8e-16
    # rotation angle: clockwise for q>0, B along +z; atan2(z - z^3/6, 1 - z^2/2 + z^4/24)
    ang = math.atan2(v0[0] * v[1] - v0[1] * v[0], v0[0] * v[0] + v0[1] * v[1])
    assert abs(-ang - math.atan2(z - z ** 3 / 6, 1 - z ** 2 / 2 + z ** 4 / 24)) < 1e-15
    assert v[2] == v0[2]                       # v_parallel untouched, exactly


def test_p2_energy_loss_300_steps():
    # SURVEY P2 probe: dKE/KE after 300 steps = -300 z^6/72 (= -6.522e-11 at z=0.01582)
    f = uniform_field((0, 0, 1.15))
    z = QM_LI * 1.15 * 1e-9
    r, v, _ = orc.rkn_advance(f, QM_LI, [0.7, 0, 0], [-V0_60, 0, 0], 0.0, 1e-9, 300)
    dke = (v @ v) / V0_60 ** 2 - 1
    assert abs(dke / (-300 * z ** 6 / 72) - 1) < 2e-3
    assert abs(dke + 6.522e-11) < 2e-14


# ---- P3: Larmor radius and gyro-period (paper scenario 1) ----------------------
def test_p3_larmor_radius_and_period():
    B = 1.0
    f = uniform_field((0, 0, B))
    dt = 1e-9
    om = QM_LI * B
    rL, T = V0_60 / om, 2 * math.pi / om
    r0 = np.array([0.0, 0.0, 0.0])
    v0 = np.array([V0_60, 0.0, 0.0])
    centre = np.array([0.0, -rL, 0.0])          # q>0, B=+z: clockwise, centre at r0 + v x b / om
    pts = []
    r, v, t = r0, v0, 0.0
    nst = int(round(T / dt)) + 2
    for _ in range(nst):
        r, v, t = orc.rkn_advance(f, QM_LI, r, v, t, dt, 1)
        pts.append((t, r.copy(), v.copy()))
    rad = np.array([np.linalg.norm(p[1] - centre) for p in pts])
    assert abs(rL - 0.093409) < 1e-6
    assert np.max(np.abs(rad / rL - 1)) < 1e-8
    # period: time at which the velocity direction returns to +x (interpolate the phase)
    ph = np.unwrap([math.atan2(-p[2][1], p[2][0]) for p in pts])
    ts = np.array([p[0] for p in pts])
    Tnum = np.interp(2 * math.pi, ph, ts)
    assert abs(T - 456.85e-9) < 1e-11
    z = om * dt
    assert abs(Tnum / T - (1 + z ** 4 / 120)) < 1e-9
    assert abs(Tnum / T - 1) < 1e-7


# ---- P4: uniform E, B=0: exact parabola (paper scenario 2, L279) ------------------------------
def test_p4_uniform_E_parabola_exact():
    f = uniform_field((0, 0, 0), E=(0.0, 0.0, 1.0))
    dt, n = 1e-9, 1000
    r0, v0 = np.array([0.1, 0.2, 0.3]), np.array([1e3, -2e3, 5e2])
    r, v, t = orc.rkn_advance(f, QM_LI, r0, v0, 0.0, dt, n)
    T = n * dt
    a = np.array([0, 0, QM_LI * 1.0])
    assert np.allclose(r, r0 + v0 * T + 0.5 * a * T * T, rtol=0, atol=2e-14)
    assert np.allclose(v, v0 + a * T, rtol=2e-13, atol=0)
    # one step is exact to rounding
    r1, v1, _ = orc.rkn_advance(f, QM_LI, r0, v0, 0.0, dt, 1)
    assert abs(r1[2] - (r0[2] + v0[2] * dt + 0.5 * a[2] * dt * dt)) < 1e-16


def test_p4b_E_cross_B_drift():
    # paper scenario 5 (L282): B=(0,0,1), E=(0,0,0.1): helix + uniform acceleration along z
    f = uniform_field((0, 0, 1.0), E=(0.0, 0.0, 0.1))
    dt, n = 1e-9, 500
    v0 = np.array([1e5, 0.0, 2e4])
    r, v, t = orc.rkn_advance(f, QM_LI, [0, 0, 0], v0, 0.0, dt, n)
    T = n * dt
    assert abs(v[2] - (v0[2] + QM_LI * 0.1 * T)) < 1e-9 * abs(v[2])
    assert abs(r[2] - (v0[2] * T + 0.5 * QM_LI * 0.1 * T * T)) < 1e-12
    assert abs(math.hypot(v[0], v[1]) / 1e5 - 1) < 1e-9


# ---- P5: kinetic energy bound in the spline field ----------------------------------------------
def test_p5_kinetic_energy_bound_cfg1_field():
    grid, nodal = wl.nodal_field_2d(65, 129)
    f = orc.OracleField(grid, nodal)
    dt, n = 1e-9, 5000
    st = orc.seed(wl.Beam(wl.MASS_LI7, wl.E_CHARGE, 60e3), wl.depth_cdf(), wl.normal_cdf(), 0, 0, 8)
    worst = 0.0
    for i in range(8):
        r = np.array([st[0][i], st[1][i], st[2][i]])
        v = np.array([st[3][i], st[4][i], st[5][i]])
        ke0 = v @ v
        bmax = 0.0
        t = 0.0
        for _ in range(10):
            r, v, t = orc.rkn_advance(f, QM_LI, r, v, t, dt, n // 10)
            bmax = max(bmax, np.linalg.norm(f.B(r)))
        worst = max(worst, abs((v @ v) / ke0 - 1))
    zmax = QM_LI * 1.15 * 0.56 / 0.25 * dt          # |B| <= B_T R0/Rmin (+ small B_pol)
    assert worst <= n * (1.05 * zmax) ** 6 / 72 + n * 4 * 2.2e-16
    assert worst < 5e-9
