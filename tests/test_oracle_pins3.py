"""Pins P10-P12 of the CPU oracle: CDF inversion / seeding, plane interpolation / binning,
independent naive evaluator end to end.  CPU only."""
import math

import numpy as np
from scipy import interpolate, stats

import oracle as orc
from paper_2506_15812_b200 import workloads as wl

QM_LI = wl.E_CHARGE / wl.MASS_LI7
V0_60 = math.sqrt(2 * 60e3 * wl.E_CHARGE / wl.MASS_LI7)


# ---- P10 -----------------------------------------------------------------------------------
def test_p10_cdf_inversion_exact_and_monotone():
    F = wl.depth_cdf()
    K = len(F) - 1
    dx = wl.DEPTH_MAX / K
    for j in (0, 1, 17, K // 2, K - 1):
        assert orc.cdf_invert(F, wl.DEPTH_MAX, F[j]) == j * dx          # node -> node
    mid = 0.5 * (F[10] + F[11])
    assert abs(orc.cdf_invert(F, wl.DEPTH_MAX, mid) - 10.5 * dx) < 1e-15
    Us = np.sort(np.random.default_rng(0).uniform(0, 1, 2000))
    xs = np.array([orc.cdf_invert(F, wl.DEPTH_MAX, u) for u in Us])
    assert np.all(np.diff(xs) >= 0) and xs[0] >= 0 and xs[-1] < wl.DEPTH_MAX
    # against numpy's interpolation of the inverse table
    assert np.allclose(xs, np.interp(Us, F, np.arange(K + 1) * dx), atol=1e-15)
    # flat bins are skipped: a table with a repeated value never divides by zero
    Ff = np.array([0.0, 0.25, 0.25, 0.25, 1.0])
    assert orc.cdf_invert(Ff, 4.0, 0.25) == 3.0
    assert orc.cdf_invert(Ff, 4.0, 0.2499999) < 1.0


def test_p10_seeding_statistics_and_structure():
    n = 200000
    beam = wl.Beam(wl.MASS_LI7, wl.E_CHARGE, 60e3, sigma_ang_rad=2e-3)
    x, y, z, vx, vy, vz = orc.seed(beam, wl.depth_cdf(), wl.normal_cdf(), 1, 0, n)
    d = 0.78 - x
    lam, dm = wl.DEPTH_LAMBDA, wl.DEPTH_MAX
    mean_exact = lam - dm * math.exp(-dm / lam) / (1 - math.exp(-dm / lam))   # truncated exp.
    assert abs(d.mean() - mean_exact) < 5 * lam / math.sqrt(n)
    assert d.min() >= 0 and d.max() < dm
    for arr, sig in ((y, 5e-3), (z, 5e-3)):
        ks = stats.kstest(arr / sig, "norm")
        assert ks.statistic < 1.36 / math.sqrt(n) * 1.5 + 12 / 4096 * 0.4
    speed = np.sqrt(vx ** 2 + vy ** 2 + vz ** 2)
    assert np.max(np.abs(speed / V0_60 - 1)) < 1e-15
    assert abs(np.std(vy / V0_60) / 2e-3 - 1) < 0.01 and abs(np.std(vz / V0_60) / 2e-3 - 1) < 0.01
    assert abs(np.corrcoef(y, z)[0, 1]) < 0.01 and abs(np.corrcoef(d, vy)[0, 1]) < 0.01
    # counter-based: ion i does not depend on the batch it is generated in
    x2 = orc.seed(beam, wl.depth_cdf(), wl.normal_cdf(), 1, 1000, 10)[0]
    assert np.array_equal(x2, x[1000:1010])
    # sigma_ang = 0: v = v0 * axis exactly
    b0 = wl.Beam(wl.MASS_LI7, wl.E_CHARGE, 60e3)
    s0 = orc.seed(b0, wl.depth_cdf(), wl.normal_cdf(), 1, 0, 5)
    assert np.all(s0[3] == -orc.beam_v0(b0)) and np.all(s0[4] == 0) and np.all(s0[5] == 0)
    # seeding formula written out for one ion (O2.3-4) with the oracle's own uniforms
    U = orc.uniforms(1, 123)
    dd = orc.cdf_invert(wl.depth_cdf(), dm, U[0])
    z1 = orc.cdf_invert(wl.normal_cdf(), 12.0, U[1]) - 6.0
    z2 = orc.cdf_invert(wl.normal_cdf(), 12.0, U[2]) - 6.0
    assert abs(x[123] - (0.78 - dd)) < 1e-16 and abs(y[123] - 5e-3 * z1) < 1e-17
    assert abs(z[123] - 5e-3 * z2) < 1e-17


# ---- P11 -----------------------------------------------------------------------------------
def test_p11_straight_line_hit_independent_of_dt():
    f = orc.OracleField(kind=orc.KIND_UNIFORM, par=(0.0, 0.0, 0.0))
    th = 0.3
    nrm = (math.cos(th), math.sin(th), 0.0)
    eu = (-math.sin(th), math.cos(th), 0.0)
    det = wl.Detector((0.82, 0.01, 0.02), nrm, eu, (0, 0, 1.0), *(np.array([-1.0]), np.array([1.0])) * 2)
    r0 = np.array([0.7, 0.0, 0.0])
    v0 = np.array([9e5, 2e5, -1e5])
    st = [np.array([c]) for c in (*r0, *v0)]
    # exact: s(t) = n.(r0 + v t - rD) = 0
    o = np.array(det.origin)
    th_exact = -np.dot(nrm, r0 - o) / np.dot(nrm, v0)
    p = r0 + v0 * th_exact
    res = {}
    for dt in (1e-9, 3.7e-9, 2.5e-10):
        r = orc.trace(f, QM_LI, st, None, dt, 100000, det, want_xyz=True)
        assert r["status"][0] == 0 and r["steps"][0] == math.ceil(th_exact / dt)
        assert np.allclose(r["xyz"][0], p, atol=1e-14)
        assert abs(r["u"][0] - np.dot(p - o, eu)) < 1e-14 and abs(r["w"][0] - (p[2] - o[2])) < 1e-14
        res[dt] = r


def test_p11_status_codes():
    grid, nodal = wl.nodal_field_2d(17, 33)
    f = orc.OracleField(grid, nodal)
    det = wl.uniform_detector(0.02, 0.18, 4, 5e-3)
    st = [np.array(c) for c in ([0.83, 0.7, 0.7, 0.2], [0, 0, 0, 0], [0, 0, 0.62, 0],
                                 [-1e6, -V0_60, 0, 1e5], [0, 0, 0, 0], [0, 0, 1e6, 0])]
    r = orc.trace(f, QM_LI, st, None, 1e-9, 50, det)
    assert r["status"][0] == -4 and r["steps"][0] == 0          # starts beyond the plane
    assert r["status"][1] == -2 and r["steps"][1] == 50         # max_steps
    assert r["status"][2] == -3 and r["steps"][2] == 6          # Z = 0.62 + k mm > 0.625 first at k=6
    assert r["status"][3] == -4                                 # starts outside the grid


def test_p11_binning_brute_force_and_invariant():
    rng = np.random.default_rng(5)
    n = 5000
    # non-uniform segments with gaps
    u_lo = np.array([-4e-3, -2.5e-3, -1e-3, 1.2e-3])
    u_hi = np.array([-2.7e-3, -1e-3, 1e-3, 3e-3])
    w_lo = np.array([-3e-3, 0.0, 2e-3])
    w_hi = np.array([-0.5e-3, 2e-3, 4e-3])
    det = wl.Detector((0.82, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), u_lo, u_hi, w_lo, w_hi)
    status = rng.choice([0, 0, 0, -2, -3, -4], n).astype(np.int32)
    u = rng.uniform(-5e-3, 4e-3, n)
    w = rng.uniform(-4e-3, 5e-3, n)
    u[:6] = [-4e-3, -2.7e-3, -1e-3, 1e-3, 3e-3, 1.2e-3 - 5e-10]      # edge cases, half-open
    w[:6] = 1e-3
    status[:6] = 0
    grp = rng.integers(0, 3, n).astype(np.uint16)
    res = dict(status=status, u=u, w=w, flags=np.zeros(n, np.uint8))
    counts, summary = orc.histogram(res, grp, det, 3)
    # independent numpy definition
    exp = np.zeros((3, 3, 4), np.uint64)
    for i in range(n):
        if status[i] != 0:
            continue
        iu = [k for k in range(4) if u_lo[k] <= u[i] < u_hi[k]]
        iw = [k for k in range(3) if w_lo[k] <= w[i] < w_hi[k]]
        if iu and iw:
            exp[grp[i], iw[0], iu[0]] += 1
            assert res["cell"][i] == iw[0] * 4 + iu[0]
        else:
            assert res["cell"][i] == -1
    assert np.array_equal(counts, exp)
    assert [int(c) for c in res["cell"][:6]] == [4, -1, 6, -1, -1, -1]
    assert np.all(res["flags"][:6] == 1)
    for g in range(3):
        assert counts[g].sum() + summary[g, 1:5].sum() == np.sum(grp == g)   # O5 invariant
        assert summary[g, 0] == counts[g].sum()


# ---- P12: independent naive evaluator ------------------------------------------------------
def test_p12_naive_evaluator_end_to_end():
    """64 ions, 9x17 grid, 4x4 detector: RKN written again in numpy with the field evaluated by
    scipy's not-a-knot splines directly along each axis (no per-cell coefficient tables)."""
    grid, nodal = wl.nodal_field_2d(9, 17)
    f = orc.OracleField(grid, nodal)
    R, Z = grid.axes()
    sp = [interpolate.RectBivariateSpline(R, Z, nodal[c][0], kx=3, ky=3, s=0) for c in range(3)]
    det = wl.uniform_detector(0.02, 0.18, 4, 10e-3)
    beam = wl.Beam(wl.MASS_LI7, wl.E_CHARGE, 60e3)
    st = orc.seed(beam, wl.depth_cdf(), wl.normal_cdf(), 9, 0, 64)
    dt, nmax = 1e-9, 600
    res = orc.trace(f, QM_LI, st, None, dt, nmax, det)

    def acc(r, v):
        Rr = np.hypot(r[:, 0], r[:, 1])
        c, s = r[:, 0] / Rr, r[:, 1] / Rr
        bR, bZ, bP = (sp[k].ev(Rr, r[:, 2]) for k in range(3))
        B = np.stack([bR * c - bP * s, bR * s + bP * c, bZ], axis=1)
        return QM_LI * np.cross(v, B)

    r = np.stack(st[0:3], axis=1)
    v = np.stack(st[3:6], axis=1)
    o, nrm = np.array(det.origin), np.array(det.normal)
    hit = np.full((64, 2), np.nan)
    steps = np.zeros(64, int)
    alive = np.ones(64, bool)
    s0 = (r - o) @ nrm
    for step in range(1, nmax + 1):
        k1 = acc(r, v)
        k2 = acc(r + v * dt / 2 + k1 * dt * dt / 8, v + k1 * dt / 2)
        k3 = acc(r + v * dt / 2 + k1 * dt * dt / 8, v + k2 * dt / 2)
        k4 = acc(r + v * dt + k3 * dt * dt / 2, v + k3 * dt)
        rn = r + v * dt + (k1 + k2 + k3) * dt * dt / 6
        vn = v + (k1 + 2 * k2 + 2 * k3 + k4) * dt / 6
        s1 = (rn - o) @ nrm
        cross = alive & (s0 < 0) & (s1 >= 0)
        lam = s0 / (s0 - s1)
        p = r + lam[:, None] * (rn - r)
        hit[cross, 0] = (p[cross] - o) @ np.array(det.eu)
        hit[cross, 1] = (p[cross] - o) @ np.array(det.ew)
        steps[cross] = step
        alive &= ~cross
        r, v, s0 = rn, vn, s1
    crossed = res["status"] == 0
    assert crossed.sum() > 40
    assert np.array_equal(crossed, ~np.isnan(hit[:, 0]))
    assert np.array_equal(res["steps"][crossed], steps[crossed])
    assert np.max(np.abs(res["u"][crossed] - hit[crossed, 0])) < 1e-12
    assert np.max(np.abs(res["w"][crossed] - hit[crossed, 1])) < 1e-12
