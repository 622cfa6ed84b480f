"""Property tests (hypothesis) of the oracle on small random inputs: SURVEY.md section 4 layer (iii).
CPU only; each property is fixed by the mathematics, not by the implementation."""
import math

import numpy as np
from hypothesis import given, settings, strategies as st

import oracle as orc
from paper_2506_15812_b200 import workloads as wl

QM = wl.E_CHARGE / wl.MASS_LI7
SET = dict(max_examples=40, deadline=None)


@settings(**SET)
@given(st.integers(2, 60), st.integers(0, 2 ** 32 - 1), st.floats(0.05, 5.0))
def test_cdf_inversion_is_the_inverse_of_the_piecewise_linear_cdf(K, seed, xmax):
    rng = np.random.default_rng(seed)
    inc = rng.uniform(0.0, 1.0, K) * (rng.uniform(0, 1, K) > 0.2)          # some flat bins
    if inc.sum() == 0:
        inc[0] = 1.0
    F = np.concatenate([[0.0], np.cumsum(inc)])
    F /= F[-1]
    F[-1] = 1.0
    U = np.sort(rng.uniform(1e-12, 1 - 1e-12, 50))
    x = np.array([orc.cdf_invert(F, xmax, u) for u in U])
    assert np.all(np.diff(x) >= -1e-15 * xmax)                              # monotone
    assert np.all((x >= 0) & (x <= xmax))
    back = np.interp(x, np.linspace(0, xmax, K + 1), F)                     # F(F^-1(U)) = U
    assert np.abs(back - U).max() < 1e-12


@settings(**SET)
@given(st.integers(4, 12), st.integers(4, 12), st.integers(0, 2 ** 32 - 1))
def test_bicubic_spline_reproduces_any_bicubic_polynomial(nR, nZ, seed):
    """Not-a-knot cubic splines have cubic precision; so has their tensor product."""
    rng = np.random.default_rng(seed)
    c = rng.standard_normal((4, 4))
    grid = wl.Grid(0, nR, nZ, 1, 0.3, 0.9, -0.5, 0.4)
    R = np.linspace(grid.Rmin, grid.Rmax, nR)[:, None]
    Z = np.linspace(grid.Zmin, grid.Zmax, nZ)[None, :]
    poly = lambda r, z: sum(c[a, b] * r ** a * z ** b for a in range(4) for b in range(4))
    nod = np.ascontiguousarray(poly(R, Z + 0 * R)).reshape(1, nR, nZ)
    f = orc.OracleField(grid, [nod, nod, nod])
    for r, z in rng.uniform([0.3, -0.5], [0.9, 0.4], (20, 2)):
        assert abs(f.cyl(r, z)[0] - poly(r, z)) < 1e-11 * (1 + np.abs(c).sum())


@settings(**SET)
@given(st.floats(-1, 1), st.floats(-1, 1), st.floats(-1, 1), st.floats(0.2, 3.0), st.floats(1e-10, 5e-9))
def test_rkn_speed_changes_by_the_rk4_factor_in_any_uniform_field(bx, by, bz, Bmag, dt):
    n = math.sqrt(bx * bx + by * by + bz * bz)
    if n < 1e-3:
        return
    B = np.array([bx, by, bz]) / n * Bmag
    f = orc.OracleField(kind=orc.KIND_UNIFORM, par=tuple(B))
    v0 = np.array([3e5, -4e5, 1.7e5])
    _, v, _ = orc.rkn_advance(f, QM, [0.7, 0.0, 0.0], v0, 0.0, dt, 1, 0)
    b = B / Bmag
    vpar0, vpar = v0 @ b, v @ b
    z = QM * Bmag * dt
    perp0, perp = v0 @ v0 - vpar0 ** 2, v @ v - vpar ** 2
    assert abs(vpar - vpar0) < 1e-9 * np.linalg.norm(v0)
    assert abs(perp / perp0 - (1 - z ** 6 / 72 + z ** 8 / 576)) < 1e-13


@settings(**SET)
@given(st.integers(1, 9), st.integers(1, 9), st.integers(0, 2 ** 32 - 1))
def test_histogram_counts_every_crosser_once_and_only_inside_its_segment(nu, nw, seed):
    rng = np.random.default_rng(seed)
    eu = np.sort(rng.uniform(-1e-2, 1e-2, 2 * nu))
    ew = np.sort(rng.uniform(-1e-2, 1e-2, 2 * nw))
    if np.any(np.diff(eu) <= 0) or np.any(np.diff(ew) <= 0):
        return
    det = wl.Detector((0.82, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), eu[0::2].copy(), eu[1::2].copy(), ew[0::2].copy(), ew[1::2].copy())
    n = 400
    status = rng.choice([0, 0, 0, -2, -3, -4], n).astype(np.int32)
    res = dict(status=status, u=rng.uniform(-1.2e-2, 1.2e-2, n), w=rng.uniform(-1.2e-2, 1.2e-2, n), flags=np.zeros(n, np.uint8))
    counts, summary = orc.histogram(res, None, det, 1)
    assert counts.sum() == summary[0, 0] and summary[0, :5].sum() == n
    assert summary[0, 0] + summary[0, 1] == (status == 0).sum()
    hit = res["cell"] >= 0
    iu, iw = res["cell"][hit] % nu, res["cell"][hit] // nu
    assert np.all((res["u"][hit] >= det.u_lo[iu]) & (res["u"][hit] < det.u_hi[iu]))
    assert np.all((res["w"][hit] >= det.w_lo[iw]) & (res["w"][hit] < det.w_hi[iw]))
    miss = (status == 0) & ~hit
    for i in np.flatnonzero(miss)[:50]:
        inside_u = np.any((res["u"][i] >= det.u_lo) & (res["u"][i] < det.u_hi))
        inside_w = np.any((res["w"][i] >= det.w_lo) & (res["w"][i] < det.w_hi))
        assert not (inside_u and inside_w)
