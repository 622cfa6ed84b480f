"""P22: uniform-disc beam cross-section (PAPER.md: "a 60 keV lithium atomic beam with a 5 mm diameter";
reading A7' in DESIGN.md).  The oracle draws the cross-section offset uniformly over the disc by rejection from the
enclosing square with counter-based retries.  Pinned against what the mathematics fixes for a uniform disc --
radius bound, P(r <= x) = (x/R)^2, uniform azimuth, second moments R^2/4, acceptance pi/4 -- and, for the counter
layout of the retries, against the Philox words themselves (known-answer pinned, P1).  CPU only."""
import dataclasses
import math

import numpy as np
from scipy import stats

import oracle as orc
from paper_2506_15812_b200 import workloads as wl

RAD = 2.5e-3
SEED = 0xC0FFEE


def _beam(**kw):
    return dataclasses.replace(wl.config(1).groups[0].beam, profile=1, radius_m=RAD, **kw)


def _u52(w0, w1):
    return (float(((w0 >> 6) << 26) + (w1 >> 6)) + 0.5) * 2.0 ** -52


def test_p22_disc_is_uniform():
    n = 200000
    st = orc.seed(_beam(), wl.depth_cdf(), wl.normal_cdf(), SEED, 0, n)
    y, z = st[1], st[2]                                   # beam frame of the configs: eT = Y, eZ = Z, axis = -X
    r = np.hypot(y, z)
    assert r.max() <= RAD and r.max() > 0.999 * RAD
    assert stats.kstest((r / RAD) ** 2, "uniform").pvalue > 1e-3           # P(r <= x) = (x/R)^2
    assert stats.kstest((np.arctan2(z, y) + math.pi) / (2 * math.pi), "uniform").pvalue > 1e-3
    # moments of the uniform disc: E y = E z = 0, Var y = Var z = R^2/4, Cov = 0 (standard errors ~ R^2 / sqrt(n))
    assert abs(y.mean()) < 5 * RAD / 2 / math.sqrt(n) and abs(z.mean()) < 5 * RAD / 2 / math.sqrt(n)
    assert abs(y.var() / (RAD ** 2 / 4) - 1) < 0.01 and abs(z.var() / (RAD ** 2 / 4) - 1) < 0.01
    assert abs(np.mean(y * z)) / (RAD ** 2 / 4) < 0.01
    # depth and velocity are what the Gaussian profile draws (same U_0; no divergence here)
    g = orc.seed(dataclasses.replace(_beam(), profile=0), wl.depth_cdf(), wl.normal_cdf(), SEED, 0, 1000)
    assert np.array_equal(g[0], st[0][:1000]) and np.array_equal(g[3], st[3][:1000])


def test_p22_first_try_and_retry_counters():
    """Try 0 is (2 U_1 - 1, 2 U_2 - 1) of the ion's standard uniforms; the k-th retry reads Philox counter
    (i_lo, i_hi, 2 + k, 0).  Recomputed here from the Philox words (P1) for every ion of a batch at indices
    beyond 2^32; the acceptance rate of try 0 is pi/4."""
    n, first = 4000, (1 << 33) + 12345
    st = orc.seed(_beam(), wl.depth_cdf(), wl.normal_cdf(), SEED, first, n)
    key = (SEED & 0xFFFFFFFF, SEED >> 32)
    first_try = 0
    for j in range(n):
        i = first + j
        U = orc.uniforms(SEED, i)
        a, c = 2.0 * U[1] - 1.0, 2.0 * U[2] - 1.0
        k = 0
        while a * a + c * c > 1.0:
            k += 1
            w = orc.philox4x32_10((i & 0xFFFFFFFF, i >> 32, 2 + k, 0), key)
            a, c = 2.0 * _u52(w[0], w[1]) - 1.0, 2.0 * _u52(w[2], w[3]) - 1.0
        first_try += k == 0
        assert st[1][j] == RAD * a and st[2][j] == RAD * c, (j, k)          # eT = (0,1,0), eZ = (0,0,1): exact products
    p = math.pi / 4
    assert abs(first_try / n - p) < 4 * math.sqrt(p * (1 - p) / n)


def test_p22_counter_based_and_tilted_frame():
    b = _beam(origin=(0.8, 0.01, -0.02), axis=(-0.6, 0.0, 0.8), eT=(0.0, 1.0, 0.0), eZ=(0.8, 0.0, 0.6), sigma_ang_rad=2e-3)
    a = orc.seed(b, wl.depth_cdf(), wl.normal_cdf(), 9, 100, 5000)
    c = orc.seed(b, wl.depth_cdf(), wl.normal_cdf(), 9, 1100, 77)
    for k in range(6):
        assert np.array_equal(a[k][1000:1077], c[k])                       # a sub-range reproduces the same ions
    # offsets from the beam axis lie in the plane spanned by eT, eZ and inside the disc
    r = np.stack([a[0], a[1], a[2]], 1) - np.array(b.origin)
    d = r @ np.array(b.axis)
    off = r - np.outer(d, b.axis)
    assert np.linalg.norm(off, axis=1).max() <= RAD * (1 + 1e-12)
    assert d.min() >= 0 and d.max() <= b.depth_max
