"""P25: the grazing flags of the oracle (north_star: results within 1e-9 m of a decision boundary are flagged and left out
of the bit-exact comparison on both sides; SURVEY.md 8(b) flag bits; PAPER.md L326 plane test, L318 grid test, L330 segments).

These bits decide WHICH ions every parity test drops, so they are pinned here against straight-line flights whose distance
to the boundary is known in closed form (B = 0 on a gridded field: r_k = r_0 + k v dt exactly, up to 1e-16 m of rounding):
  bit 2 (plane): |s| < 1e-9 m at the start or at an end of a step -- 5e-10 m before / behind the plane sets it, 2e-9 m does not;
  bit 4 (grid):  within 1e-9 m of Rmin / Rmax / Zmin / Zmax at the start or at an end of a step, inside or outside;
  bit 1 (edge):  hit within 1e-9 m of a segment edge in u or w; every other hit has flags == 0."""
import numpy as np

import oracle as orc
from paper_2506_15812_b200 import workloads as wl

QM_LI = wl.E_CHARGE / wl.MASS_LI7
DT, V = 1e-9, 1e6            # 1 mm per step


def _zero_field():
    grid, nodal = wl.nodal_field_2d(9, 17)               # R in [0.25, 0.875], Z in [-0.625, 0.625]
    return grid, orc.OracleField(grid, [np.zeros_like(c) for c in nodal])


def _fly(f, det, x0, vx=V, z0=0.0, vz=0.0, nmax=20):
    n = len(x0)
    st = [np.asarray(x0, float), np.zeros(n), np.full(n, z0), np.full(n, vx), np.zeros(n), np.full(n, vz)]
    return orc.trace(f, QM_LI, st, None, DT, nmax, det)


def test_p25_plane_flag():
    grid, f = _zero_field()
    XD = 0.80
    det = wl.Detector((XD, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), *([np.array([-1.0]), np.array([1.0])] * 2))
    #        ends step 3 just before | just behind | 2e-9 before | 2e-9 behind | mid-step crossing | starts 5e-10 before the plane
    x0 = XD - 3e-3 + np.array([-5e-10, +5e-10, -2e-9, +2e-9, -0.5e-3, 3e-3 - 5e-10])
    r = _fly(f, det, x0)
    assert list(r["status"]) == [0] * 6
    assert list(r["steps"]) == [4, 3, 4, 3, 4, 1]         # s1 >= 0 decides the crossing step: graze or not, the count is exact
    assert list(r["flags"]) == [2, 2, 0, 0, 0, 2]
    assert np.abs(r["u"]).max() < 1e-15 and np.abs(r["w"]).max() < 1e-15
    # the threshold itself: 0.9e-9 is flagged, 1.1e-9 is not (both sides of the plane)
    r = _fly(f, det, XD - 3e-3 + np.array([-0.9e-9, 0.9e-9, -1.1e-9, 1.1e-9]))
    assert list(r["flags"]) == [2, 2, 0, 0]
    # a start on or behind the plane is a bad start, flagged when within the threshold
    r = _fly(f, det, XD + np.array([0.0, 5e-10, 1e-3]))
    assert list(r["status"]) == [-4, -4, -4] and list(r["flags"]) == [2, 2, 0] and list(r["steps"]) == [0, 0, 0]


def test_p25_grid_flag():
    grid, f = _zero_field()
    far = wl.Detector((5.0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), *([np.array([-1.0]), np.array([1.0])] * 2))
    # outward in +x (R = x): step 3 ends 5e-10 inside Rmax | 5e-10 outside | 2e-9 inside | 2e-9 outside | mid-step
    x0 = grid.Rmax - 3e-3 + np.array([-5e-10, +5e-10, -2e-9, +2e-9, -0.5e-3])
    r = _fly(f, far, x0)
    assert list(r["status"]) == [-3] * 5
    assert list(r["steps"]) == [4, 3, 4, 3, 4]
    assert list(r["flags"]) == [4, 4, 0, 0, 0]
    # inward towards Rmin, and vertically towards Zmax / Zmin
    back = wl.Detector((-5.0, 0, 0), (-1, 0, 0), (0, 1, 0), (0, 0, 1), *([np.array([-1.0]), np.array([1.0])] * 2))
    r = _fly(f, back, grid.Rmin + 3e-3 + np.array([5e-10, -5e-10, 2e-9, -2e-9]), vx=-V)
    assert list(r["status"]) == [-3] * 4 and list(r["steps"]) == [4, 3, 4, 3] and list(r["flags"]) == [4, 4, 0, 0]
    for zb, sgn in ((grid.Zmax, 1.0), (grid.Zmin, -1.0)):
        n = 4
        z0 = zb - sgn * 3e-3 + sgn * np.array([-5e-10, 5e-10, -2e-9, 2e-9])
        st = [np.full(n, 0.5), np.zeros(n), z0, np.full(n, 1.0), np.zeros(n), np.full(n, sgn * V)]
        r = orc.trace(f, QM_LI, st, None, DT, 20, far)
        assert list(r["status"]) == [-3] * 4 and list(r["steps"]) == [4, 3, 4, 3] and list(r["flags"]) == [4, 4, 0, 0]
    # a start within the threshold of the boundary: inside -> flagged and traced, outside -> bad start, flagged
    r = _fly(f, far, grid.Rmax + np.array([-5e-10, 5e-10, 1e-3]))
    assert list(r["status"]) == [-3, -4, -4] and list(r["flags"]) == [4, 4, 0]


def test_p25_edge_flag_only_near_an_edge():
    rng = np.random.default_rng(25)
    u_lo, u_hi = np.array([-4e-3, -2.5e-3, -1e-3, 1.2e-3]), np.array([-2.7e-3, -1e-3, 1e-3, 3e-3])
    w_lo, w_hi = np.array([-3e-3, 0.0, 2e-3]), np.array([-0.5e-3, 2e-3, 4e-3])
    det = wl.Detector((0.82, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), u_lo, u_hi, w_lo, w_hi)
    n = 4000
    u, w = rng.uniform(-5e-3, 4e-3, n), rng.uniform(-4e-3, 5e-3, n)
    eu, ew = np.concatenate([u_lo, u_hi]), np.concatenate([w_lo, w_hi])
    k = 200                                               # a few hundred hits placed at known distances from an edge
    d = rng.choice([-5e-10, 5e-10, -0.9e-9, 0.9e-9, -1.1e-9, 1.1e-9, -2e-9, 2e-9], 2 * k)
    u[:k] = rng.choice(eu, k) + d[:k]
    w[k:2 * k] = rng.choice(ew, k) + d[k:]
    status = rng.choice([0, 0, 0, -2, -3, -4], n).astype(np.int32)
    status[:2 * k:2] = 0
    pre = rng.choice([0, 2, 4], n).astype(np.uint8)       # bits the trace set before: kept
    res = dict(status=status, u=u, w=w, flags=pre.copy())
    orc.histogram(res, None, det, 1)
    near = (np.abs(u[:, None] - eu[None, :]).min(axis=1) < 1e-9) | (np.abs(w[:, None] - ew[None, :]).min(axis=1) < 1e-9)
    crossed = status == 0
    assert near[crossed].sum() > 100 and (~near[crossed]).sum() > 1500
    assert np.array_equal(res["flags"], pre | (near & crossed).astype(np.uint8))
    assert np.all(res["flags"][crossed & ~near & (pre == 0)] == 0)          # interior hits carry no flag at all
