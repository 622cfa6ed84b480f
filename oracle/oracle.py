"""TEST INFRASTRUCTURE -- NOT PRODUCT CODE.

ctypes front-end of the CPU oracle (oracle/taiga_oracle.cpp).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
It imports nothing from the CUDA path; inputs come from paper_2506_15812_b200.workloads,
which holds no method arithmetic.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build as _build  # noqa: E402

_lib = C.CDLL(_build.build())

_dp = C.POINTER(C.c_double)
D3 = C.c_double * 3


class Field(C.Structure):
    _fields_ = [("kind", C.c_int), ("nR", C.c_int), ("nZ", C.c_int), ("nS", C.c_int),
                ("Rmin", C.c_double), ("Rmax", C.c_double), ("Zmin", C.c_double),
                ("Zmax", C.c_double), ("s0", C.c_double), ("ds", C.c_double),
                ("coef", _dp * 3), ("par", C.c_double * 8), ("E", C.c_double * 3), ("ecoef", _dp * 3)]


class DetectorS(C.Structure):
    _fields_ = [("origin", D3), ("normal", D3), ("eu", D3), ("ew", D3),
                ("nu", C.c_int), ("nw", C.c_int),
                ("u_lo", _dp), ("u_hi", _dp), ("w_lo", _dp), ("w_hi", _dp)]


class BeamS(C.Structure):
    _fields_ = [("v0", C.c_double), ("origin", D3), ("axis", D3), ("eT", D3), ("eZ", D3),
                ("cdf_depth", _dp), ("n_depth", C.c_int), ("depth_max", C.c_double),
                ("cdf_normal", _dp), ("n_normal", C.c_int), ("z_max", C.c_double),
                ("sigma_pos", C.c_double), ("sigma_ang", C.c_double),
                ("profile", C.c_int), ("radius", C.c_double)]


def _p(a):
    return a.ctypes.data_as(_dp)


_lib.orc_cdf_invert.restype = C.c_double
_lib.orc_cdf_invert.argtypes = [_dp, C.c_int, C.c_double, C.c_double]
_lib.orc_build_tables.restype = C.c_int
_lib.orc_spline_notaknot.restype = C.c_int
_lib.orc_spline_periodic.restype = C.c_int
_lib.orc_max_threads.restype = C.c_int

KIND_UNIFORM, KIND_GRADB, KIND_INVR, KIND_SOLOVEV = 10, 11, 12, 13


def max_threads() -> int:
    return int(_lib.orc_max_threads())


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    _lib.orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def uniforms(seed: int, index: int):
    u = (C.c_double * 5)()
    _lib.orc_uniforms(C.c_uint64(seed), C.c_uint64(index), u)
    return np.array(u[:])


def cdf_invert(F, x_max, U):
    F = np.ascontiguousarray(F, dtype=np.float64)
    return float(_lib.orc_cdf_invert(_p(F), len(F) - 1, x_max, U))


def spline_notaknot(y):
    y = np.ascontiguousarray(y, dtype=np.float64)
    c = np.empty((len(y) - 1, 4))
    assert _lib.orc_spline_notaknot(len(y), _p(y), _p(c)) == 0
    return c


def spline_periodic(y):
    y = np.ascontiguousarray(y, dtype=np.float64)
    c = np.empty((len(y), 4))
    assert _lib.orc_spline_periodic(len(y), _p(y), _p(c)) == 0
    return c


class OracleField:
    """Spline-table field (kind 0/1/2) built from nodal grids, or an analytic pin field."""

    def __init__(self, grid=None, nodal=None, kind=None, par=(), E=(0.0, 0.0, 0.0), E_nodal=None, E_grid=None):
        """E: uniform electric field; E_nodal: (E_R, E_Z, E_phi) nodal values [nR][nZ] of a static gridded field on the
        (R, Z) grid of `grid` (or of `E_grid` for the analytic pin fields)."""
        self.s = Field()
        self._keep = []
        if E_nodal is not None:
            g = grid if grid is not None else E_grid
            self.etables = []
            for c in range(3):
                nod = np.ascontiguousarray(np.asarray(E_nodal[c], dtype=np.float64).reshape(1, g.nR, g.nZ))
                tab = np.empty((1, g.nR - 1, g.nZ - 1, 16))
                assert _lib.orc_build_tables(C.c_int(0), C.c_int(g.nR), C.c_int(g.nZ), C.c_int(1), _p(nod), _p(tab)) == 0
                self.etables.append(tab)
                self.s.ecoef[c] = _p(tab)
            if grid is None:
                self.s.nR, self.s.nZ, self.s.nS = g.nR, g.nZ, 1
                self.s.Rmin, self.s.Rmax, self.s.Zmin, self.s.Zmax = g.Rmin, g.Rmax, g.Zmin, g.Zmax
        if grid is not None:
            g = grid
            self.s.kind, self.s.nR, self.s.nZ, self.s.nS = g.kind, g.nR, g.nZ, g.nS
            self.s.Rmin, self.s.Rmax, self.s.Zmin, self.s.Zmax = g.Rmin, g.Rmax, g.Zmin, g.Zmax
            self.s.s0, self.s.ds = g.s0, g.ds
            per = 64 if g.kind == 2 else 16
            self.tables = []
            for c in range(3):
                nod = np.ascontiguousarray(nodal[c], dtype=np.float64)
                assert nod.shape == (g.nS, g.nR, g.nZ)
                tab = np.empty((g.nS, g.nR - 1, g.nZ - 1, per))
                rc = _lib.orc_build_tables(C.c_int(g.kind), C.c_int(g.nR), C.c_int(g.nZ),
                                           C.c_int(g.nS), _p(nod), _p(tab))
                assert rc == 0
                self.tables.append(tab)
                self.s.coef[c] = _p(tab)
        else:
            self.s.kind = kind
            for i, v in enumerate(par):
                self.s.par[i] = v
        for i in range(3):
            self.s.E[i] = E[i]

    def B(self, r, t=0.0):
        out = D3()
        _lib.orc_field_B(C.byref(self.s), D3(*r), C.c_double(t), out)
        return np.array(out[:])

    def E(self, r):
        out = D3()
        _lib.orc_field_E(C.byref(self.s), D3(*r), out)
        return np.array(out[:])

    def cyl(self, R, Z, s=0.0):
        out = D3()
        _lib.orc_field_cyl(C.byref(self.s), C.c_double(R), C.c_double(Z), C.c_double(s), out)
        return np.array(out[:])


def rkn_advance(field: OracleField, qm, r, v, t, dt, nsteps, variant=0):
    rr, vv, tt = D3(*r), D3(*v), C.c_double(t)
    _lib.orc_rkn_advance(C.byref(field.s), C.c_double(qm), C.c_int(variant), rr, vv,
                         C.byref(tt), C.c_double(dt), C.c_uint64(nsteps))
    return np.array(rr[:]), np.array(vv[:]), tt.value


def _det_struct(det):
    d = DetectorS()
    d.origin, d.normal, d.eu, d.ew = D3(*det.origin), D3(*det.normal), D3(*det.eu), D3(*det.ew)
    d.nu, d.nw = det.nu, det.nw
    keep = [np.ascontiguousarray(a, dtype=np.float64) for a in (det.u_lo, det.u_hi, det.w_lo, det.w_hi)]
    d.u_lo, d.u_hi, d.w_lo, d.w_hi = (_p(a) for a in keep)
    return d, keep


def beam_v0(beam) -> float:
    """v0 = sqrt(2 E e / m), non-relativistic (O0)."""
    return math.sqrt(2.0 * beam.energy_eV * beam.charge_C / beam.mass_kg)


def seed(beam, cdf_depth, cdf_normal, seed_value, first_index, n):
    b = BeamS()
    b.v0 = beam_v0(beam)
    b.origin, b.axis, b.eT, b.eZ = D3(*beam.origin), D3(*beam.axis), D3(*beam.eT), D3(*beam.eZ)
    cd = np.ascontiguousarray(cdf_depth, dtype=np.float64)
    cn = np.ascontiguousarray(cdf_normal, dtype=np.float64)
    b.cdf_depth, b.n_depth, b.depth_max = _p(cd), len(cd) - 1, beam.depth_max
    b.cdf_normal, b.n_normal, b.z_max = _p(cn), len(cn) - 1, beam.z_max
    b.sigma_pos, b.sigma_ang = beam.sigma_pos_m, beam.sigma_ang_rad
    b.profile, b.radius = int(getattr(beam, "profile", 0)), float(getattr(beam, "radius_m", 0.0))
    out = [np.empty(n) for _ in range(6)]
    _lib.orc_seed(C.byref(b), C.c_uint64(seed_value), C.c_uint64(first_index), C.c_uint64(n),
                  *[_p(a) for a in out])
    return out


def seed_grid(beam, cdf_depth, cdf_normal, nd, nT, nZ, z_lim, first_index, n):
    """Deterministic weighted-grid initialisation (L314, reading D1): returns (state6, w0)."""
    b = BeamS()
    b.v0 = beam_v0(beam)
    b.origin, b.axis, b.eT, b.eZ = D3(*beam.origin), D3(*beam.axis), D3(*beam.eT), D3(*beam.eZ)
    cd = np.ascontiguousarray(cdf_depth, dtype=np.float64)
    cn = np.ascontiguousarray(cdf_normal, dtype=np.float64)
    b.cdf_depth, b.n_depth, b.depth_max = _p(cd), len(cd) - 1, beam.depth_max
    b.cdf_normal, b.n_normal, b.z_max = _p(cn), len(cn) - 1, beam.z_max
    b.sigma_pos, b.sigma_ang = beam.sigma_pos_m, 0.0
    out = [np.empty(n) for _ in range(7)]
    _lib.orc_seed_grid(C.byref(b), C.c_int(nd), C.c_int(nT), C.c_int(nZ), C.c_double(z_lim),
                       C.c_uint64(first_index), C.c_uint64(n), *[_p(a) for a in out])
    return out[:6], out[6]


def trace(field: OracleField, qm, state, t0, dt, max_steps, det, variant=0, nthreads=0,
          want_xyz=False, interp=0):
    x, y, z, vx, vy, vz = [np.ascontiguousarray(a, dtype=np.float64) for a in state]
    n = len(x)
    d, keep = _det_struct(det)
    status = np.empty(n, dtype=np.int32)
    u, w = np.empty(n), np.empty(n)
    steps = np.empty(n, dtype=np.uint32)
    flags = np.empty(n, dtype=np.uint8)
    xyz = np.empty((n, 3)) if want_xyz else None
    t0a = None if t0 is None else np.ascontiguousarray(t0, dtype=np.float64)
    _lib.orc_trace_interp(C.byref(field.s), C.c_double(qm), C.c_int(variant), C.c_int(interp), C.c_uint64(n),
                   _p(x), _p(y), _p(z), _p(vx), _p(vy), _p(vz),
                   _p(t0a) if t0a is not None else None,
                   C.c_double(dt), C.c_uint32(max_steps), C.byref(d),
                   status.ctypes.data_as(C.c_void_p), _p(u), _p(w),
                   _p(xyz) if want_xyz else None,
                   steps.ctypes.data_as(C.c_void_p), flags.ctypes.data_as(C.c_void_p),
                   C.c_int(nthreads))
    res = dict(status=status, u=u, w=w, steps=steps, flags=flags)
    if want_xyz:
        res["xyz"] = xyz
    return res


def histogram(res, group, det, n_hist, counts=None, summary=None):
    """Bins res (from trace) in place: adds 'cell', updates 'flags'; returns counts, summary."""
    n = len(res["status"])
    d, keep = _det_struct(det)
    cell = res["status"].copy()
    if counts is None:
        counts = np.zeros((n_hist, det.nw, det.nu), dtype=np.uint64)
    if summary is None:
        summary = np.zeros((n_hist, 6), dtype=np.uint64)
    grp = None if group is None else np.ascontiguousarray(group, dtype=np.uint16)
    _lib.orc_histogram(C.c_uint64(n), cell.ctypes.data_as(C.c_void_p), _p(res["u"]), _p(res["w"]),
                       grp.ctypes.data_as(C.c_void_p) if grp is not None else None,
                       res["flags"].ctypes.data_as(C.c_void_p), C.byref(d), C.c_int(n_hist),
                       counts.ctypes.data_as(C.c_void_p), summary.ctypes.data_as(C.c_void_p))
    res["cell"] = cell
    return counts, summary


def run_config(cfg, field: OracleField | None = None, nthreads=0, variant=0, interp=0):
    """Whole hot path (a1-a5) of one workloads.Config on the CPU oracle."""
    from paper_2506_15812_b200 import workloads as wl
    if field is None:
        grid, nodal = cfg.field_builder()
        field = OracleField(grid, nodal)
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    counts = np.zeros((cfg.n_hist, (cfg.detector or cfg.groups[0].detector).nw,
                       (cfg.detector or cfg.groups[0].detector).nu), dtype=np.uint64)
    summary = np.zeros((cfg.n_hist, 6), dtype=np.uint64)
    per_group = []
    for g in cfg.groups:
        det = g.detector or cfg.detector
        st = seed(g.beam, cd, cn, cfg.seed, g.first_index, g.n_ions)
        qm = g.beam.charge_C / g.beam.mass_kg
        t0 = np.full(g.n_ions, g.t0)
        res = trace(field, qm, st, t0, cfg.dt, cfg.max_steps, det, variant, nthreads, interp=interp)
        grp = np.full(g.n_ions, g.group, dtype=np.uint16)
        histogram(res, grp, det, cfg.n_hist, counts, summary)
        res["state0"] = st
        res["group"] = grp
        per_group.append(res)
    return dict(counts=counts, summary=summary, groups=per_group, field=field)


# ---- secondary-ionisation loss (Eq. 2) -----------------
class LossS(C.Structure):
    _fields_ = [("psi_coef", _dp), ("n", C.c_int), ("psi0", C.c_double), ("dpsi", C.c_double),
                ("rate", _dp)]


_lib.orc_mcwhirter_rate.restype = C.c_double
_lib.orc_mcwhirter_rate.argtypes = [C.c_double, C.c_double, C.c_double]


def mcwhirter_rate(ne, Te, E12):
    """Eq. 2: per-ion secondary ionisation rate [1/s]; scalars or arrays."""
    ne, Te = np.broadcast_arrays(np.asarray(ne, dtype=np.float64), np.asarray(Te, dtype=np.float64))
    out = np.array([_lib.orc_mcwhirter_rate(float(a), float(b), float(E12)) for a, b in zip(ne.ravel(), Te.ravel())])
    return out.reshape(ne.shape) if ne.shape else float(out[0])


class OracleLoss:
    """psi(R,Z) spline table on the field's (R,Z) grid + rate profile nu(psi0 + k dpsi)."""

    def __init__(self, grid, psi_nodal, psi0, dpsi, rate):
        nod = np.ascontiguousarray(psi_nodal, dtype=np.float64).reshape(1, grid.nR, grid.nZ)
        self.table = np.empty((1, grid.nR - 1, grid.nZ - 1, 16))
        rc = _lib.orc_build_tables(C.c_int(0), C.c_int(grid.nR), C.c_int(grid.nZ), C.c_int(1), _p(nod), _p(self.table))
        assert rc == 0
        self.rate = np.ascontiguousarray(rate, dtype=np.float64)
        self.s = LossS(_p(self.table), len(self.rate), float(psi0), float(dpsi), _p(self.rate))


def trace_loss(field: OracleField, loss: OracleLoss, qm, state, t0, dt, max_steps, det, variant=0, nthreads=0, w0=None, interp=0):
    x, y, z, vx, vy, vz = [np.ascontiguousarray(a, dtype=np.float64) for a in state]
    n = len(x)
    d, keep = _det_struct(det)
    status = np.empty(n, dtype=np.int32)
    u, w, weight = np.empty(n), np.empty(n), np.empty(n)
    steps = np.empty(n, dtype=np.uint32)
    flags = np.empty(n, dtype=np.uint8)
    t0a = None if t0 is None else np.ascontiguousarray(t0, dtype=np.float64)
    _lib.orc_trace_loss_interp(C.byref(field.s), C.byref(loss.s), C.c_double(qm), C.c_int(variant), C.c_int(interp), C.c_uint64(n),
                        _p(x), _p(y), _p(z), _p(vx), _p(vy), _p(vz),
                        _p(t0a) if t0a is not None else None,
                        C.c_double(dt), C.c_uint32(max_steps), C.byref(d),
                        status.ctypes.data_as(C.c_void_p), _p(u), _p(w),
                        steps.ctypes.data_as(C.c_void_p), flags.ctypes.data_as(C.c_void_p),
                        _p(np.ascontiguousarray(w0, dtype=np.float64)) if w0 is not None else None, _p(weight),
                        C.c_int(nthreads))
    return dict(status=status, u=u, w=w, steps=steps, flags=flags, weight=weight)


def histogram_weighted(res, group, det, n_hist, wcounts=None, wsummary=None):
    """32.32 fixed-point weighted counters of res (after histogram(): needs res['cell'])."""
    n = len(res["cell"])
    d, keep = _det_struct(det)
    if wcounts is None:
        wcounts = np.zeros((n_hist, det.nw, det.nu), dtype=np.uint64)
    if wsummary is None:
        wsummary = np.zeros((n_hist, 4), dtype=np.uint64)
    grp = None if group is None else np.ascontiguousarray(group, dtype=np.uint16)
    cell = np.ascontiguousarray(res["cell"], dtype=np.int32)
    wt = np.ascontiguousarray(res["weight"], dtype=np.float64)
    _lib.orc_histogram_weighted(C.c_uint64(n), cell.ctypes.data_as(C.c_void_p), _p(wt),
                                grp.ctypes.data_as(C.c_void_p) if grp is not None else None,
                                C.byref(d), C.c_int(n_hist), wcounts.ctypes.data_as(C.c_void_p),
                                wsummary.ctypes.data_as(C.c_void_p))
    return wcounts, wsummary
