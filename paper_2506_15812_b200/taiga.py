"""Thin ctypes binding of the C ABI in include/taiga.h (libtaiga.so).

Argument marshalling only: every step of the hot path runs in the CUDA kernels behind the ABI.
PyTorch is used for device memory and streams.  Importing this module fails loudly when the
library has not been built; there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtaiga.so")
if not os.path.exists(LIB_PATH):
    raise ImportError("libtaiga.so is missing: run `python paper_2506_15812_b200/build.py` "
                      "(or __graft_entry__.build()); there is no CPU fallback")
_lib = C.CDLL(LIB_PATH)

_dp = C.POINTER(C.c_double)
D3 = C.c_double * 3

OK, E_ARG, E_STATE, E_CUDA, E_NOMEM = 0, -1, -2, -3, -4
CELL_MISS, CELL_MAXSTEPS, CELL_OUT, CELL_BADSTART = -1, -2, -3, -4
FLAG_EDGE, FLAG_PLANE, FLAG_GRID = 1, 2, 4
STATIC_MAX_SEGMENTS = 2048       # TAIGA_STATIC_MAX_SEGMENTS

EXPORTS = ["taiga_create", "taiga_destroy", "taiga_last_error", "taiga_load_field", "taiga_load_loss",
           "taiga_detector_histogram_weighted", "taiga_seed_beam_grid",
           "taiga_field_eval", "taiga_field_table", "taiga_seed_beam", "taiga_trace",
           "taiga_detector_histogram", "taiga_set_efield", "taiga_load_efield", "taiga_set_option", "taiga_get_stats",
           "taiga_measure_fp64_peak", "taiga_measure_l1_gather_peak", "taiga_measure_dmma_peak", "taiga_measure_mixed_fp64_peak",
           "taiga_loss_statistics", "taiga_detector_histogram_static"]


class GridS(C.Structure):
    _fields_ = [("kind", C.c_int), ("nR", C.c_int), ("nZ", C.c_int), ("nS", C.c_int),
                ("Rmin", C.c_double), ("Rmax", C.c_double), ("Zmin", C.c_double),
                ("Zmax", C.c_double), ("s0", C.c_double), ("ds", C.c_double)]


class CoeffsS(C.Structure):
    _fields_ = [("form", C.c_int), ("BR", C.c_void_p), ("BZ", C.c_void_p), ("Bphi", C.c_void_p),
                ("on_device", C.c_int)]


class BeamS(C.Structure):
    _fields_ = [("mass_kg", C.c_double), ("charge_C", C.c_double), ("energy_eV", C.c_double),
                ("origin", D3), ("axis", D3), ("eT", D3), ("eZ", D3),
                ("cdf_depth", C.c_void_p), ("n_depth", C.c_int), ("depth_max", C.c_double),
                ("cdf_normal", C.c_void_p), ("n_normal", C.c_int), ("z_max", C.c_double),
                ("sigma_pos_m", C.c_double), ("sigma_ang_rad", C.c_double),
                ("first_index", C.c_uint64), ("group", C.c_uint16), ("t0", C.c_double),
                ("profile", C.c_int), ("radius_m", C.c_double)]


class IonsS(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("x", "y", "z", "vx", "vy", "vz", "hit_u", "hit_w",
                                          "cell", "steps", "flags", "group", "t0", "weight", "w0")] + [("n", C.c_uint64)]


class SeedGridS(C.Structure):
    _fields_ = [("nd", C.c_int), ("nT", C.c_int), ("nZ", C.c_int), ("z_lim", C.c_double)]


class LossProfileS(C.Structure):
    _fields_ = [("n", C.c_int), ("psi0", C.c_double), ("dpsi", C.c_double), ("ne", C.c_void_p),
                ("Te", C.c_void_p), ("E12", C.c_double)]


class DetS(C.Structure):
    _fields_ = [("origin", D3), ("normal", D3), ("eu", D3), ("ew", D3), ("nu", C.c_int),
                ("nw", C.c_int), ("u_lo", C.c_void_p), ("u_hi", C.c_void_p),
                ("w_lo", C.c_void_p), ("w_hi", C.c_void_p)]


_lib.taiga_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p]
_lib.taiga_destroy.argtypes = [C.c_void_p]
_lib.taiga_last_error.argtypes = [C.c_void_p]
_lib.taiga_last_error.restype = C.c_char_p
_lib.taiga_load_field.argtypes = [C.c_void_p, C.POINTER(GridS), C.POINTER(CoeffsS)]
_lib.taiga_field_eval.argtypes = [C.c_void_p, C.c_uint64] + [C.c_void_p] * 6
_lib.taiga_field_table.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
_lib.taiga_seed_beam.argtypes = [C.c_void_p, C.POINTER(BeamS), C.c_uint64, C.POINTER(IonsS)]
_lib.taiga_trace.argtypes = [C.c_void_p, C.POINTER(IonsS), C.c_double, C.c_double, C.c_uint32,
                             C.POINTER(DetS), C.c_int]
_lib.taiga_detector_histogram.argtypes = [C.c_void_p, C.POINTER(IonsS), C.POINTER(DetS), C.c_int,
                                          C.c_void_p, C.c_void_p]
_lib.taiga_detector_histogram_static.argtypes = _lib.taiga_detector_histogram.argtypes
_lib.taiga_seed_beam_grid.argtypes = [C.c_void_p, C.POINTER(BeamS), C.POINTER(SeedGridS), C.POINTER(IonsS)]
_lib.taiga_load_loss.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.POINTER(LossProfileS)]
_lib.taiga_detector_histogram_weighted.argtypes = [C.c_void_p, C.POINTER(IonsS), C.POINTER(DetS), C.c_int,
                                                   C.c_void_p, C.c_void_p]
_lib.taiga_set_efield.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
_lib.taiga_load_efield.argtypes = [C.c_void_p, C.POINTER(CoeffsS)]
_lib.taiga_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_longlong]
_lib.taiga_get_stats.argtypes = [C.c_void_p, C.POINTER(C.c_ulonglong * 8)]
_lib.taiga_measure_fp64_peak.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
_lib.taiga_measure_l1_gather_peak.argtypes = [C.c_void_p, C.c_double, C.c_int, C.POINTER(C.c_double)]
_lib.taiga_measure_dmma_peak.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
_lib.taiga_measure_mixed_fp64_peak.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_double)]
_lib.taiga_loss_statistics.argtypes = [C.POINTER(C.c_ulonglong * 4), C.POINTER(C.c_double * 3)]


class TaigaError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("taiga error %d: %s" % (code, msg))
        self.code = code


class Ions:
    """SoA ion storage on the device (torch tensors); `view(a, b)` gives a sub-range."""
    _specs = (("x", torch.float64), ("y", torch.float64), ("z", torch.float64),
              ("vx", torch.float64), ("vy", torch.float64), ("vz", torch.float64),
              ("hit_u", torch.float64), ("hit_w", torch.float64), ("cell", torch.int32),
              ("steps", torch.int32), ("flags", torch.uint8), ("group", torch.int16),
              ("t0", torch.float64), ("weight", torch.float64), ("w0", torch.float64))

    def __init__(self, n, device="cuda:0", _arrays=None, _meta=None):
        self.n = int(n)
        if _arrays is None:
            _arrays = {k: torch.zeros(self.n, dtype=dt, device=device) for k, dt in self._specs}
        self.a = _arrays
        # use_w0: the w0 array holds initial weights (set by seed_beam_grid, cleared by seed_beam);
        # otherwise a null w0 pointer (= weight 1) is passed to the library
        self.meta = _meta if _meta is not None else {"use_w0": False}

    def view(self, lo, hi):
        return Ions(hi - lo, _arrays={k: v[lo:hi] for k, v in self.a.items()}, _meta=self.meta)

    def struct(self, weight=True):
        s = IonsS()
        for k, _ in self._specs:
            setattr(s, k, self.a[k].data_ptr() if self.n else None)
        if not self.meta["use_w0"]:
            s.w0 = None
        if not weight:
            s.weight = None
        s.n = self.n
        return s

    def __getattr__(self, k):
        if k in ("a", "n", "meta"):
            raise AttributeError(k)
        return self.a[k]


def _host(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Taiga:
    """One context = one device + one stream (torch's current stream at construction)."""

    def __init__(self, device=0):
        self.device = int(device)
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = _lib.taiga_create(C.byref(h), self.device, C.c_void_p(self.stream.cuda_stream))
        if rc:
            raise TaigaError(rc, "taiga_create failed (no sm_100 device?)")
        self.h = h
        self._keep = []

    def close(self):
        if self.h:
            _lib.taiga_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc):
        if rc:
            raise TaigaError(rc, _lib.taiga_last_error(self.h).decode())

    def load_field(self, grid, comps, form=0):
        """comps: (BR, BZ, Bphi) numpy arrays (host) or torch cuda tensors (device)."""
        g = GridS(grid.kind, grid.nR, grid.nZ, grid.nS, grid.Rmin, grid.Rmax, grid.Zmin, grid.Zmax,
                  grid.s0, grid.ds)
        on_dev = isinstance(comps[0], torch.Tensor)
        if on_dev:
            keep = [c.contiguous() for c in comps]
            ptrs = [c.data_ptr() for c in keep]
        else:
            keep = [_host(c) for c in comps]
            ptrs = [c.ctypes.data for c in keep]
        co = CoeffsS(form, ptrs[0], ptrs[1], ptrs[2], 1 if on_dev else 0)
        self._chk(_lib.taiga_load_field(self.h, C.byref(g), C.byref(co)))
        if on_dev:
            self._keep = keep            # device inputs are read asynchronously

    def load_efield(self, comps):
        """comps: (E_R, E_Z, E_phi) nodal arrays [nR][nZ] on the loaded grid (numpy or torch cuda), or None to remove."""
        if comps is None:
            self._chk(_lib.taiga_load_efield(self.h, None))
            return
        on_dev = isinstance(comps[0], torch.Tensor)
        if on_dev:
            keep = [c.contiguous() for c in comps]
            ptrs = [c.data_ptr() for c in keep]
        else:
            keep = [_host(c) for c in comps]
            ptrs = [c.ctypes.data for c in keep]
        co = CoeffsS(0, ptrs[0], ptrs[1], ptrs[2], 1 if on_dev else 0)
        self._chk(_lib.taiga_load_efield(self.h, C.byref(co)))
        if on_dev:
            self._keep_e = keep

    def field_eval(self, R, Z, s=None):
        R, Z = R.contiguous(), Z.contiguous()
        out = [torch.empty_like(R) for _ in range(3)]
        self._chk(_lib.taiga_field_eval(self.h, R.numel(), R.data_ptr(), Z.data_ptr(),
                                        s.contiguous().data_ptr() if s is not None else None,
                                        *[o.data_ptr() for o in out]))
        return out

    def field_table(self, comp, shape):
        host = np.empty(shape, dtype=np.float64)
        self._chk(_lib.taiga_field_table(self.h, comp, host.ctypes.data))
        return host

    def seed_beam(self, beam, cdf_depth, cdf_normal, seed, ions, first_index=0, group=0, t0=0.0):
        cd, cn = _host(cdf_depth), _host(cdf_normal)
        p = BeamS()
        p.mass_kg, p.charge_C, p.energy_eV = beam.mass_kg, beam.charge_C, beam.energy_eV
        p.origin, p.axis, p.eT, p.eZ = D3(*beam.origin), D3(*beam.axis), D3(*beam.eT), D3(*beam.eZ)
        p.cdf_depth, p.n_depth, p.depth_max = cd.ctypes.data, len(cd) - 1, beam.depth_max
        p.cdf_normal, p.n_normal, p.z_max = cn.ctypes.data, len(cn) - 1, beam.z_max
        p.sigma_pos_m, p.sigma_ang_rad = beam.sigma_pos_m, beam.sigma_ang_rad
        p.first_index, p.group, p.t0 = int(first_index), int(group), float(t0)
        p.profile, p.radius_m = int(getattr(beam, "profile", 0)), float(getattr(beam, "radius_m", 0.0))
        ions.meta["use_w0"] = False
        s = ions.struct()
        self._chk(_lib.taiga_seed_beam(self.h, C.byref(p), C.c_uint64(seed), C.byref(s)))

    def seed_beam_grid(self, beam, cdf_depth, cdf_normal, nd, nT, nZ, z_lim, ions, first_index=0, group=0, t0=0.0):
        """Deterministic weighted-grid initialisation; writes ions.w0."""
        cd, cn = _host(cdf_depth), _host(cdf_normal)
        p = BeamS()
        p.mass_kg, p.charge_C, p.energy_eV = beam.mass_kg, beam.charge_C, beam.energy_eV
        p.origin, p.axis, p.eT, p.eZ = D3(*beam.origin), D3(*beam.axis), D3(*beam.eT), D3(*beam.eZ)
        p.cdf_depth, p.n_depth, p.depth_max = cd.ctypes.data, len(cd) - 1, beam.depth_max
        p.cdf_normal, p.n_normal, p.z_max = cn.ctypes.data, len(cn) - 1, beam.z_max
        p.sigma_pos_m, p.sigma_ang_rad = beam.sigma_pos_m, 0.0
        p.first_index, p.group, p.t0 = int(first_index), int(group), float(t0)
        g = SeedGridS(int(nd), int(nT), int(nZ), float(z_lim))
        ions.meta["use_w0"] = True
        s = ions.struct()
        self._chk(_lib.taiga_seed_beam_grid(self.h, C.byref(p), C.byref(g), C.byref(s)))

    @staticmethod
    def _det(det):
        keep = [_host(a) for a in (det.u_lo, det.u_hi, det.w_lo, det.w_hi)]
        d = DetS(D3(*det.origin), D3(*det.normal), D3(*det.eu), D3(*det.ew), len(keep[0]), len(keep[2]),
                 *[k.ctypes.data for k in keep])
        return d, keep

    def trace(self, ions, q_over_m, dt, max_steps, det, rkn_variant=0):
        d, keep = self._det(det)
        s = ions.struct()
        self._chk(_lib.taiga_trace(self.h, C.byref(s), q_over_m, dt, int(max_steps), C.byref(d),
                                   int(rkn_variant)))

    def load_loss(self, psi_nodal, psi0=0.0, dpsi=1.0, ne=None, Te=None, E12=1.0):
        """psi_nodal: [nR][nZ] numpy (host) or CUDA tensor, or None to unload; ne / Te: host arrays."""
        if psi_nodal is None:
            self._chk(_lib.taiga_load_loss(self.h, None, 0, None))
            return
        ne, Te = _host(ne), _host(Te)
        assert len(ne) == len(Te)
        prof = LossProfileS(len(ne), float(psi0), float(dpsi), ne.ctypes.data, Te.ctypes.data, float(E12))
        if isinstance(psi_nodal, torch.Tensor):
            assert psi_nodal.is_cuda and psi_nodal.dtype == torch.float64 and psi_nodal.is_contiguous()
            self._chk(_lib.taiga_load_loss(self.h, psi_nodal.data_ptr(), 1, C.byref(prof)))
        else:
            a = _host(psi_nodal)
            self._chk(_lib.taiga_load_loss(self.h, a.ctypes.data, 0, C.byref(prof)))

    def detector_histogram_weighted(self, ions, det, n_hist, wcounts, wsummary, use_loss_weight=True):
        """use_loss_weight=False: weight by ions.w0 only (no loss model traced; with True the library refuses
        weights that the last trace did not write)."""
        d, keep = self._det(det)
        s = ions.struct(weight=use_loss_weight)
        assert wcounts.dtype == torch.int64 and wsummary.dtype == torch.int64
        assert wcounts.numel() == n_hist * d.nu * d.nw and wsummary.numel() == n_hist * 4
        self._chk(_lib.taiga_detector_histogram_weighted(self.h, C.byref(s), C.byref(d), int(n_hist),
                                                         wcounts.data_ptr(), wsummary.data_ptr()))

    def set_efield(self, E):
        self._chk(_lib.taiga_set_efield(self.h, D3(*[float(e) for e in E])))

    def detector_histogram(self, ions, det, n_hist, counts, summary):
        d, keep = self._det(det)
        s = ions.struct()
        assert counts.dtype == torch.int64 and summary.dtype == torch.int64
        assert counts.numel() == n_hist * d.nu * d.nw and summary.numel() == n_hist * 6
        self._chk(_lib.taiga_detector_histogram(self.h, C.byref(s), C.byref(d), int(n_hist),
                                                counts.data_ptr(), summary.data_ptr()))

    def detector_histogram_static(self, ions, det, n_hist, counts, summary):
        """detector_histogram without any allocation inside the library (taiga_detector_histogram_static): for loops that
        must not stall the device's other streams or that run under a memory pool owning the GPU.  The segment edges go to
        a fixed 32 KB array of the library, so det.nu + det.nw <= STATIC_MAX_SEGMENTS (TaigaError otherwise), and calls
        on one device must not overlap on the GPU."""
        d, keep = self._det(det)
        s = ions.struct()
        assert counts.dtype == torch.int64 and summary.dtype == torch.int64
        assert counts.numel() == n_hist * d.nu * d.nw and summary.numel() == n_hist * 6
        self._chk(_lib.taiga_detector_histogram_static(self.h, C.byref(s), C.byref(d), int(n_hist),
                                                       counts.data_ptr(), summary.data_ptr()))

    def set_option(self, key, value):
        self._chk(_lib.taiga_set_option(self.h, key.encode(), int(value)))

    def stats(self):
        out = (C.c_ulonglong * 8)()
        self._chk(_lib.taiga_get_stats(self.h, C.byref(out)))
        return dict(ion_steps=out[0], lane_slots=out[1], passes=out[2], launches=out[3], reloads=out[4])

    def l1_gather_peak(self, ms=50.0, spread=1):
        r = C.c_double()
        self._chk(_lib.taiga_measure_l1_gather_peak(self.h, ms, int(spread), C.byref(r)))
        return r.value

    def fp64_peak(self, ms=50.0):
        r = C.c_double()
        self._chk(_lib.taiga_measure_fp64_peak(self.h, ms, C.byref(r)))
        return r.value

    def dmma_peak(self, ms=50.0):
        r = C.c_double()
        self._chk(_lib.taiga_measure_dmma_peak(self.h, ms, C.byref(r)))
        return r.value

    def mixed_fp64_peak(self, ms=50.0):
        r = C.c_double()
        self._chk(_lib.taiga_measure_mixed_fp64_peak(self.h, ms, C.byref(r)))
        return r.value


def loss_statistics(wsummary):
    """taiga_loss_statistics per histogram: (mean loss, spread of the loss) over the plane-crossing ions, the form of
    PAPER.md Table 1; wsummary[n_hist][4] as written by detector_histogram_weighted (device tensor or host array)."""
    ws = np.ascontiguousarray(wsummary.detach().cpu().numpy() if isinstance(wsummary, torch.Tensor) else wsummary).astype(np.uint64)
    mean, spread = np.empty(len(ws)), np.empty(len(ws))
    for h, row in enumerate(ws):
        out = (C.c_double * 3)()
        rc = _lib.taiga_loss_statistics(C.byref((C.c_ulonglong * 4)(*[int(v) for v in row])), C.byref(out))
        if rc:
            raise TaigaError(rc, "taiga_loss_statistics")
        mean[h], spread[h] = out[0], out[1]
    return mean, spread


def run_config(tg: Taiga, cfg, field_loaded=False, host_field=True, ions=None, rkn_variant=0):
    """Whole hot path (a1-a5) of one workloads.Config through the C ABI.  Returns
    (ions, counts, summary) with counts/summary as device int64 tensors."""
    from . import workloads as wl
    dev = "cuda:%d" % tg.device
    if not field_loaded:
        grid, nodal = cfg.field_builder()
        tg.load_field(grid, nodal if host_field else [torch.from_numpy(c).to(dev) for c in nodal])
    if ions is None:
        ions = Ions(cfg.n_ions, dev)
    det0 = cfg.detector or cfg.groups[0].detector
    counts = torch.zeros((cfg.n_hist, det0.nw, det0.nu), dtype=torch.int64, device=dev)
    summary = torch.zeros((cfg.n_hist, 6), dtype=torch.int64, device=dev)
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    off, spans = 0, []
    for g in cfg.groups:
        v = ions.view(off, off + g.n_ions)
        tg.seed_beam(g.beam, cd, cn, cfg.seed, v, g.first_index, g.group, g.t0)
        spans.append((off, off + g.n_ions, g))
        off += g.n_ions
    if cfg.detector is not None:          # one trace over all groups
        qm = cfg.groups[0].beam.charge_C / cfg.groups[0].beam.mass_kg
        tg.trace(ions, qm, cfg.dt, cfg.max_steps, cfg.detector, rkn_variant)
        tg.detector_histogram(ions, cfg.detector, cfg.n_hist, counts, summary)
    else:                                 # one detector per group (energy scan)
        for lo, hi, g in spans:
            v = ions.view(lo, hi)
            tg.trace(v, g.beam.charge_C / g.beam.mass_kg, cfg.dt, cfg.max_steps, g.detector, rkn_variant)
            tg.detector_histogram(v, g.detector, cfg.n_hist, counts, summary)
    return ions, counts, summary
