"""Seeded, synthetic, COMPASS-shaped inputs for the five BASELINE.json configs.

This module only *generates input data* (nodal field grids, tabulated CDFs, detector
descriptors, beam parameters).  It contains none of the method's arithmetic (no spline fit,
no RNG, no integrator, no binning) and is the one module that both the CUDA path
(``paper_2506_15812_b200.taiga``) and the CPU oracle (``oracle/``) are fed from.

The inputs stand in for the paper's COMPASS workloads (EFIT field of #17178, RENATE-OD
ionisation profile, the real Faraday-cup geometry), none of which are available; shapes and
scales follow PAPER.md: R0=0.56 m, a~0.2 m, B_T~1.15 T, I_p 160-250 kA (L370, L378), Li/Na at
40-100 keV (L147-156, L370-386), 5 mm beam (L179, L370), 1e6 ions (L400), dt~1e-9 s (L284),
ionisation path 7-10 cm (L122).  Recipe and readings: DESIGN.md section 4 and SURVEY.md 8(c,d).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# ---- physical constants (CODATA-2018, atomic mass minus one electron)
E_CHARGE = 1.602176634e-19            # C
AMU = 1.66053906660e-27               # kg
M_ELECTRON_U = 5.48579909065e-4       # u
MASS_LI7 = (7.0160034366 - M_ELECTRON_U) * AMU
MASS_NA23 = (22.9897692820 - M_ELECTRON_U) * AMU
MU0 = 4.0e-7 * math.pi

# ---- Solov'ev equilibrium (A14, A15)
R0, A_MINOR, KAPPA, B_T, I_P = 0.56, 0.2, 1.6, 1.15, 200.0e3
PSI_A = MU0 * I_P * R0 / (4.0 * math.pi * math.sqrt((1.0 + KAPPA**2) / 2.0))

# ---- grid box: spacings 0.625/(n-1) are exact binary fractions
R_MIN, R_MAX, Z_MIN, Z_MAX = 0.25, 0.875, -0.625, 0.625

# ---- beam (configs): entry point, direction, tables
BEAM_ORIGIN = (0.78, 0.0, 0.0)
BEAM_AXIS = (-1.0, 0.0, 0.0)
BEAM_ET = (0.0, 1.0, 0.0)             # toroidal-tangent cross-section axis
BEAM_EZ = (0.0, 0.0, 1.0)             # vertical cross-section axis
DEPTH_LAMBDA, DEPTH_MAX, DEPTH_K = 0.02, 0.20, 2048
NORMAL_ZMAX, NORMAL_K = 6.0, 4096
DETECTOR_X = 0.82


def solovev_psi(R, Z):
    """Poloidal flux of the synthetic equilibrium (A15)."""
    return PSI_A * (((R * R - R0 * R0) / (2.0 * R0 * A_MINOR)) ** 2
                    + (R * Z / (R0 * KAPPA * A_MINOR)) ** 2)


# synthetic plasma profiles for the secondary-ionisation loss (NEXT-1; stand in for the COMPASS
# Thomson profiles of PAPER.md L71-81): n_e, T_e against normalised flux psi_N = psi / PSI_A
E12_LI, E12_NA = 75.6400937, 47.28636          # second ionisation energies [eV]
NE0, TE0 = 6.0e19, 900.0                      # core density [m^-3] and temperature [eV]
LOSS_K, LOSS_PSIN_MAX = 257, 1.6              # profile table: psi_N = 0 .. 1.6


def plasma_profiles(psin):
    """H-mode-like profiles: parabolic core, exponential scrape-off layer beyond psi_N = 1."""
    psin = np.asarray(psin, dtype=np.float64)
    core = np.clip(1.0 - psin, 0.0, 1.0)
    sol = np.exp(-np.clip(psin - 1.0, 0.0, None) / 0.05)
    ne = NE0 * (0.08 * sol + 0.92 * core ** 0.6 * (psin < 1.0))
    te = TE0 * (0.04 * sol + 0.96 * core ** 1.2 * (psin < 1.0))
    return ne, te


def loss_profile_inputs():
    """(psi0, dpsi, n_e[k], T_e[k]) tabulated on psi = psi0 + k dpsi, k < LOSS_K."""
    psin = np.linspace(0.0, LOSS_PSIN_MAX, LOSS_K)
    ne, te = plasma_profiles(psin)
    return 0.0, PSI_A * LOSS_PSIN_MAX / (LOSS_K - 1), ne, te


def nodal_psi(grid):
    """Nodal poloidal flux [Wb/rad] on a grid's (R, Z) nodes."""
    R = np.linspace(grid.Rmin, grid.Rmax, grid.nR)[:, None]
    Z = np.linspace(grid.Zmin, grid.Zmax, grid.nZ)[None, :]
    return np.ascontiguousarray(solovev_psi(R, Z + 0.0 * R))


def solovev_B(R, Z):
    """(B_R, B_Z, B_phi) of the synthetic equilibrium at arrays R, Z (A14, A15)."""
    R = np.asarray(R, dtype=np.float64)
    Z = np.asarray(Z, dtype=np.float64)
    BR = -2.0 * PSI_A * R * Z / (R0 * KAPPA * A_MINOR) ** 2
    BZ = PSI_A * ((R * R - R0 * R0) / (R0 * A_MINOR) ** 2
                  + 2.0 * Z * Z / (R0 * KAPPA * A_MINOR) ** 2)
    Bphi = -B_T * R0 / R + 0.0 * Z
    return BR, BZ, Bphi


@dataclass
class Grid:
    kind: int                      # 0 (R,Z); 1 (R,Z,t); 2 (R,Z,phi) periodic
    nR: int
    nZ: int
    nS: int = 1
    Rmin: float = R_MIN
    Rmax: float = R_MAX
    Zmin: float = Z_MIN
    Zmax: float = Z_MAX
    s0: float = 0.0
    ds: float = 1.0

    def axes(self):
        R = self.Rmin + (self.Rmax - self.Rmin) * (np.arange(self.nR) / (self.nR - 1))
        Z = self.Zmin + (self.Zmax - self.Zmin) * (np.arange(self.nZ) / (self.nZ - 1))
        return R, Z


def nodal_field_2d(nR, nZ):
    """Nodal (BR, BZ, Bphi), each [1][nR][nZ], of the static axisymmetric field."""
    g = Grid(0, nR, nZ, 1)
    R, Z = g.axes()
    RR, ZZ = np.meshgrid(R, Z, indexing="ij")
    BR, BZ, Bp = solovev_B(RR, ZZ)
    return g, tuple(np.ascontiguousarray(b[None]) for b in (BR, BZ, Bp))


def nodal_field_time_slices(nR=129, nZ=257, nS=64, dt_slice=1.0e-6, amp=1.0e-3,
                            m=3, period=16.0e-6):
    """Config 4: B_pol*(1+amp*cos(m*theta - 2 pi t/period)), theta=atan2(Z,R-R0); B_phi
    unperturbed; nS slices dt_slice apart (SURVEY.md 8(d) cfg 4, A16)."""
    g = Grid(1, nR, nZ, nS, s0=0.0, ds=dt_slice)
    R, Z = g.axes()
    RR, ZZ = np.meshgrid(R, Z, indexing="ij")
    BR0, BZ0, Bp0 = solovev_B(RR, ZZ)
    theta = np.arctan2(ZZ, RR - R0)
    BR = np.empty((nS, nR, nZ))
    BZ = np.empty((nS, nR, nZ))
    Bp = np.empty((nS, nR, nZ))
    for k in range(nS):
        f = 1.0 + amp * np.cos(m * theta - 2.0 * math.pi * (k * dt_slice) / period)
        BR[k], BZ[k], Bp[k] = BR0 * f, BZ0 * f, Bp0
    return g, (BR, BZ, Bp)


def nodal_field_ripple(nR=129, nZ=257, nS=32, ncoil=16, amp=0.01, Rc=0.82):
    """Config 5: Solov'ev + vacuum ripple dB_R=d0 (R/Rc)^(n-1) sin(n phi),
    dB_phi=d0 (R/Rc)^(n-1) cos(n phi), d0=amp*B_T*R0/Rc, on nS planes spanning ONE ripple
    period 2 pi/ncoil, periodic (A17)."""
    dphi = 2.0 * math.pi / ncoil / nS
    g = Grid(2, nR, nZ, nS, s0=0.0, ds=dphi)
    R, Z = g.axes()
    RR, ZZ = np.meshgrid(R, Z, indexing="ij")
    BR0, BZ0, Bp0 = solovev_B(RR, ZZ)
    d0 = amp * B_T * R0 / Rc
    rad = d0 * (RR / Rc) ** (ncoil - 1)
    BR = np.empty((nS, nR, nZ))
    BZ = np.empty((nS, nR, nZ))
    Bp = np.empty((nS, nR, nZ))
    for k in range(nS):
        phi = k * dphi
        BR[k] = BR0 + rad * math.sin(ncoil * phi)
        BZ[k] = BZ0
        Bp[k] = Bp0 + rad * math.cos(ncoil * phi)
    return g, (BR, BZ, Bp)


def depth_cdf(lam=DEPTH_LAMBDA, dmax=DEPTH_MAX, K=DEPTH_K):
    """Attenuation CDF of a truncated exponential on a uniform depth grid: F_0=0, F_K=1."""
    d = dmax * (np.arange(K + 1) / K)
    F = -np.expm1(-d / lam) / -math.expm1(-dmax / lam)
    F[0], F[-1] = 0.0, 1.0
    return np.ascontiguousarray(F)


def normal_cdf(zmax=NORMAL_ZMAX, K=NORMAL_K):
    """Standard-normal CDF on a uniform grid over [-zmax, zmax], renormalised to [0,1]."""
    z = -zmax + 2.0 * zmax * (np.arange(K + 1) / K)
    phi = np.array([0.5 * math.erfc(-zz / math.sqrt(2.0)) for zz in z])
    F = (phi - phi[0]) / (phi[-1] - phi[0])
    F[0], F[-1] = 0.0, 1.0
    return np.ascontiguousarray(F)


@dataclass
class Beam:
    mass_kg: float
    charge_C: float
    energy_eV: float
    sigma_pos_m: float = 5.0e-3
    sigma_ang_rad: float = 0.0
    origin: tuple = BEAM_ORIGIN
    axis: tuple = BEAM_AXIS
    eT: tuple = BEAM_ET
    eZ: tuple = BEAM_EZ
    depth_max: float = DEPTH_MAX
    z_max: float = NORMAL_ZMAX
    profile: int = 0               # cross-section: 0 = Gaussian sigma_pos_m, 1 = uniform disc of radius_m
    radius_m: float = 2.5e-3


@dataclass
class Detector:
    """Plane + perpendicular grid of segments; u along eu, w along ew,
    both measured from `origin` (the matrix centre)."""
    origin: tuple
    normal: tuple
    eu: tuple
    ew: tuple
    u_lo: np.ndarray
    u_hi: np.ndarray
    w_lo: np.ndarray
    w_hi: np.ndarray

    @property
    def nu(self):
        return len(self.u_lo)

    @property
    def nw(self):
        return len(self.w_lo)


def uniform_detector(centre_T, centre_Z, n, pitch, x_plane=DETECTOR_X):
    """n x n segments of `pitch`, zero gaps, centred on (T, Z) in the plane X=x_plane
    (A9, A11, A18).  hi[k] is bit-identical to lo[k+1]."""
    edges = (np.arange(n + 1) - n / 2.0) * pitch
    lo, hi = np.ascontiguousarray(edges[:-1]), np.ascontiguousarray(edges[1:])
    return Detector((x_plane, centre_T, centre_Z), (1.0, 0.0, 0.0), (0.0, 1.0, 0.0),
                    (0.0, 0.0, 1.0), lo, hi, lo.copy(), hi.copy())


def gapped_detector(det: Detector, gap_frac: float = 0.15, jitter: float = 0.3, seed: int = 7) -> Detector:
    """The same plane and centre as `det`, its segments made non-uniform with gaps ("optional
    non-uniform size and gaps"): every segment keeps its centre, its width is the pitch times (1 - gap_frac) times a
    seeded factor in [1 - jitter, 1]; segments stay ordered and disjoint.  Takes the binary-search path of a5."""
    rng = np.random.default_rng(seed)

    def axis(lo, hi):
        c, wid = 0.5 * (lo + hi), (hi - lo) * (1.0 - gap_frac) * (1.0 - jitter * rng.random(len(lo)))
        return np.ascontiguousarray(c - 0.5 * wid), np.ascontiguousarray(c + 0.5 * wid)

    ul, uh = axis(det.u_lo, det.u_hi)
    wl_, wh = axis(det.w_lo, det.w_hi)
    return Detector(det.origin, det.normal, det.eu, det.ew, ul, uh, wl_, wh)


@dataclass
class Group:
    """One seeding call: a contiguous run of ions sharing beam, group id, birth time and
    (for the energy scan) detector."""
    beam: Beam
    n_ions: int
    first_index: int          # Philox counter of the first ion (global ion index)
    group: int = 0
    t0: float = 0.0
    detector: Detector | None = None


@dataclass
class Config:
    name: str
    field_builder: object      # () -> (Grid, (BR,BZ,Bphi))
    groups: list
    dt: float
    max_steps: int
    seed: int
    n_hist: int
    detector: Detector | None = None     # shared detector (None when per-group)
    note: str = ""

    @property
    def n_ions(self):
        return sum(g.n_ions for g in self.groups)


# Detector centres (T, Z) [m]: frozen from an oracle pilot run (A10): component-wise median
# (u, w) of plane-crossing ions, rounded to 0.1 mm.  Written by oracle/freeze_detector_centres.py
# (which calls only oracle/); never changed afterwards.
DETECTOR_CENTRES = {
    "cfg1": (0.0205, 0.1812),
    "cfg2": (0.0203, 0.1811),
    "cfg3_20keV": (0.0134, 0.0953),
    "cfg3_40keV": (0.0178, 0.1453),
    "cfg3_60keV": (0.0204, 0.1811),
    "cfg3_80keV": (0.0217, 0.2095),
    "cfg4": (0.0228, 0.2652),
    "cfg5": (0.0203, 0.1811),
}


def _li(energy, **kw):
    return Beam(MASS_LI7, E_CHARGE, energy, **kw)


def config(i: int, n_override: int | None = None) -> Config:
    """BASELINE.json configs[i-1] (1-based).  `n_override` gives the
    ion count per group for prefix-subsample parity runs (identical ions: the Philox counter is
    the global ion index)."""
    if i == 1:
        n = n_override or 4096
        det = uniform_detector(*DETECTOR_CENTRES["cfg1"], 8, 2.5e-3)
        return Config("cfg1", lambda: nodal_field_2d(65, 129), [Group(_li(60e3), n, 0)],
                      1e-9, 5000, 0, 1, det)
    if i == 2:
        n = n_override or 1048576
        det = uniform_detector(*DETECTOR_CENTRES["cfg2"], 32, 1e-3)
        return Config("cfg2", lambda: nodal_field_2d(257, 513), [Group(_li(60e3), n, 0)],
                      5e-10, 20000, 1, 1, det)
    if i == 3:
        n = n_override or 4194304
        groups = []
        for g, e in enumerate((20e3, 40e3, 60e3, 80e3)):
            det = uniform_detector(*DETECTOR_CENTRES["cfg3_%dkeV" % int(e / 1e3)], 32, 1e-3)
            groups.append(Group(_li(e, sigma_ang_rad=2e-3), n, g * 4194304, g, 0.0, det))
        return Config("cfg3", lambda: nodal_field_2d(257, 513), groups, 5e-10, 20000, 2, 4,
                      None, "energy scan, one detector per energy")
    if i == 4:
        n_total = 2097152
        per = n_total // 64
        n = n_override or per
        det = uniform_detector(*DETECTOR_CENTRES["cfg4"], 32, 1e-3)
        beam = Beam(MASS_NA23, E_CHARGE, 40e3)
        groups = [Group(beam, n, g * per, g, g * 1.0e-6) for g in range(64)]
        return Config("cfg4", nodal_field_time_slices, groups, 1e-9, 20000, 3, 64, det,
                      "64 time slices, histogram per birth slice (A16)")
    if i == 5:
        n = n_override or 67108864
        det = uniform_detector(*DETECTOR_CENTRES["cfg5"], 64, 0.5e-3)
        return Config("cfg5", nodal_field_ripple, [Group(_li(60e3), n, 0)], 5e-10, 40000, 4,
                      1, det, "3-D ripple field, tricubic")
    raise ValueError("config index must be 1..5")
