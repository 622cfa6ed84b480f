"""GPU-vs-oracle parity through the C ABI (run on the B200 box: -m gpu).

Acceptance (BASELINE.json north_star): initial conditions bit-exact; cell / status / steps /
histograms bit-exact excluding ions flagged (by either side) as grazing within 1e-9 m;
(u, w) within 1e-9 m."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import oracle as orc  # noqa: E402
from paper_2506_15812_b200 import workloads as wl  # noqa: E402

TOL_UW = 1e-9


@pytest.fixture
def tg():
    """A fresh context per test: every test starts from the library defaults (the launch configuration
    bench.py times); options a test sets never leak into the next one."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2506_15812_b200 import taiga
    t = taiga.Taiga(0)
    yield t
    t.close()


def _np(t):
    return t.detach().cpu().numpy()


def compare_groups(ions, ref, label=""):
    """Element-by-element comparison of a run_config result with the oracle's."""
    off = 0
    stats = dict(n=0, flagged=0, max_du=0.0, max_dw=0.0)
    for g in ref["groups"]:
        n = len(g["status"])
        v = ions.view(off, off + n)
        for k, a in zip(("x", "y", "z", "vx", "vy", "vz"), g["state0"]):
            assert np.array_equal(_np(v.a[k]), a), "%s: seeding not bit-exact (%s)" % (label, k)
        assert np.array_equal(_np(v.group).astype(np.uint16), g["group"])
        fl = (_np(v.flags) | g["flags"]) != 0
        ok = ~fl
        cell, steps = _np(v.cell), _np(v.steps).astype(np.uint32)
        bad = ok & ((cell != g["cell"]) | (steps != g["steps"]))
        assert not bad.any(), "%s: %d unflagged ions differ, first %s: gpu cell/steps %s/%s oracle %s/%s" % (
            label, bad.sum(), np.flatnonzero(bad)[:5], cell[bad][:5], steps[bad][:5], g["cell"][bad][:5], g["steps"][bad][:5])
        cr = ok & (g["status"] == 0)
        if cr.any():
            du = np.abs(_np(v.hit_u)[cr] - g["u"][cr]).max()
            dw = np.abs(_np(v.hit_w)[cr] - g["w"][cr]).max()
            assert du < TOL_UW and dw < TOL_UW, (label, du, dw)
            stats["max_du"], stats["max_dw"] = max(stats["max_du"], du), max(stats["max_dw"], dw)
        stats["n"] += n
        stats["flagged"] += int(fl.sum())
        off += n
    return stats


def check_histogram(cfg, ions, counts, summary, ref):
    """Histograms bit-exact after removing the flagged ions from both sides."""
    c_gpu = _np(counts).astype(np.int64).copy()
    c_ref = ref["counts"].astype(np.int64).copy()
    off = 0
    for g in ref["groups"]:
        n = len(g["status"])
        v = ions.view(off, off + n)
        fl = (_np(v.flags) | g["flags"]) != 0
        det = None
        for i in np.flatnonzero(fl):
            gi = int(g["group"][i])
            cg, cr = int(_np(v.cell)[i]), int(g["cell"][i])
            if cg >= 0:
                c_gpu[gi].reshape(-1)[cg] -= 1
            if cr >= 0:
                c_ref[gi].reshape(-1)[cr] -= 1
        off += n
    assert np.array_equal(c_gpu, c_ref)
    s = _np(summary)
    for h in range(cfg.n_hist):
        n_h = sum(int(np.sum(g["group"] == h)) for g in ref["groups"])
        assert s[h, 0] == _np(counts)[h].sum()
        assert s[h, :5].sum() == n_h                       # O5 invariant


@pytest.mark.parametrize("opts", [dict(), dict(sort=0), dict(variant=1), dict(min_active=1), dict(min_active=12), dict(variant=4), dict(variant=5)])
def test_cfg1_full_parity(tg, opts):
    """dict() = the library defaults (sort=1, variant=0, min_active=32: whole-tile refill), the others are the
    alternative launch options of taiga_set_option."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(1)
    for k, v in opts.items():
        tg.set_option(k, v)
    ions, counts, summary = taiga.run_config(tg, cfg)
    torch.cuda.synchronize()
    ref = orc.run_config(cfg)
    st = compare_groups(ions, ref, "cfg1 %s" % opts)
    check_histogram(cfg, ions, counts, summary, ref)
    assert st["flagged"] < 20


def test_cfg1_printed_k3_variant(tg):
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(1)
    ions, counts, summary = taiga.run_config(tg, cfg, rkn_variant=1)
    torch.cuda.synchronize()
    ref = orc.run_config(cfg, variant=1)
    compare_groups(ions, ref, "cfg1 k3-from-k2")
    ref0 = orc.run_config(cfg, variant=0)
    cr = (ref0["groups"][0]["status"] == 0) & (ref["groups"][0]["status"] == 0)
    # the two readings differ by more than the tolerance (A1): the switch is live
    assert np.abs(ref0["groups"][0]["u"][cr] - ref["groups"][0]["u"][cr]).max() > 5e-10


@pytest.mark.parametrize("icfg,n", [(2, 16384), (3, 4096), (4, 256), (5, 4096)])
def test_prefix_parity(tg, icfg, n):
    """Prefix subsamples of configs 2-5: identical ions (Philox counter = global ion index),
    sizes spanning many warps plus a ragged tail (n is per group)."""
    from paper_2506_15812_b200 import taiga
    n = n + 37 if icfg in (2, 5) else n
    cfg = wl.config(icfg, n_override=n)
    ions, counts, summary = taiga.run_config(tg, cfg)
    torch.cuda.synchronize()
    ref = orc.run_config(cfg)
    st = compare_groups(ions, ref, cfg.name)
    check_histogram(cfg, ions, counts, summary, ref)
    assert st["flagged"] <= max(8, st["n"] // 500)
    ngpu = int(_np(ions.steps).astype(np.int64).sum())
    assert tg.stats()["launches"] >= 1
    assert ngpu > 0


@pytest.mark.parametrize("icfg,n,opts", [
    (4, 96, dict(variant=6)),                      # kind 1: blended cache, slice difference gathered through L1 (r2a)
    (4, 96, dict(variant=4)),                      # kind 1: slice cache with rolling refill (r1e)
    (4, 96, dict(variant=1)),                      # kind 1: no cache
    (4, 96, dict(mma=1)),                          # kind 1 on the DMMA tracer
    (4, 96, dict(sort=0)),                         # queue in ion-index order (slices interleaved per tile boundary)
    (5, 4096 + 5, dict(mma=0)),                    # kind 2: per-lane gathers with the CTA re-sort (r1e)
    (5, 4096 + 5, dict(mma=0, regroup=0)),         # ... per-warp tiles
    (5, 4096 + 5, dict(mma_geom=1)), (5, 4096 + 5, dict(mma_geom=2)), (5, 4096 + 5, dict(mma_geom=3)),
    (5, 4096 + 5, dict(mma_geom=5)),
    (5, 4096 + 5, dict(refill_cta=16, regroup=3)), (5, 4096 + 5, dict(sort=0)),
])
def test_kernel_options_of_the_sliced_fields(tg, icfg, n, opts):
    """Every kernel variant and launch geometry `taiga_set_option` offers for the time-sliced and (R, Z, phi) tables
    gives the oracle's result (the defaults are covered by the prefix and full-histogram tests)."""
    from paper_2506_15812_b200 import taiga
    for k, v in opts.items():
        tg.set_option(k, v)
    cfg = wl.config(icfg, n_override=n)
    ions, counts, summary = taiga.run_config(tg, cfg)
    torch.cuda.synchronize()
    ref = orc.run_config(cfg)
    st = compare_groups(ions, ref, "%s %s" % (cfg.name, opts))
    check_histogram(cfg, ions, counts, summary, ref)
    assert st["flagged"] <= 8, st


@pytest.mark.parametrize("nS,ncoil", [(16, 1), (32, 1), (32, 4), (32, 8)])
@pytest.mark.parametrize("mma", [1, 0])
def test_coarse_toroidal_planes_parity(tg, nS, ncoil, mma):
    """(R, Z, phi) tables whose planes are far apart: 16 and 32 planes round the whole torus (ds = 0.39, 0.20), 0.049 just
    above and 0.0245 below the spacing up to which the cooperative tracer's asin series is exact to rounding
    (TG_MMA_MAX_DS = 0.04: coarser tables take the atan2 path whatever "mma" says).  Same 1e-9 m bar on every one."""
    from paper_2506_15812_b200 import taiga
    tg.set_option("mma", mma)
    cfg = wl.config(5, n_override=2048 + 5)
    cfg.field_builder = lambda: wl.nodal_field_ripple(65, 129, nS, ncoil)
    ions, counts, summary = taiga.run_config(tg, cfg)
    torch.cuda.synchronize()
    ref = orc.run_config(cfg)
    st = compare_groups(ions, ref, "kind 2, %d planes x %d periods, mma=%d" % (nS, ncoil, mma))
    check_histogram(cfg, ions, counts, summary, ref)
    assert st["flagged"] <= 8 and int(summary[0, 0]) > 1000


def test_roofline_denominators_are_consistent(tg):
    """The microkernels behind bench.py's roofline: the DFMA and DMMA issue rates are within 3 % of 148 x 64 FMA per clock
    at the clock nvidia-smi reports as maximum (never above it), and interleaving both does not exceed either (one FP64 datapath)."""
    import subprocess
    mhz = float(subprocess.run(["nvidia-smi", "-i", "0", "--query-gpu=clocks.max.sm", "--format=csv,noheader,nounits"],
                               capture_output=True, text=True).stdout.strip().splitlines()[0])
    sm = torch.cuda.get_device_properties(0).multi_processor_count
    nominal = sm * 64 * mhz * 1e6
    dfma, dmma, mixed = tg.fp64_peak(30.0), tg.dmma_peak(30.0), tg.mixed_fp64_peak(30.0)
    # lower bounds loose: a power- or thermally capped clock lowers the rates without making them wrong
    assert 0.60 * nominal < dfma < 1.03 * nominal, (dfma, nominal)
    assert 0.60 * nominal < dmma < 1.03 * nominal, (dmma, nominal)
    assert 0.5 * dfma < mixed < 1.03 * max(dfma, dmma), (mixed, dfma, dmma)


@pytest.mark.parametrize("icfg,n", [(2, None), (3, 262144 + 21), (4, 2048 + 3), (4, None), (5, 1048576 + 77)])
def test_full_histogram_parity(tg, icfg, n):
    """The method's output is the counters.  COMPLETE detector histograms + summary, bit for bit
    (ions flagged as grazing by either side removed from both), and cell / steps / (u, w) of EVERY ion, in the launch
    configuration bench.py times (library defaults): configs 2 and 4 in full (1,048,576 and 2,097,152 ions: the oracle needs
    20 and 40 s on 16 threads), configs 3 / 4 / 5 on prefixes of 65,557 ions per energy, 2,051 per time slice (131,264 ions
    over all 64 slices) and 65,613 ions: multi-tile
    queues, ragged tails, the CTA refill / re-sort of the cooperative kernel all active."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(icfg, n_override=n)
    ions, counts, summary = taiga.run_config(tg, cfg)
    torch.cuda.synchronize()
    if cfg.detector is not None:                   # one trace over all groups: its counters cover every ion
        assert tg.stats()["ion_steps"] == int(ions.steps.to(torch.int64).sum().item())
    ref = orc.run_config(cfg)
    st = compare_groups(ions, ref, cfg.name + " full histogram")
    check_histogram(cfg, ions, counts, summary, ref)
    assert st["flagged"] <= max(8, st["n"] // 2000), st
    assert np.array_equal(_np(summary)[:, :5].sum(axis=1), [sum(g.n_ions for g in cfg.groups if g.group == h) for h in range(cfg.n_hist)])


def test_seeding_bit_exact_large_indices_and_divergence(tg):
    from paper_2506_15812_b200 import taiga
    beam = wl.Beam(wl.MASS_NA23, wl.E_CHARGE, 40e3, sigma_pos_m=7e-3, sigma_ang_rad=3e-3,
                   origin=(0.8, 0.01, -0.02), axis=(-0.6, 0.0, 0.8), eT=(0.0, 1.0, 0.0), eZ=(0.8, 0.0, 0.6))
    cd, cn = wl.depth_cdf(0.035, 0.15, 777), wl.normal_cdf(5.0, 1000)
    beam.depth_max, beam.z_max = 0.15, 5.0
    for first, seed, n in ((0, 0, 1), ((1 << 40) + 12345, 0xDEADBEEFCAFEF00D, 10007), (2 ** 32 - 5, 7, 64)):
        ions = taiga.Ions(n)
        tg.seed_beam(beam, cd, cn, seed, ions, first_index=first, group=3, t0=2.5e-6)
        torch.cuda.synchronize()
        ref = orc.seed(beam, cd, cn, seed, first, n)
        for k, a in zip(("x", "y", "z", "vx", "vy", "vz"), ref):
            assert np.array_equal(_np(ions.a[k]), a), (k, first)
        assert np.all(_np(ions.group) == 3) and np.all(_np(ions.t0) == 2.5e-6)


def test_disc_beam_profile_bit_exact(tg):
    """Uniform-disc cross-section (PAPER.md: "5 mm diameter"; reading A7'): bit-exact against the oracle at
    indices beyond 2^32, with divergence and a tilted frame, retries included; then the whole path on config 1."""
    import dataclasses
    from paper_2506_15812_b200 import taiga
    beam = wl.Beam(wl.MASS_LI7, wl.E_CHARGE, 60e3, sigma_ang_rad=3e-3, origin=(0.8, 0.01, -0.02), axis=(-0.6, 0.0, 0.8),
                   eT=(0.0, 1.0, 0.0), eZ=(0.8, 0.0, 0.6), profile=1, radius_m=2.5e-3)
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    for first, seed, n in ((0, 0, 1), ((1 << 40) + 999, 0xDEADBEEFCAFEF00D, 100003), (2 ** 32 - 7, 11, 257)):
        ions = taiga.Ions(n)
        tg.seed_beam(beam, cd, cn, seed, ions, first_index=first)
        torch.cuda.synchronize()
        ref = orc.seed(beam, cd, cn, seed, first, n)
        for k, a in zip(("x", "y", "z", "vx", "vy", "vz"), ref):
            assert np.array_equal(_np(ions.a[k]), a), (k, first)
    with pytest.raises(taiga.TaigaError):
        tg.seed_beam(dataclasses.replace(beam, radius_m=0.0), cd, cn, 0, taiga.Ions(4))
    with pytest.raises(taiga.TaigaError):
        tg.seed_beam(dataclasses.replace(beam, profile=7), cd, cn, 0, taiga.Ions(4))
    cfg = wl.config(1)
    cfg.groups[0].beam = dataclasses.replace(cfg.groups[0].beam, profile=1, radius_m=2.5e-3)
    ions, counts, summary = taiga.run_config(tg, cfg)
    torch.cuda.synchronize()
    ref = orc.run_config(cfg)
    compare_groups(ions, ref, "cfg1 disc beam")
    check_histogram(cfg, ions, counts, summary, ref)
    y, z = _np(ions.a["y"]), _np(ions.a["z"])
    assert np.hypot(y, z).max() <= 2.5e-3


def test_time_dependent_field_against_an_independent_ode_solution(tg):
    """Reading A3 through the product path (both tracers of kind-1 fields): two slices of uniform B_Z give a field
    exactly linear in t, whose equations of motion scipy's DOP853 integrates to 1e-13; wrong stage times or a
    frozen t move the hit by ~1e-4 m (tests/test_oracle_pins7.py has the same pin for the oracle)."""
    from scipy.integrate import solve_ivp
    from paper_2506_15812_b200 import taiga
    B0, B1, DS = 1.0, 2.0, 1e-6
    qm = wl.E_CHARGE / wl.MASS_LI7
    v0 = math.sqrt(2 * 60e3 * qm)
    grid, nodal = wl.nodal_field_time_slices(9, 17, 2)
    grid.s0, grid.ds = 0.0, DS
    nod = [np.zeros_like(nodal[0]) for _ in range(3)]
    nod[1][0], nod[1][1] = B0, B1
    det = wl.Detector((0.50, 0.0, 0.0), (-1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0),
                      np.array([-1.0]), np.array([1.0]), np.array([-1.0]), np.array([1.0]))
    t0s = np.array([0.0, 1.0e-7, 3.0e-7] * 43)
    n = len(t0s)
    tg.load_field(grid, nod)
    for mma in (1, 0):
        tg.set_option("mma", mma)
        ions = taiga.Ions(n)
        for k, val in (("x", 0.55), ("y", 0.0), ("z", 0.0), ("vx", v0), ("vy", 0.0), ("vz", 3.0e4)):
            ions.a[k].fill_(val)
        ions.a["t0"].copy_(torch.from_numpy(t0s))
        dt = 2.5e-10
        tg.trace(ions, qm, dt, 20000, det)
        torch.cuda.synchronize()
        assert np.all(_np(ions.cell) == -1)                       # crossed the plane (segment assigned by a5)
        for i in range(3):
            def rhs(t, y):
                bz = B0 + (B1 - B0) * t / DS
                return [y[3], y[4], y[5], qm * y[4] * bz, -qm * y[3] * bz, 0.0]
            ev = lambda t, y: 0.50 - y[0]
            ev.terminal, ev.direction = True, 1.0
            sol = solve_ivp(rhs, (t0s[i], t0s[i] + 2e-6), [0.55, 0.0, 0.0, v0, 0.0, 3.0e4], method="DOP853",
                            rtol=1e-13, atol=1e-16, events=ev)
            ye = sol.y_events[0][0]
            sel = np.arange(i, n, 3)
            assert np.all(_np(ions.steps)[sel] == math.ceil((sol.t_events[0][0] - t0s[i]) / dt - 1e-9))
            assert np.abs(_np(ions.hit_u)[sel] - ye[1]).max() < 5e-7 and np.abs(_np(ions.hit_w)[sel] - ye[2]).max() < 5e-7


@pytest.mark.parametrize("kind", [0, 1, 2])
def test_field_precompute_vs_oracle_tables(tg, kind):
    if kind == 0:
        grid, nodal = wl.nodal_field_2d(33, 65)
    elif kind == 1:
        grid, nodal = wl.nodal_field_time_slices(17, 33, 5)
    else:
        grid, nodal = wl.nodal_field_ripple(17, 33, 8)
    rng = np.random.default_rng(kind)
    nodal = [c + 1e-3 * rng.standard_normal(c.shape) for c in nodal]      # not a polynomial
    f = orc.OracleField(grid, nodal)
    for host in (True, False):
        tg.load_field(grid, nodal if host else [torch.from_numpy(np.ascontiguousarray(c)).cuda() for c in nodal])
        for comp in range(3):
            tab = tg.field_table(comp, f.tables[comp].shape)
            scale = np.abs(f.tables[comp]).max()
            assert np.abs(tab - f.tables[comp]).max() < 2e-13 * max(scale, 1.0), (kind, comp)
    # evaluation at random points, inside and outside (extrapolation) the grid
    n = 4000
    R = rng.uniform(grid.Rmin - 0.01, grid.Rmax + 0.01, n)
    Z = rng.uniform(grid.Zmin - 0.01, grid.Zmax + 0.01, n)
    s = rng.uniform(-2 * grid.ds, (grid.nS + 2) * grid.ds, n)
    out = tg.field_eval(torch.from_numpy(R).cuda(), torch.from_numpy(Z).cuda(), torch.from_numpy(s).cuda())
    out = [_np(o) for o in out]
    for i in range(0, n, 7):
        b = f.cyl(R[i], Z[i], s[i])
        for c in range(3):
            assert abs(out[c][i] - b[c]) < 1e-12, (kind, i, c)
    # form 1: ready coefficients (the paper's "read from the preprocessing database" mode)
    tg.load_field(grid, f.tables, form=1)
    out1 = [_np(o) for o in tg.field_eval(torch.from_numpy(R).cuda(), torch.from_numpy(Z).cuda(), torch.from_numpy(s).cuda())]
    for c in range(3):
        assert np.abs(out1[c] - out[c]).max() < 1e-12


def test_periodic_spline_at_the_plane_limit(tg):
    """128 toroidal planes, the most taiga_load_field takes for a kind-2 table (129 are refused with a message): the closed-form
    circulant inverse against the oracle's dense cyclic elimination, every plane including the seam 127 -> 0."""
    from paper_2506_15812_b200 import taiga
    grid, nodal = wl.nodal_field_ripple(5, 6, 128, ncoil=1)
    rng = np.random.default_rng(5)
    nodal = [c + 1e-3 * rng.standard_normal(c.shape) for c in nodal]
    f = orc.OracleField(grid, nodal)
    tg.load_field(grid, nodal)
    for comp in range(3):
        tab = tg.field_table(comp, f.tables[comp].shape)
        err = np.abs(tab - f.tables[comp]).reshape(128, -1).max(axis=1)
        assert err.max() < 2e-13 * max(np.abs(f.tables[comp]).max(), 1.0), (comp, int(err.argmax()), err.max())
    with pytest.raises(taiga.TaigaError) as e:
        tg.load_field(*wl.nodal_field_ripple(5, 6, 129, ncoil=1))
    assert e.value.code == taiga.E_ARG and "128" in str(e.value)


@pytest.mark.parametrize("n_hist,nu,nw", [(3, 4, 3), (40, 16, 16)])
def test_histogram_vs_oracle_gapped_detector(tg, n_hist, nu, nw):
    from paper_2506_15812_b200 import taiga
    rng = np.random.default_rng(11)
    n = 100003
    eu = np.sort(rng.uniform(-5e-3, 5e-3, 2 * nu))
    ew = np.sort(rng.uniform(-5e-3, 5e-3, 2 * nw))
    det = wl.Detector((0.82, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), eu[0::2].copy(), eu[1::2].copy(),
                      ew[0::2].copy(), ew[1::2].copy())
    status = rng.choice([-1, -1, -1, -2, -3, -4], n).astype(np.int32)
    u = rng.uniform(-6e-3, 6e-3, n)
    w = rng.uniform(-6e-3, 6e-3, n)
    u[:nu] = det.u_lo                     # exactly on edges
    u[nu:2 * nu] = det.u_hi
    status[:2 * nu] = -1
    grp = rng.integers(0, n_hist + 1, n).astype(np.uint16)      # some out-of-range groups: skipped
    ions = taiga.Ions(n)
    ions.a["cell"].copy_(torch.from_numpy(status))
    ions.a["hit_u"].copy_(torch.from_numpy(u))
    ions.a["hit_w"].copy_(torch.from_numpy(w))
    ions.a["group"].copy_(torch.from_numpy(grp.astype(np.int16)))
    counts = torch.zeros((n_hist, nw, nu), dtype=torch.int64, device="cuda")
    summary = torch.zeros((n_hist, 6), dtype=torch.int64, device="cuda")
    tg.detector_histogram(ions, det, n_hist, counts, summary)
    torch.cuda.synchronize()
    res = dict(status=np.where(status == -1, 0, status).astype(np.int32), u=u, w=w, flags=np.zeros(n, np.uint8))
    c_ref, s_ref = orc.histogram(res, grp, det, n_hist)
    assert np.array_equal(_np(counts).astype(np.uint64), c_ref)
    assert np.array_equal(_np(summary).astype(np.uint64), s_ref)
    valid = grp < n_hist
    assert np.array_equal(_np(ions.cell)[valid], res["cell"][valid])
    assert np.array_equal(_np(ions.flags)[valid], res["flags"][valid])


@pytest.mark.parametrize("n_hist,nu,nw,interleaved", [(3, 8, 8, True), (5, 32, 32, True), (4, 16, 16, False)])
def test_weighted_histogram_vs_oracle_synthetic(tg, n_hist, nu, nw, interleaved):
    """The 32.32 fixed-point weighted counters on synthetic hits: shared-memory (<= 4096 counters) and global counting
    paths, groups interleaved ion by ion (every warp mixed: per-lane summary atomics) and in contiguous runs with borders
    inside warps (warp-reduced summary), some groups out of range, weights incl. 0, negative, NaN and > 2^20 (clamped,
    reading L3').  Integer sums: bit for bit."""
    from paper_2506_15812_b200 import taiga
    rng = np.random.default_rng(n_hist * 100 + nu)
    n = 70001
    det = wl.uniform_detector(0.0, 0.0, nu, 1e-3)
    det.w_lo, det.w_hi = det.w_lo[:nw].copy(), det.w_hi[:nw].copy()
    status = rng.choice([-1, -1, -1, -2, -3, -4], n).astype(np.int32)
    u = rng.uniform(-0.6e-3 * nu, 0.6e-3 * nu, n)
    w = rng.uniform(-0.6e-3 * nu, 0.6e-3 * nu, n)
    grp = rng.integers(0, n_hist + 1, n).astype(np.uint16) if interleaved else np.sort(rng.integers(0, n_hist + 1, n)).astype(np.uint16)
    wt = rng.uniform(0.0, 1.0, n)
    wt[:8] = [0.0, -1.0, np.nan, 2.0 ** 21, 1.0, 2.0 ** -33, 0.5 + 2.0 ** -33, 1048576.0]
    status[:8] = -1
    ions = taiga.Ions(n)
    for k, a in (("cell", status), ("hit_u", u), ("hit_w", w), ("group", grp.astype(np.int16)), ("w0", wt)):
        ions.a[k].copy_(torch.from_numpy(a))
    ions.meta["use_w0"] = True
    counts = torch.zeros((n_hist, nw, nu), dtype=torch.int64, device="cuda")
    summary = torch.zeros((n_hist, 6), dtype=torch.int64, device="cuda")
    wcounts, wsummary = torch.zeros_like(counts), torch.zeros((n_hist, 4), dtype=torch.int64, device="cuda")
    tg.detector_histogram(ions, det, n_hist, counts, summary)
    tg.detector_histogram_weighted(ions, det, n_hist, wcounts, wsummary, use_loss_weight=False)
    torch.cuda.synchronize()
    res = dict(status=np.where(status == -1, 0, status).astype(np.int32), u=u, w=w, flags=np.zeros(n, np.uint8), weight=wt)
    orc.histogram(res, grp, det, n_hist)
    wc_ref, ws_ref = orc.histogram_weighted(res, grp, det, n_hist)
    assert np.array_equal(_np(wcounts).astype(np.uint64), wc_ref)
    assert np.array_equal(_np(wsummary).astype(np.uint64), ws_ref)
    assert ws_ref[:, 3].sum() > 20000 and ws_ref[:, 1].min() > 0


@pytest.mark.parametrize("icfg,n,optsets", [
    (2, 40000 + 3, [dict(), dict(ctas_per_sm=3), dict(ctas_per_sm=16, sort=0)]),
    (4, 512, [dict(), dict(ctas_per_sm=1), dict(sort_sub=4, ctas_per_sm=3)]),
    (5, 16384 + 9, [dict(), dict(regroup=3), dict(regroup=16, ctas_per_sm=2)]),
])
def test_results_do_not_depend_on_the_launch_geometry(icfg, n, optsets):
    """Race / order check that stands in for the sanitizer layer: the same ions traced under
    three launch geometries (CTAs per SM, queue order, re-sort period of the cooperative tracer) land on different lanes,
    warps and shared-memory slots at different times; every output array must come out bit for bit the same, since an
    ion's arithmetic never depends on where it runs.  A lost update or a stale shared-memory slot shows up here."""
    from paper_2506_15812_b200 import taiga
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    cfg = wl.config(icfg, n_override=n)
    base = None
    for opts in optsets:
        t = taiga.Taiga(0)
        try:
            for k, v in opts.items():
                t.set_option(k, v)
            ions, counts, summary = taiga.run_config(t, cfg)
            torch.cuda.synchronize()
            got = {k: _np(ions.a[k]).copy() for k in ("hit_u", "hit_w", "cell", "steps", "flags")}
            got["counts"], got["summary"] = _np(counts).copy(), _np(summary).copy()
        finally:
            t.close()
        if base is None:
            base = got
            assert int(got["summary"][:, 0].sum()) > n // 2
            continue
        for k in base:
            same = base[k] == got[k] if base[k].dtype.kind != "f" else base[k].view(np.int64) == got[k].view(np.int64)
            assert same.all(), "%s differs under %s at %s" % (k, opts, np.flatnonzero(~same.reshape(-1))[:5])


def test_grazing_flags_match_the_oracle(tg):
    """The flag bits decide which ions parity leaves out, so the CUDA path must set them where the oracle does (whose own
    bits are pinned on the CPU, P25): straight flights in a zero field ending a step 5e-10 / 0.9e-9 / 1.1e-9 / 2e-9 m before
    and behind the detector plane and the four grid boundaries, and starts within the threshold.  cell and steps bit for
    bit; plane bit identical; grid bit set exactly where the point that left the grid is within the threshold, never where
    the oracle has none."""
    from paper_2506_15812_b200 import taiga
    grid, nodal = wl.nodal_field_2d(9, 17)
    nodal = [np.zeros_like(c) for c in nodal]
    tg.load_field(grid, nodal)
    f = orc.OracleField(grid, nodal)
    qm = wl.E_CHARGE / wl.MASS_LI7
    one = [np.array([-1.0]), np.array([1.0])] * 2
    d = np.array([-5e-10, 5e-10, -0.9e-9, 0.9e-9, -1.1e-9, 1.1e-9, -2e-9, 2e-9, -0.5e-3])
    cases = []                                               # (detector, x0, z0, vx, vz)
    det = wl.Detector((0.80, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), *one)
    cases.append((det, np.concatenate([0.80 - 3e-3 + d, 0.80 + np.array([-5e-10, 0.0, 5e-10, 1e-3])]), 0.0, 1e6, 0.0))
    far = wl.Detector((5.0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), *one)
    cases.append((far, np.concatenate([grid.Rmax - 3e-3 + d, grid.Rmax + np.array([-5e-10, 5e-10, 1e-3])]), 0.0, 1e6, 0.0))
    back = wl.Detector((-5.0, 0, 0), (-1, 0, 0), (0, 1, 0), (0, 0, 1), *one)
    cases.append((back, grid.Rmin + 3e-3 + d, 0.0, -1e6, 0.0))
    cases.append((far, np.full(len(d), 0.5), grid.Zmax - 3e-3 + d, 1.0, 1e6))
    cases.append((far, np.full(len(d), 0.5), grid.Zmin + 3e-3 - d, 1.0, -1e6))
    seen = 0
    for det, x0, z0, vx, vz in cases:
        n = len(x0)
        st = [np.asarray(x0, float), np.zeros(n), np.broadcast_to(np.asarray(z0, float), (n,)).copy(), np.full(n, vx), np.zeros(n), np.full(n, vz)]
        ref = orc.trace(f, qm, st, None, 1e-9, 20, det)
        ions = taiga.Ions(n)
        for k, a in zip(("x", "y", "z", "vx", "vy", "vz"), st):
            ions.a[k].copy_(torch.from_numpy(a))
        tg.trace(ions, qm, 1e-9, 20, det)
        torch.cuda.synchronize()
        fg, fr = _np(ions.flags), ref["flags"]
        assert np.array_equal(fg & 2, fr & 2), (fg, fr)              # plane bit: the same ions
        # grid bit: the kernels test the point that left the grid (taiga.h: "when leaving it"), the oracle every step end,
        # so a last INSIDE point within 1e-9 m of the boundary is flagged by the oracle only (parity ORs both sides' flags)
        k = ref["steps"].astype(float)
        Rend, Zend = st[0] + k * 1e-9 * st[3], st[2] + k * 1e-9 * st[5]
        left = (ref["status"] == -3) | ((ref["status"] == -4) & ((fr & 2) == 0))
        near_out = left & ((np.abs(Rend - grid.Rmin) < 1e-9) | (np.abs(Rend - grid.Rmax) < 1e-9) |
                           (np.abs(Zend - grid.Zmin) < 1e-9) | (np.abs(Zend - grid.Zmax) < 1e-9))
        assert np.array_equal((fg & 4) != 0, near_out), (fg, fr, near_out)
        assert np.all((fg & ~fr) == 0) and np.all(fg[fr == 0] == 0)
        assert np.array_equal(_np(ions.steps).astype(np.uint32), ref["steps"])
        assert np.array_equal(_np(ions.cell), np.where(ref["status"] == 0, -1, ref["status"]))
        seen |= int(np.bitwise_or.reduce(ref["flags"]))
        assert (ref["flags"] == 0).sum() >= 3
    assert seen == 6


def test_edge_cases_and_errors(tg):
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(1)
    grid, nodal = cfg.field_builder()
    t2 = taiga.Taiga(0)
    ions = taiga.Ions(8)
    with pytest.raises(taiga.TaigaError) as e:
        t2.trace(ions, 1.0, 1e-9, 10, cfg.detector)
    assert e.value.code == taiga.E_STATE
    t2.load_field(grid, nodal)
    for bad in (dict(dt=-1.0), dict(qm=0.0)):
        with pytest.raises(taiga.TaigaError) as e:
            t2.trace(ions, bad.get("qm", 1.0), bad.get("dt", 1e-9), 10, cfg.detector)
        assert e.value.code == taiga.E_ARG
    skew = wl.Detector((0.82, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0.1, 1.0), *([np.array([0.0]), np.array([1.0])] * 2))
    with pytest.raises(taiga.TaigaError):
        t2.trace(ions, 1.0, 1e-9, 10, skew)
    badcdf = wl.depth_cdf().copy()
    badcdf[5] = 0.9
    with pytest.raises(taiga.TaigaError):
        t2.seed_beam(cfg.groups[0].beam, badcdf, wl.normal_cdf(), 0, ions)
    # empty and tiny inputs
    t2.seed_beam(cfg.groups[0].beam, wl.depth_cdf(), wl.normal_cdf(), 0, taiga.Ions(0))
    t2.trace(taiga.Ions(0), 1.0, 1e-9, 10, cfg.detector)
    for n in (1, 31, 33):
        c = wl.config(1, n_override=n)
        io, counts, summary = taiga.run_config(t2, c, field_loaded=True)
        torch.cuda.synchronize()
        compare_groups(io, orc.run_config(c), "n=%d" % n)
    # degenerate: max_steps = 0 and 1; every ion starts behind the plane
    c = wl.config(1, n_override=257)
    for ms in (0, 1):
        c.max_steps = ms
        io, counts, summary = taiga.run_config(t2, c, field_loaded=True)
        torch.cuda.synchronize()
        compare_groups(io, orc.run_config(c), "max_steps=%d" % ms)
        assert int(summary[0, 2]) == 257
    c = wl.config(1, n_override=100)
    c.detector = wl.uniform_detector(0.02, 0.18, 8, 2.5e-3, x_plane=0.5)
    io, counts, summary = taiga.run_config(t2, c, field_loaded=True)
    torch.cuda.synchronize()
    compare_groups(io, orc.run_config(c), "behind plane")
    assert int(summary[0, 4]) == 100
    t2.close()


def test_cfg2_full_size_bench_configuration(tg):
    """BASELINE config 2 at full size in the launch configuration bench.py times: invariants at
    any size + sampled ions checked one by one against the oracle."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(2)
    ions, counts, summary = taiga.run_config(tg, cfg)
    torch.cuda.synchronize()
    s = _np(summary)[0]
    assert s[:5].sum() == cfg.n_ions and s[0] == _np(counts).sum()
    st = tg.stats()
    assert st["ion_steps"] == int(_np(ions.steps).astype(np.int64).sum())
    rng = np.random.default_rng(2)
    idx = np.sort(rng.choice(cfg.n_ions, 6000, replace=False))
    grid, nodal = cfg.field_builder()
    f = orc.OracleField(grid, nodal)
    g = cfg.groups[0]
    state = [_np(ions.a[k])[idx] for k in ("x", "y", "z", "vx", "vy", "vz")]
    seeds = orc.seed(g.beam, wl.depth_cdf(), wl.normal_cdf(), cfg.seed, 0, int(idx.max()) + 1)
    for a, b in zip(state, seeds):
        assert np.array_equal(a, b[idx])
    res = orc.trace(f, g.beam.charge_C / g.beam.mass_kg, state, None, cfg.dt, cfg.max_steps, cfg.detector)
    orc.histogram(res, None, cfg.detector, 1)
    fl = (_np(ions.flags)[idx] | res["flags"]) != 0
    ok = ~fl
    assert np.array_equal(_np(ions.cell)[idx][ok], res["cell"][ok])
    assert np.array_equal(_np(ions.steps)[idx][ok].astype(np.uint32), res["steps"][ok])
    cr = ok & (res["status"] == 0)
    assert np.abs(_np(ions.hit_u)[idx][cr] - res["u"][cr]).max() < TOL_UW
    assert np.abs(_np(ions.hit_w)[idx][cr] - res["w"][cr]).max() < TOL_UW
    # mean steps / structure of the workload (SURVEY 8(d) probe: ~1038 steps/ion, 96.3 % cross)
    assert 900 < st["ion_steps"] / cfg.n_ions < 1200
    assert 0.955 < (s[0] + s[1]) / cfg.n_ions < 0.97


def _full_size_check(tg, icfg, windows, width, max_flag_frac=0.01):
    """A BASELINE config at FULL size: invariants that hold at any size, plus windows of
    consecutive ions per group re-seeded and re-traced one by one by the oracle."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(icfg)
    ions, counts, summary = taiga.run_config(tg, cfg)
    torch.cuda.synchronize()
    s = _np(summary)
    assert s[:, :5].sum() == cfg.n_ions                                   # O5 counting invariant
    assert np.array_equal(s[:, 0], _np(counts).reshape(cfg.n_hist, -1).sum(axis=1))
    cell_all = ions.cell
    assert int((cell_all >= 0).sum().item()) == int(s[:, 0].sum())
    assert int((cell_all < -4).sum().item()) == 0
    grid, nodal = cfg.field_builder()
    f = orc.OracleField(grid, nodal)
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    rng = np.random.default_rng(100 + icfg)
    off, n_cmp, n_flag, max_d = 0, 0, 0, 0.0
    for g in cfg.groups:
        det = cfg.detector or g.detector
        for lo in sorted(rng.integers(0, g.n_ions - width, windows).tolist()) + [g.n_ions - width]:
            v = ions.view(off + lo, off + lo + width)
            seeds = orc.seed(g.beam, cd, cn, cfg.seed, g.first_index + lo, width)
            state = [_np(v.a[k]) for k in ("x", "y", "z", "vx", "vy", "vz")]
            for a, b in zip(state, seeds):
                assert np.array_equal(a, b), (icfg, g.group, lo)
            t0 = np.full(width, g.t0) if grid.kind == 1 else None
            res = orc.trace(f, g.beam.charge_C / g.beam.mass_kg, state, t0, cfg.dt, cfg.max_steps, det)
            orc.histogram(res, None, det, 1)
            fl = (_np(v.flags) | res["flags"]) != 0
            ok = ~fl
            assert np.array_equal(_np(v.cell)[ok], res["cell"][ok]), (icfg, g.group, lo)
            assert np.array_equal(_np(v.steps)[ok].astype(np.uint32), res["steps"][ok]), (icfg, g.group, lo)
            assert np.all(_np(v.group) == g.group)
            cr = ok & (res["status"] == 0)
            if cr.any():
                max_d = max(max_d, np.abs(_np(v.hit_u)[cr] - res["u"][cr]).max(), np.abs(_np(v.hit_w)[cr] - res["w"][cr]).max())
            n_cmp += width
            n_flag += int(fl.sum())
        off += g.n_ions
    assert max_d < TOL_UW, max_d
    assert n_flag <= max(4, int(max_flag_frac * n_cmp))
    return cfg, s


def test_cfg3_full_size_energy_scan(tg):
    """16,777,216 ions, four energies with their own detectors, 2 mrad divergence."""
    cfg, s = _full_size_check(tg, 3, windows=3, width=96)
    frac = (s[:, 0] + s[:, 1]) / (cfg.n_ions / 4)
    # SURVEY 8(d) probe: crossers 69.5 / 90.6 / 96.3 / 98.1 %
    assert np.all(np.abs(frac - np.array([0.695, 0.906, 0.963, 0.981])) < 0.02), frac


def test_cfg4_full_size_time_slices(tg):
    """2,097,152 Na+ ions over 64 time slices, one histogram per slice."""
    cfg, s = _full_size_check(tg, 4, windows=1, width=64)
    assert np.all(s[:, :5].sum(axis=1) == cfg.n_ions // 64)
    assert 0.99 < (s[:, 0] + s[:, 1]).sum() / cfg.n_ions < 1.0


def test_cfg5_full_size_ripple_3d(tg):
    """67,108,864 ions in the periodic-tricubic (R, Z, phi) field: the largest configuration
    (6.2 GB of ion state, 1.6 GB of tables)."""
    cfg, s = _full_size_check(tg, 5, windows=2, width=64)
    assert 0.95 < (s[0, 0] + s[0, 1]) / cfg.n_ions < 0.975


@pytest.mark.parametrize("icfg,n", [(1, 2048 + 19), (4, 128), (5, 1024 + 5)])
@pytest.mark.parametrize("solver", [2, 3, 4])
def test_other_solvers_parity(tg, icfg, n, solver):
    """linearised RK4 (Eq. 4) and Boris (Eq. 7-8, both position readings)
    on all three field kinds, same acceptance as the RKN path."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(icfg, n_override=n)
    ions, counts, summary = taiga.run_config(tg, cfg, rkn_variant=solver)
    torch.cuda.synchronize()
    ref = orc.run_config(cfg, variant=solver)
    st = compare_groups(ions, ref, "%s solver %d" % (cfg.name, solver))
    check_histogram(cfg, ions, counts, summary, ref)
    assert st["flagged"] <= max(8, st["n"] // 200)
    # the solver switch is live: Boris at the production step lands micrometres-millimetres from RKN
    if solver >= 3:
        ref0 = orc.run_config(cfg, field=ref["field"], variant=0)
        g, g0 = ref["groups"][0], ref0["groups"][0]
        cr = (g["status"] == 0) & (g0["status"] == 0)
        assert np.abs(g["w"][cr] - g0["w"][cr]).max() > 1e-7


@pytest.mark.parametrize("solver", [0, 1, 2, 3])
def test_uniform_E_field_parity(tg, solver):
    """Eq. 3 with a uniform ("parametric", L175) electric field, through every solver; an
    E of 50 kV/m moves the hits by far more than the tolerance, so the term is live."""
    from paper_2506_15812_b200 import taiga
    E = (3.0e4, -2.0e4, 5.0e4)
    cfg = wl.config(1, n_override=1500)
    grid, nodal = cfg.field_builder()
    try:
        tg.set_efield(E)
        ions, counts, summary = taiga.run_config(tg, cfg, rkn_variant=solver)
        torch.cuda.synchronize()
    finally:
        tg.set_efield((0.0, 0.0, 0.0))
    fE = orc.OracleField(grid, nodal, E=E)
    ref = orc.run_config(cfg, field=fE, variant=solver)
    compare_groups(ions, ref, "cfg1 E solver %d" % solver)
    check_histogram(cfg, ions, counts, summary, ref)
    ref0 = orc.run_config(cfg, variant=solver)
    g, g0 = ref["groups"][0], ref0["groups"][0]
    cr = (g["status"] == 0) & (g0["status"] == 0)
    assert np.abs(g["w"][cr] - g0["w"][cr]).max() > 1e-5


@pytest.mark.parametrize("icfg,n,solver", [(1, 1200 + 7, 0), (1, 1200 + 7, 1), (1, 1200 + 7, 2), (1, 1200 + 7, 3), (1, 1200 + 7, 4),
                                           (4, 48, 0), (4, 48, 3), (5, 1024 + 3, 0), (5, 1024 + 3, 2), (5, 1024 + 3, 3)])
def test_gridded_E_field_parity(tg, icfg, n, solver):
    """Eq. 3 with E(R, Z) given on the poloidal grid like B (taiga_load_efield, reading E1), added to a uniform E, through
    every solver and all three kinds of B (kind 2: the DMMA tracer).  Sheath-like radial field growing towards the outer
    wall, a vertical field linear in Z and a constant toroidal component: tens of kV/m, which move the hits by far more
    than the tolerance."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(icfg, n_override=n)
    grid, nodal = cfg.field_builder()
    R = np.linspace(grid.Rmin, grid.Rmax, grid.nR)[:, None] * np.ones((1, grid.nZ))
    Z = np.ones((grid.nR, 1)) * np.linspace(grid.Zmin, grid.Zmax, grid.nZ)[None, :]
    En = (4.0e4 * np.exp((R - 0.8) / 0.05) - 1.0e4 * 0.56 / R, 6.0e4 * Z, 2.0e4 + 0.0 * R)
    Eu = (1.0e4, 0.0, -5.0e3)
    tg.load_field(grid, nodal)
    tg.load_efield(En)
    tg.set_efield(Eu)
    ions, counts, summary = taiga.run_config(tg, cfg, field_loaded=True, rkn_variant=solver)
    torch.cuda.synchronize()
    fE = orc.OracleField(grid, nodal, E=Eu, E_nodal=En)
    ref = orc.run_config(cfg, field=fE, variant=solver)
    compare_groups(ions, ref, "%s gridded E solver %d" % (cfg.name, solver))
    check_histogram(cfg, ions, counts, summary, ref)
    # the gridded part is live, and removing it restores the uniform-E result
    tg.load_efield(None)
    ions2, _, _ = taiga.run_config(tg, cfg, field_loaded=True, rkn_variant=solver)
    torch.cuda.synchronize()
    ref2 = orc.run_config(cfg, field=orc.OracleField(grid, nodal, E=Eu), variant=solver)
    compare_groups(ions2, ref2, "%s uniform E after removing the grid" % cfg.name)
    a, b = ref["groups"][0], ref2["groups"][0]
    cr = (a["status"] == 0) & (b["status"] == 0)
    assert np.abs(a["w"][cr] - b["w"][cr]).max() > 1e-5


def test_cfg5_fp32_variant(tg):
    """BASELINE config 5 'fp32 variant' (reading A19): the tricubic field evaluation and its table
    in fp32, the ion state integrated in fp64.  north_star: hit coordinates within 1e-5 m of the
    fp64 oracle; integer outputs are not expected to be bit-exact (fp32 decides no integer here,
    but the trajectories differ at the 1e-7 m level), so agreement rates are asserted instead."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(5, n_override=65536 + 21)
    try:
        tg.set_option("precision", 32)
        ions, counts, summary = taiga.run_config(tg, cfg)
        torch.cuda.synchronize()
    finally:
        tg.set_option("precision", 64)
    ref = orc.run_config(cfg)
    g = ref["groups"][0]
    n = cfg.n_ions
    for k, a in zip(("x", "y", "z", "vx", "vy", "vz"), g["state0"]):
        assert np.array_equal(_np(ions.a[k]), a)                           # seeding stays fp64, bit-exact
    cell, steps = _np(ions.cell), _np(ions.steps).astype(np.uint32)
    status_gpu = np.where(cell >= -1, 0, cell)
    same_status = status_gpu == g["status"]
    assert same_status.mean() > 0.995
    cr = same_status & (g["status"] == 0)
    same_steps = steps[cr] == g["steps"][cr]
    assert same_steps.mean() > 0.999
    sel = np.flatnonzero(cr)[same_steps]
    du = np.abs(_np(ions.hit_u)[sel] - g["u"][sel])
    dw = np.abs(_np(ions.hit_w)[sel] - g["w"][sel])
    assert max(du.max(), dw.max()) < 1e-5, (du.max(), dw.max())
    assert np.median(np.maximum(du, dw)) < 1e-6
    assert max(du.max(), dw.max()) > 1e-10                                 # fp32 really ran
    assert (cell[cr] == g["cell"][cr]).mean() > 0.99                       # 0.5 mm segments, 1e-7 m errors
    s = _np(summary)[0]
    assert s[:5].sum() == n and s[0] == _np(counts).sum()
    # fp32 is refused where it is not offered
    cfg1 = wl.config(1, n_override=64)
    try:
        tg.set_option("precision", 32)
        with pytest.raises(taiga.TaigaError):
            taiga.run_config(tg, cfg1)
    finally:
        tg.set_option("precision", 64)


@pytest.mark.parametrize("icfg,n,species", [(1, 3000 + 7, "li"), (2, 4096, "li"), (4, 64, "na"), (5, 1024, "li"), (5, 16384 + 3, "li")])
def test_secondary_ionisation_loss_parity(tg, icfg, n, species):
    """SURVEY 8(f) NEXT-1 (Eq. 2): per-ion surviving fraction and the 32.32
    fixed-point weighted counters against the oracle.  Tolerance on the weight: 1e-12 relative
    (the integral is a sum of <= max_steps terms of fp64 rounding differences; exp() differs by an
    ulp between libm and the device); integer outputs as in the plain path; fixed-point sums may
    differ by one unit (2^-32) per ion whose weight rounds differently."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(icfg, n_override=n)
    grid, nodal = cfg.field_builder()
    psi0, dpsi, ne, te = wl.loss_profile_inputs()
    E12 = wl.E12_LI if species == "li" else wl.E12_NA
    psi_nodal = wl.nodal_psi(grid)
    tg.load_field(grid, nodal)
    try:
        tg.load_loss(psi_nodal, psi0, dpsi, ne, te, E12)
        ions, counts, summary = taiga.run_config(tg, cfg, field_loaded=True)
        det0 = cfg.detector or cfg.groups[0].detector
        wcounts = torch.zeros((cfg.n_hist, det0.nw, det0.nu), dtype=torch.int64, device="cuda")
        wsummary = torch.zeros((cfg.n_hist, 4), dtype=torch.int64, device="cuda")
        off = 0
        for g in cfg.groups:
            tg.detector_histogram_weighted(ions.view(off, off + g.n_ions), g.detector or cfg.detector, cfg.n_hist, wcounts, wsummary)
            off += g.n_ions
        torch.cuda.synchronize()
    finally:
        tg.load_loss(None)
    f = orc.OracleField(grid, nodal)
    L = orc.OracleLoss(grid, psi_nodal, psi0, dpsi, orc.mcwhirter_rate(ne, te, E12))
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    wc_ref = np.zeros((cfg.n_hist, det0.nw, det0.nu), dtype=np.uint64)
    ws_ref = np.zeros((cfg.n_hist, 4), dtype=np.uint64)
    off, n_cross, worst, n_round = 0, 0, 0.0, 0
    ref_weights = []
    for g in cfg.groups:
        det = g.detector or cfg.detector
        st = orc.seed(g.beam, cd, cn, cfg.seed, g.first_index, g.n_ions)
        t0 = np.full(g.n_ions, g.t0)
        res = orc.trace_loss(f, L, g.beam.charge_C / g.beam.mass_kg, st, t0, cfg.dt, cfg.max_steps, det)
        grp = np.full(g.n_ions, g.group, dtype=np.uint16)
        orc.histogram(res, grp, det, cfg.n_hist)
        v = ions.view(off, off + g.n_ions)
        fl = (_np(v.flags) | res["flags"]) != 0
        ok = ~fl
        assert np.array_equal(_np(v.cell)[ok], res["cell"][ok]) and np.array_equal(_np(v.steps)[ok].astype(np.uint32), res["steps"][ok])
        wg, wr = _np(v.weight), res["weight"]
        assert np.all((wg > 0) & (wg <= 1.0))
        rel = np.abs(wg[ok] / wr[ok] - 1)
        worst = max(worst, rel.max())
        # weighted counters: the oracle's sums over the GPU's unflagged set + the GPU's own flagged ions
        res_w = dict(cell=np.where(ok, res["cell"], _np(v.cell)).astype(np.int32), weight=np.where(ok, wr, wg))
        orc.histogram_weighted(res_w, grp, det, cfg.n_hist, wc_ref, ws_ref)
        qg = np.floor(wg * 4294967296.0 + 0.5); qr = np.floor(res_w["weight"] * 4294967296.0 + 0.5)
        n_round += int((qg != qr).sum())
        n_cross += int((res["status"] == 0).sum())
        ref_weights.append(res["weight"][res["status"] == 0])
        off += g.n_ions
    assert worst < 1e-12, worst
    wc, ws = _np(wcounts).astype(np.int64), _np(wsummary).astype(np.int64)
    assert np.abs(wc - wc_ref.astype(np.int64)).sum() <= n_round
    assert np.abs(ws[:, :2] - ws_ref[:, :2].astype(np.int64)).sum() <= n_round
    assert np.abs(ws[:, 2] - ws_ref[:, 2].astype(np.int64)).sum() <= 2 * n_round + 2
    assert np.array_equal(ws[:, 3], ws_ref[:, 3].astype(np.int64))
    assert n_round <= max(2, n_cross // 50)
    # the loss is live: percent level for these profiles
    loss = 1.0 - ws[:, :2].sum() / 4294967296.0 / max(ws[:, 3].sum(), 1)
    assert 1e-3 < loss < 0.5, loss
    # Table-1 style statistics from the fixed-point sums against the oracle's per-ion weights
    if cfg.n_hist == 1:
        mean_loss, std_loss = taiga.loss_statistics(wsummary)
        wr_all = np.concatenate([r for r in ref_weights])
        assert abs(mean_loss[0] - (1.0 - wr_all.mean())) < 1e-9 and abs(std_loss[0] - wr_all.std()) < 1e-6
    # without a loss model the same call leaves the weights alone
    ions.a["weight"].fill_(7.0)
    taiga.run_config(tg, wl.config(icfg, n_override=64), field_loaded=True, ions=ions.view(0, 64 * len(cfg.groups)))
    torch.cuda.synchronize()
    assert float(ions.weight[:64].min()) == 7.0


@pytest.mark.parametrize("icfg,n", [(1, 4096), (4, 128), (5, 1024 + 3), (5, 16384 + 5)])
def test_bezier_plane_interpolation_parity(tg, icfg, n):
    """quadratic Bezier interpolation to the detector plane."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(icfg, n_override=n)
    try:
        tg.set_option("plane_interp", 1)
        ions, counts, summary = taiga.run_config(tg, cfg)
        torch.cuda.synchronize()
    finally:
        tg.set_option("plane_interp", 0)
    ref = orc.run_config(cfg, interp=1)
    compare_groups(ions, ref, "%s bezier" % cfg.name)
    check_histogram(cfg, ions, counts, summary, ref)
    lin = orc.run_config(cfg, field=ref["field"], interp=0)
    g, g0 = ref["groups"][0], lin["groups"][0]
    cr = (g["status"] == 0) & (g0["status"] == 0)
    d = np.hypot(g["u"][cr] - g0["u"][cr], g["w"][cr] - g0["w"][cr]).max()
    assert 1e-8 < d < 1e-3                    # micrometres (more at grazing incidence): the switch is live


@pytest.mark.parametrize("icfg,n,solver,mode", [
    (1, 1500 + 3, 0, "loss+E"), (1, 1500 + 3, 1, "loss+E"), (1, 1500 + 3, 2, "loss"), (1, 1500 + 3, 3, "loss"), (1, 1500 + 3, 4, "loss+E"),
    (1, 1500 + 3, 0, "bezier+E"), (1, 1500 + 3, 1, "bezier+E"),
    (4, 40, 0, "loss+E"), (4, 40, 2, "loss"), (4, 40, 0, "bezier+E"),
    (5, 1024 + 9, 0, "loss+E"), (5, 1024 + 9, 2, "loss"), (5, 1024 + 9, 3, "loss+E"), (5, 1024 + 9, 0, "bezier+E"),
    (1, 1500 + 3, 0, "loss+bezier"), (1, 1500 + 3, 1, "loss+bezier+E"), (4, 40, 0, "loss+bezier+E"), (5, 1024 + 9, 0, "loss+bezier"),
    (5, 1024 + 9, 0, "loss+bezier+E"),
])
def test_loss_and_bezier_with_E_and_the_other_solvers(tg, icfg, n, solver, mode):
    """The loss integral (Eq. 2) along trajectories of every solver, with or without an electric field, and the Bezier
    plane interpolation (L338) with an electric field and with the loss integral (the crossing step counts up to the curve
    parameter of the hit, reading L2'): the combinations round 1 refused."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(icfg, n_override=n)
    grid, nodal = cfg.field_builder()
    E = (2.0e4, -1.0e4, 3.0e4) if "+E" in mode else (0.0, 0.0, 0.0)
    tg.load_field(grid, nodal)
    tg.set_efield(E)
    f = orc.OracleField(grid, nodal, E=E)
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    interp = 1 if "bezier" in mode else 0
    tg.set_option("plane_interp", interp)
    if mode.startswith("bezier"):
        ions, counts, summary = taiga.run_config(tg, cfg, field_loaded=True, rkn_variant=solver)
        torch.cuda.synchronize()
        ref = orc.run_config(cfg, field=f, variant=solver, interp=1)
        compare_groups(ions, ref, "%s %s solver %d" % (cfg.name, mode, solver))
        check_histogram(cfg, ions, counts, summary, ref)
        return
    species_E12 = wl.E12_NA if icfg == 4 else wl.E12_LI
    psi0, dpsi, ne, te = wl.loss_profile_inputs()
    psi_nodal = wl.nodal_psi(grid)
    tg.load_loss(psi_nodal, psi0, dpsi, ne, te, species_E12)
    ions, counts, summary = taiga.run_config(tg, cfg, field_loaded=True, rkn_variant=solver)
    torch.cuda.synchronize()
    L = orc.OracleLoss(grid, psi_nodal, psi0, dpsi, orc.mcwhirter_rate(ne, te, species_E12))
    off, worst, ncross = 0, 0.0, 0
    for g in cfg.groups:
        det = g.detector or cfg.detector
        st = orc.seed(g.beam, cd, cn, cfg.seed, g.first_index, g.n_ions)
        res = orc.trace_loss(f, L, g.beam.charge_C / g.beam.mass_kg, st, np.full(g.n_ions, g.t0), cfg.dt, cfg.max_steps, det, variant=solver,
                             interp=interp)
        orc.histogram(res, np.full(g.n_ions, g.group, dtype=np.uint16), det, cfg.n_hist)
        v = ions.view(off, off + g.n_ions)
        ok = ((_np(v.flags) | res["flags"]) == 0)
        assert np.array_equal(_np(v.cell)[ok], res["cell"][ok]) and np.array_equal(_np(v.steps)[ok].astype(np.uint32), res["steps"][ok])
        cr = ok & (res["status"] == 0)
        if cr.any():
            assert np.abs(_np(v.hit_u)[cr] - res["u"][cr]).max() < TOL_UW and np.abs(_np(v.hit_w)[cr] - res["w"][cr]).max() < TOL_UW
        wg, wr = _np(v.weight), res["weight"]
        assert np.all((wg > 0) & (wg <= 1.0))
        worst = max(worst, np.abs(wg[ok] / wr[ok] - 1).max())
        ncross += int(cr.sum())
        off += g.n_ions
    assert worst < 1e-12, worst
    assert ncross > 0


def test_deterministic_grid_seeding_parity(tg):
    """weighted-grid initialisation, bit-exact against the
    oracle (positions, velocities, weights), incl. sub-ranges (sharding) and a tilted beam frame;
    then the whole path: trace + loss + weighted counters with the initial weights."""
    from paper_2506_15812_b200 import taiga
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    tilted = wl.Beam(wl.MASS_NA23, wl.E_CHARGE, 40e3, sigma_pos_m=7e-3, sigma_ang_rad=0.0,
                     origin=(0.8, 0.01, -0.02), axis=(-0.6, 0.0, 0.8), eT=(0.0, 1.0, 0.0), eZ=(0.8, 0.0, 0.6))
    tilted.depth_max, tilted.z_max = wl.DEPTH_MAX, wl.NORMAL_ZMAX
    for beam, (nd, nT, nZ, zl), first, n in ((wl.config(1).groups[0].beam, (64, 9, 11, 6.0), 0, 64 * 9 * 11),
                                               (tilted, (1000, 31, 17, 3.5), 123457, 10007),
                                               (tilted, (3, 1, 1, 0.5), 2, 1)):
        ions = taiga.Ions(n)
        tg.seed_beam_grid(beam, cd, cn, nd, nT, nZ, zl, ions, first_index=first, group=2, t0=1e-6)
        torch.cuda.synchronize()
        st, w0 = orc.seed_grid(beam, cd, cn, nd, nT, nZ, zl, first, n)
        for k, a in zip(("x", "y", "z", "vx", "vy", "vz"), st):
            assert np.array_equal(_np(ions.a[k]), a), k
        assert np.array_equal(_np(ions.w0), w0)
        assert np.all(_np(ions.group) == 2) and np.all(_np(ions.t0) == 1e-6)
    with pytest.raises(taiga.TaigaError):
        tg.seed_beam_grid(tilted, cd, cn, 3, 1, 1, 0.5, taiga.Ions(2), first_index=2)       # beyond the grid
    # whole path on config 1's field: grid seeding -> trace with the loss model -> weighted counters
    cfg = wl.config(1)
    grid, nodal = cfg.field_builder()
    g = cfg.groups[0]
    nd, nT, nZ, zl = 128, 7, 7, 4.0
    n = nd * nT * nZ
    psi0, dpsi, ne, te = wl.loss_profile_inputs()
    psi_nodal = wl.nodal_psi(grid)
    tg.load_field(grid, nodal)
    ions = taiga.Ions(n)
    counts = torch.zeros((1, 8, 8), dtype=torch.int64, device="cuda")
    summary = torch.zeros((1, 6), dtype=torch.int64, device="cuda")
    wcounts = torch.zeros((1, 8, 8), dtype=torch.int64, device="cuda")
    wsummary = torch.zeros((1, 4), dtype=torch.int64, device="cuda")
    w0counts, w0summary = torch.zeros_like(wcounts), torch.zeros_like(wsummary)
    qm = g.beam.charge_C / g.beam.mass_kg
    try:
        tg.load_loss(psi_nodal, psi0, dpsi, ne, te, wl.E12_LI)
        tg.seed_beam_grid(g.beam, cd, cn, nd, nT, nZ, zl, ions)
        tg.trace(ions, qm, cfg.dt, cfg.max_steps, cfg.detector)
        tg.detector_histogram(ions, cfg.detector, 1, counts, summary)
        tg.detector_histogram_weighted(ions, cfg.detector, 1, wcounts, wsummary)
        tg.detector_histogram_weighted(ions, cfg.detector, 1, w0counts, w0summary, use_loss_weight=False)
        torch.cuda.synchronize()
    finally:
        tg.load_loss(None)
    f = orc.OracleField(grid, nodal)
    L = orc.OracleLoss(grid, psi_nodal, psi0, dpsi, orc.mcwhirter_rate(ne, te, wl.E12_LI))
    st, w0 = orc.seed_grid(g.beam, cd, cn, nd, nT, nZ, zl, 0, n)
    res = orc.trace_loss(f, L, qm, st, None, cfg.dt, cfg.max_steps, cfg.detector, w0=w0)
    orc.histogram(res, None, cfg.detector, 1)
    ok = ((_np(ions.flags) | res["flags"]) == 0)
    assert ok.mean() > 0.99
    assert np.array_equal(_np(ions.cell)[ok], res["cell"][ok]) and np.array_equal(_np(ions.steps)[ok].astype(np.uint32), res["steps"][ok])
    nz = ok & (res["weight"] > 0)
    assert np.abs(_np(ions.weight)[nz] / res["weight"][nz] - 1).max() < 1e-12
    assert np.array_equal(_np(ions.weight)[ok & ~nz], res["weight"][ok & ~nz])
    wc_ref, ws_ref = orc.histogram_weighted(dict(cell=np.where(ok, res["cell"], _np(ions.cell)).astype(np.int32),
                                                 weight=np.where(ok, res["weight"], _np(ions.weight))), None, cfg.detector, 1)
    assert np.abs(_np(wcounts) - wc_ref.astype(np.int64)).sum() <= 8 and np.abs(_np(wsummary)[:, :2] - ws_ref[:, :2].astype(np.int64)).sum() <= 8
    # w0-only counters: exact integers (identical doubles on both sides)
    w0_ref, w0s_ref = orc.histogram_weighted(dict(cell=_np(ions.cell), weight=w0), None, cfg.detector, 1)
    assert np.array_equal(_np(w0counts), w0_ref.astype(np.int64)) and np.array_equal(_np(w0summary), w0s_ref.astype(np.int64))
    # the loss reduces the weighted signal by about a percent for these profiles
    ratio = _np(wsummary)[0, :2].sum() / _np(w0summary)[0, :2].sum()
    assert 0.95 < ratio < 0.999


def test_error_paths_of_the_widened_entry_points(tg):
    """Combinations that are not offered are refused (TAIGA_E_ARG / TAIGA_E_STATE), never computed
    differently; null / malformed inputs are rejected."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(1, n_override=64)
    grid, nodal = cfg.field_builder()
    psi0, dpsi, ne, te = wl.loss_profile_inputs()
    g = cfg.groups[0]
    qm = g.beam.charge_C / g.beam.mass_kg
    t2 = taiga.Taiga(0)
    with pytest.raises(taiga.TaigaError) as e:
        t2.load_loss(wl.nodal_psi(grid), psi0, dpsi, ne, te, wl.E12_LI)            # before load_field
    assert e.value.code == taiga.E_STATE
    with pytest.raises(taiga.TaigaError) as e:
        t2.load_efield([nodal[0][0], nodal[1][0], nodal[2][0]])                    # the grid of B carries E: before load_field
    assert e.value.code == taiga.E_STATE
    t2.load_field(grid, nodal)
    for bad in (dict(dpsi=0.0), dict(E12=-1.0), dict(ne=-ne), dict(ne=ne[:1], te=te[:1])):
        kw = dict(psi0=psi0, dpsi=dpsi, ne=ne, Te=te, E12=wl.E12_LI)
        kw.update({("Te" if k == "te" else k): v for k, v in bad.items()})
        with pytest.raises(taiga.TaigaError) as e:
            t2.load_loss(wl.nodal_psi(grid), **kw)
        assert e.value.code == taiga.E_ARG
    ions = taiga.Ions(64)
    t2.seed_beam(g.beam, wl.depth_cdf(), wl.normal_cdf(), 0, ions)
    with pytest.raises(taiga.TaigaError):
        t2.trace(ions, qm, cfg.dt, 100, cfg.detector, 5)                            # unknown solver
    with pytest.raises(taiga.TaigaError):
        t2.set_efield((float("nan"), 0.0, 0.0))
    t2.load_loss(wl.nodal_psi(grid), psi0, dpsi, ne, te, wl.E12_LI)
    t2.set_option("plane_interp", 1)
    t2.trace(ions, qm, cfg.dt, 100, cfg.detector)                                   # loss + Bezier, loss + E, loss + Boris: offered since round 2
    t2.set_option("plane_interp", 0)
    t2.set_efield((1e3, 0, 0))
    t2.trace(ions, qm, cfg.dt, 100, cfg.detector)
    t2.trace(ions, qm, cfg.dt, 100, cfg.detector, 3)
    t2.set_efield((0, 0, 0))
    t2.set_option("precision", 32)
    with pytest.raises(taiga.TaigaError) as e:
        t2.trace(ions, qm, cfg.dt, 100, cfg.detector)                               # fp32 is kind 2 + RKN, no loss model
    assert e.value.code == taiga.E_ARG
    t2.set_option("precision", 64)
    t2.load_loss(None)
    t2.set_option("plane_interp", 1)
    with pytest.raises(taiga.TaigaError):
        t2.trace(ions, qm, cfg.dt, 100, cfg.detector, 2)                            # Bezier + RK4
    t2.set_option("plane_interp", 0)
    for key, bad in (("precision", 16), ("ctas_per_sm", 1 << 20), ("variant", 99), ("regroup", -1), ("no_such_option", 1)):
        with pytest.raises(taiga.TaigaError) as e:                                 # options are validated when set
            t2.set_option(key, bad)
        assert e.value.code == taiga.E_ARG
    t2.trace(ions, qm, cfg.dt, 100, cfg.detector)                                   # and a rejected value changes nothing
    # a new field invalidates the loss model (psi lives on the old grid)
    t2.load_loss(wl.nodal_psi(grid), psi0, dpsi, ne, te, wl.E12_LI)
    t2.load_field(grid, nodal)
    ions.a["weight"].fill_(5.0)
    t2.trace(ions, qm, cfg.dt, 100, cfg.detector)
    torch.cuda.synchronize()
    assert float(ions.weight.min()) == 5.0
    # weighted histogram needs weights
    wc = torch.zeros((1, 8, 8), dtype=torch.int64, device="cuda"); ws = torch.zeros((1, 4), dtype=torch.int64, device="cuda")
    with pytest.raises(taiga.TaigaError) as e:                # weights the last trace did not write (no loss model) are refused
        t2.detector_histogram_weighted(ions, cfg.detector, 1, wc, ws)
    assert e.value.code == taiga.E_STATE
    # ... per weight array, not per context: trace A with the model, then B, then A's weights still count and C's do not
    t2.load_loss(wl.nodal_psi(grid), psi0, dpsi, ne, te, wl.E12_LI)
    ionsB, ionsC = taiga.Ions(64), taiga.Ions(64)
    for io in (ionsB, ionsC):
        t2.seed_beam(g.beam, wl.depth_cdf(), wl.normal_cdf(), 0, io)
    t2.trace(ions, qm, cfg.dt, 5000, cfg.detector)
    t2.trace(ionsB, qm, cfg.dt, 5000, cfg.detector)
    for io in (ions, ionsB, ions.view(8, 40)):
        t2.detector_histogram_weighted(io, cfg.detector, 1, wc, ws)
    with pytest.raises(taiga.TaigaError) as e:
        t2.detector_histogram_weighted(ionsC, cfg.detector, 1, wc, ws)
    assert e.value.code == taiga.E_STATE
    t2.load_loss(None)
    t2.trace(ionsB, qm, cfg.dt, 5000, cfg.detector)           # B's weights are stale now, A's are not
    t2.detector_histogram_weighted(ions, cfg.detector, 1, wc, ws)
    with pytest.raises(taiga.TaigaError) as e:
        t2.detector_histogram_weighted(ionsB, cfg.detector, 1, wc, ws)
    assert e.value.code == taiga.E_STATE
    # fp32 evaluation with an electric field is not offered
    g5, n5 = wl.nodal_field_ripple(9, 9, 8)
    t2.load_field(g5, n5)
    t2.set_option("precision", 32)
    t2.set_efield((1e3, 0, 0))
    with pytest.raises(taiga.TaigaError) as e:
        t2.trace(ions, qm, cfg.dt, 10, cfg.detector)
    assert e.value.code == taiga.E_ARG and "electric" in str(e.value)
    t2.set_efield((0, 0, 0))
    t2.trace(ions, qm, cfg.dt, 10, cfg.detector)
    t2.set_option("precision", 64)
    t2.load_field(grid, nodal)
    ions.a["weight"].fill_(5.0)
    s = ions.struct(weight=False)
    assert s.w0 is None
    with pytest.raises(taiga.TaigaError):
        t2.detector_histogram_weighted(ions, cfg.detector, 1, wc, ws, use_loss_weight=False)
    t2.close()


def test_printed_k3_variant_with_loss_and_with_bezier(tg):
    """The printed-Eq. 6 RKN reading (solver 1) through the loss and the Bezier kernels (uncached
    instantiations, since k2 and k3 no longer share their position)."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(1, n_override=1024 + 9)
    grid, nodal = cfg.field_builder()
    g = cfg.groups[0]
    qm = g.beam.charge_C / g.beam.mass_kg
    psi0, dpsi, ne, te = wl.loss_profile_inputs()
    psi_nodal = wl.nodal_psi(grid)
    f = orc.OracleField(grid, nodal)
    st = orc.seed(g.beam, wl.depth_cdf(), wl.normal_cdf(), cfg.seed, 0, cfg.n_ions)
    tg.load_field(grid, nodal)
    try:
        tg.load_loss(psi_nodal, psi0, dpsi, ne, te, wl.E12_LI)
        ions, counts, summary = taiga.run_config(tg, cfg, field_loaded=True, rkn_variant=1)
        torch.cuda.synchronize()
    finally:
        tg.load_loss(None)
    L = orc.OracleLoss(grid, psi_nodal, psi0, dpsi, orc.mcwhirter_rate(ne, te, wl.E12_LI))
    res = orc.trace_loss(f, L, qm, st, None, cfg.dt, cfg.max_steps, cfg.detector, variant=1)
    orc.histogram(res, None, cfg.detector, 1)
    ok = (_np(ions.flags) | res["flags"]) == 0
    assert np.array_equal(_np(ions.cell)[ok], res["cell"][ok]) and np.array_equal(_np(ions.steps)[ok].astype(np.uint32), res["steps"][ok])
    assert np.abs(_np(ions.weight)[ok] / res["weight"][ok] - 1).max() < 1e-12
    cr = ok & (res["status"] == 0)
    assert np.abs(_np(ions.hit_w)[cr] - res["w"][cr]).max() < TOL_UW
    try:
        tg.set_option("plane_interp", 1)
        ions, counts, summary = taiga.run_config(tg, cfg, field_loaded=True, rkn_variant=1)
        torch.cuda.synchronize()
    finally:
        tg.set_option("plane_interp", 0)
    ref = orc.run_config(cfg, field=f, variant=1, interp=1)
    compare_groups(ions, ref, "cfg1 printed k3 + bezier")


def _random_scenario(rng):
    """A small random but physically sensible setup: grid size, field kind, species, energy, beam
    direction tilt, divergence, tilted detector plane with a gapped non-uniform matrix, dt, solver,
    E field, plane interpolation."""
    kind = int(rng.integers(0, 3))
    nR, nZ = int(rng.integers(9, 41)), int(rng.integers(12, 61))
    if kind == 0:
        fb = lambda: wl.nodal_field_2d(nR, nZ)
    elif kind == 1:
        nS = int(rng.integers(2, 7))
        fb = lambda: wl.nodal_field_time_slices(nR, nZ, nS, dt_slice=2.0e-7)
    else:
        nS = int(rng.integers(3, 9))
        fb = lambda: wl.nodal_field_ripple(nR, nZ, nS)
    species = wl.MASS_LI7 if rng.random() < 0.6 else wl.MASS_NA23
    energy = float(rng.uniform(20e3, 90e3))
    tilt = rng.normal(0, 0.05, 2)
    axis = np.array([-1.0, tilt[0], tilt[1]]); axis /= np.linalg.norm(axis)
    eT = np.cross([0.0, 0.0, 1.0], axis); eT /= np.linalg.norm(eT)
    eZ = np.cross(axis, eT)
    beam = wl.Beam(species, wl.E_CHARGE, energy, sigma_pos_m=float(rng.uniform(1e-3, 8e-3)),
                   sigma_ang_rad=float(rng.choice([0.0, 1e-3, 4e-3])), origin=(0.78, 0.0, float(rng.uniform(-0.03, 0.03))),
                   axis=tuple(axis), eT=tuple(eT), eZ=tuple(eZ))
    beam.depth_max, beam.z_max = wl.DEPTH_MAX, wl.NORMAL_ZMAX
    # detector plane: normal tilted a few degrees from +X, anywhere the ions pass (most will miss the matrix)
    a, b = rng.normal(0, 0.06, 2)
    nrm = np.array([1.0, a, b]); nrm /= np.linalg.norm(nrm)
    eu = np.cross([0.0, 0.0, 1.0], nrm); eu /= np.linalg.norm(eu)
    ew = np.cross(nrm, eu)
    nu, nw = int(rng.integers(1, 9)), int(rng.integers(1, 9))
    cu, cw = rng.uniform(-0.01, 0.05), rng.uniform(0.02, 0.3)
    edges_u = cu + np.sort(rng.uniform(-0.03, 0.03, 2 * nu)); edges_w = cw + np.sort(rng.uniform(-0.05, 0.05, 2 * nw))
    det = wl.Detector((float(rng.uniform(0.80, 0.84)), 0.0, 0.0), tuple(nrm), tuple(eu), tuple(ew),
                      edges_u[0::2].copy(), edges_u[1::2].copy(), edges_w[0::2].copy(), edges_w[1::2].copy())
    n = int(rng.integers(1, 400))
    groups = [wl.Group(beam, n, int(rng.integers(0, 2 ** 40)), 0, float(rng.uniform(0, 3e-7)) if kind == 1 else 0.0)]
    cfg = wl.Config("rand", fb, groups, float(rng.choice([2e-10, 5e-10, 1e-9, 2e-9])), int(rng.integers(1, 3000)),
                    int(rng.integers(0, 2 ** 62)), 1, det)
    solver = int(rng.choice([0, 0, 0, 1, 2, 3, 4]))
    E = tuple(rng.normal(0, 3e4, 3)) if rng.random() < 0.3 else (0.0, 0.0, 0.0)
    interp = int(rng.random() < 0.3) if (solver <= 1 and not any(E)) else 0
    return cfg, solver, E, interp


@pytest.mark.parametrize("seed", range(16))
def test_random_scenarios_parity(tg, seed):
    """Randomised end-to-end parity: grids, kinds, species, tilted beams and detector planes,
    gapped matrices, step sizes, step limits, solvers, E fields, plane interpolation."""
    from paper_2506_15812_b200 import taiga
    rng = np.random.default_rng(1000 + seed)
    cfg, solver, E, interp = _random_scenario(rng)
    grid, nodal = cfg.field_builder()
    try:
        tg.set_efield(E); tg.set_option("plane_interp", interp)
        ions, counts, summary = taiga.run_config(tg, cfg, rkn_variant=solver)
        torch.cuda.synchronize()
    finally:
        tg.set_efield((0.0, 0.0, 0.0)); tg.set_option("plane_interp", 0)
    f = orc.OracleField(grid, nodal, E=E)
    ref = orc.run_config(cfg, field=f, variant=solver, interp=interp)
    st = compare_groups(ions, ref, "random %d (kind %d solver %d interp %d)" % (seed, grid.kind, solver, interp))
    check_histogram(cfg, ions, counts, summary, ref)
    assert st["flagged"] <= max(3, st["n"] // 50)


def test_philox_against_curand_device_generator():
    """Pin P1 on the GPU box: the oracle's Philox4x32-10 against cuRAND's
    Philox4_32_10 device generator -- a library routine independent of the oracle and of libtaiga --
    and through it the product's seeding (bit-exact against the oracle in the tests above)."""
    import ctypes
    import os
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    lib_path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cuda", "libphilox_curand.so")
    assert os.path.exists(lib_path), "run __graft_entry__.build() (tests/cuda/build.py)"
    lib = ctypes.CDLL(lib_path)
    rng = np.random.default_rng(99)
    n = 257
    sub = rng.integers(0, 2 ** 63, n, dtype=np.uint64); sub[:3] = (0, 1, 2)
    off = rng.integers(0, 2 ** 60, n, dtype=np.uint64); off[:4] = (0, 1, 2 ** 32 - 1, 2 ** 32)
    for seed in (0, 1, 0xDEADBEEFCAFEF00D):
        out = np.zeros((n, 4), dtype=np.uint32)
        rc = lib.philox_curand_words(ctypes.c_ulonglong(seed), sub.ctypes.data_as(ctypes.c_void_p), off.ctypes.data_as(ctypes.c_void_p),
                                     ctypes.c_int(n), out.ctypes.data_as(ctypes.c_void_p))
        assert rc == 0
        for i in range(n):
            ctr = (int(off[i]) & 0xFFFFFFFF, int(off[i]) >> 32, int(sub[i]) & 0xFFFFFFFF, int(sub[i]) >> 32)
            key = (seed & 0xFFFFFFFF, seed >> 32)
            assert tuple(int(x) for x in out[i]) == tuple(int(x) for x in orc.philox4x32_10(ctr, key)), (seed, i)
    # the counter layout of the seeding (O2.1): counter = (i lo, i hi, block j, 0) = cuRAND (offset i, subsequence j)
    i_ion, seed = (1 << 40) + 12345, 7
    U = orc.uniforms(seed, i_ion)
    sub3 = np.array([0, 1, 2], dtype=np.uint64); off3 = np.full(3, i_ion, dtype=np.uint64)
    out = np.zeros((3, 4), dtype=np.uint32)
    assert lib.philox_curand_words(ctypes.c_ulonglong(seed), sub3.ctypes.data_as(ctypes.c_void_p), off3.ctypes.data_as(ctypes.c_void_p),
                                   ctypes.c_int(3), out.ctypes.data_as(ctypes.c_void_p)) == 0
    w = out.reshape(-1)
    for k in range(5):
        nk = (int(w[2 * k]) >> 6) * 2 ** 26 + (int(w[2 * k + 1]) >> 6)
        assert U[k] == (nk + 0.5) * 2.0 ** -52


def test_loss_table_shape_energy_and_species(tg):
    """The form of PAPER.md Table 1 (L147-158) through the product path, on the synthetic profiles:
    percent-level mean loss with a spread over the ionisation depth that is a fraction of the mean, and
    Na+ losing several times more than Li+ (E12 = 47.3 eV against 75.6 eV; the paper: ~20 % against
    ~4.7 %).  The paper's own percentages and their fall with beam energy need the COMPASS profiles and the
    per-energy RENATE-OD ionisation profiles (parity unpinned); with ONE depth profile for all energies the
    faster ions reach hotter, denser plasma and lose more."""
    from paper_2506_15812_b200 import taiga
    cfg = wl.config(1)
    grid, nodal = cfg.field_builder()
    psi0, dpsi, ne, te = wl.loss_profile_inputs()
    psi_nodal = wl.nodal_psi(grid)
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    tg.load_field(grid, nodal)
    n = 8192
    table = {}
    try:
        for species, mass, e12 in (("li", wl.MASS_LI7, wl.E12_LI), ("na", wl.MASS_NA23, wl.E12_NA)):
            tg.load_loss(psi_nodal, psi0, dpsi, ne, te, e12)
            for energy in (40e3, 60e3, 80e3):
                beam = wl.Beam(mass, wl.E_CHARGE, energy)
                beam.depth_max, beam.z_max = wl.DEPTH_MAX, wl.NORMAL_ZMAX
                ions = taiga.Ions(n)
                counts = torch.zeros((1, 8, 8), dtype=torch.int64, device="cuda"); summary = torch.zeros((1, 6), dtype=torch.int64, device="cuda")
                wc = torch.zeros((1, 8, 8), dtype=torch.int64, device="cuda"); ws = torch.zeros((1, 4), dtype=torch.int64, device="cuda")
                tg.seed_beam(beam, cd, cn, 11, ions)
                tg.trace(ions, wl.E_CHARGE / mass, cfg.dt, 20000, cfg.detector)
                tg.detector_histogram(ions, cfg.detector, 1, counts, summary)
                tg.detector_histogram_weighted(ions, cfg.detector, 1, wc, ws)
                torch.cuda.synchronize()
                mean, std = taiga.loss_statistics(ws)
                assert int(ws[0, 3]) > n // 3                                  # enough plane crossers
                table[species, energy] = (float(mean[0]), float(std[0]))
    finally:
        tg.load_loss(None)
    for species in ("li", "na"):
        m = [table[species, e][0] for e in (40e3, 60e3, 80e3)]
        assert all(1e-3 < x < 0.3 for x in m), (species, m)
        for e in (40e3, 60e3, 80e3):
            assert 0.02 * table[species, e][0] < table[species, e][1] < table[species, e][0]
    for e in (40e3, 60e3, 80e3):
        assert 2.0 < table["na", e][0] / table["li", e][0] < 12.0, table
