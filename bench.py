#!/usr/bin/env python
"""bench.py -- whole hot path (a1 field precompute -> a2 seeding -> a3/a4 RKN trace -> a5
histogram) of BASELINE.json config 2 (1,048,576 7Li+ ions, 257x513 grid) on N GPUs of one node.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2] [--scaling weak|strong]

With --gpus N > 1 and no torchrun environment (WORLD_SIZE unset) it re-executes itself under
`python -m torch.distributed.run --standalone --nproc-per-node N`, one rank per GPU (rank r on cuda:r).

Prints ONE JSON line (rank 0).  `value` = ion-steps/s with inputs resident in HBM; `e2e` = the
same through the C ABI with HOST buffers (pinned nodal field H2D + counter D2H inside the timed
region); `roofline` = the trace kernel against the FP64 issue rate measured live by a
register-resident DFMA microkernel; `cpu_baseline` = the oracle timed on the host cores on a
bounded prefix sample.  --impl reference times the oracle itself (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# FP64-pipe instructions per ion-step of the classical RKN step on a 2-D bicubic field
# (3 field evaluations x 61 + 4 cross products x 6 + stage/Eq.5/plane 45).
ALG_FP64_INSTR_PER_ION_STEP = {0: 252.0, 1: 402.0, 2: 840.0}
# roofline.traffic (dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel at the FULL size of the
# config) is not measured by this run: it is read from profiles/traffic.json, which names the `ncu --set full` capture each
# figure comes from and the hash of the kernel sources it was taken at (csrc_hash below); any later change under csrc/
# makes the figure stale and the line prints traffic = null.
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")


def csrc_hash():
    """sha256 (first 16 hex digits) over the names and contents of paper_2506_15812_b200/csrc/*.{cu,cuh,h}."""
    import glob
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2506_15812_b200", "csrc")
    for f in sorted(glob.glob(os.path.join(d, "*"))):
        if f.endswith((".cu", ".cuh", ".h")):
            h.update(os.path.basename(f).encode())
            h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(config, default_run):
    """(bytes per launch | None, source string | None) for `config` at its default launch configuration."""
    if not default_run:
        return None, "not the configuration the capture was taken in (options / size / detector / solver changed)"
    try:
        ent = json.load(open(TRAFFIC_JSON))["configs"].get(str(config))
    except (OSError, ValueError, KeyError):
        ent = None
    if not ent:
        return None, "no ncu --set full capture recorded for config %d in profiles/traffic.json" % config
    if ent.get("csrc_hash") != csrc_hash():
        return None, "stale: %s was taken at csrc hash %s, the sources are now %s" % (ent.get("capture"), ent.get("csrc_hash"), csrc_hash())
    return float(ent["dram_bytes_per_launch"]), "per launch, from the ncu --set full capture in %s (not measured by this run)" % ent["capture"]


NOMINAL_FP64_INSTR_PER_S = 148 * 64 * 1.965e9      # B200: 148 SMs x 64 FP64 lanes x 1965 MHz
# kinds 1 and 2 are bound by the L1 -> register delivery of the gathered coefficients:
# bytes per ion-step = 3 evaluations x (384: slice difference, kind 1 | 1536: tricubic cell, kind 2; fp32 halves it)
ALG_L1_BYTES_PER_ION_STEP = {1: 1152.0, 2: 4608.0}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--ions", type=int, default=0, help="override ions per group (debug)")
    ap.add_argument("--oracle-sample", type=int, default=131072)
    ap.add_argument("--solver", type=int, default=0, help="0 RKN (default, the metric), 1 printed-k3 RKN, 2 RK4, 3/4 Boris")
    ap.add_argument("--opt", action="append", default=[], help="key=value for taiga_set_option")
    ap.add_argument("--detector", default="config", choices=["config", "gapped"],
                    help="gapped: the config's matrix with non-uniform segments and gaps (PAPER.md L330; binary-search path of a5)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank traces the config's ions (default), strong = the config's ions are split")
    ap.add_argument("--oracle-full", action="store_true", help="time the oracle ONCE on the full config (16 threads and 1 thread on a prefix) and exit")
    ap.add_argument("--extras", default="auto", choices=["auto", "on", "off"],
                    help="configs 1, 3, 4, 5 and the variant kernels in the same line (auto: on for the default line on one GPU)")
    ap.add_argument("--extras-ions", type=int, default=0, help="ions per group for the extras (default: full size)")
    ap.add_argument("--csrc-hash", action="store_true", help="print the hash of the kernel sources that profiles/traffic.json entries carry, and exit")
    ap.add_argument("--dry-run-ranks", action="store_true", help="stop after the rank / shard set-up (CPU test of the launch path)")
    return ap.parse_args()


def spawn_command(argv, n):
    """The command that runs this script as n ranks of one node (what the driver runs for N > 1)."""
    return [sys.executable, "-m", "torch.distributed.run", "--standalone", "--nnodes=1", "--nproc-per-node", str(n),
            "--local-addr", "127.0.0.1", os.path.abspath(__file__)] + list(argv)


def maybe_spawn(args):
    """--gpus N > 1 without a torchrun environment: become the launcher of N ranks."""
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        env = dict(os.environ, MASTER_ADDR="127.0.0.1")
        sys.exit(subprocess.run(spawn_command(sys.argv[1:], args.gpus), env=env).returncode)


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            time.sleep(0.05)

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
                for nme, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nme)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_run(cfg_index, sample, nthreads=0, solver=0):
    """The oracle as it stands on a prefix sample (sample = 0: the full config); returns (ion_steps, ions, seconds, threads, cfg)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import oracle as orc
    from paper_2506_15812_b200 import workloads as wl
    cfg = wl.config(cfg_index, n_override=max(sample // len(wl.config(cfg_index).groups), 1) if sample else None)
    t0 = time.perf_counter()
    res = orc.run_config(cfg, nthreads=nthreads, variant=solver)
    dt = time.perf_counter() - t0
    steps = sum(int(g["steps"].astype("int64").sum()) for g in res["groups"])
    return steps, cfg.n_ions, dt, (nthreads or orc.max_threads()), cfg


def main_oracle_full(args):
    """the oracle timed once on the FULL config on all host threads, and on one thread on a
    prefix (numbers kept in profiles/; not part of the per-run bench line)."""
    s, n, dt, cores, cfg = oracle_run(args.config, 0, solver=args.solver)
    s1, n1, dt1, _, _ = oracle_run(args.config, min(args.oracle_sample, 16384), nthreads=1, solver=args.solver)
    print(json.dumps({"oracle_full": {"config": args.config, "ions": n, "ion_steps": s, "seconds": dt, "cores": cores,
                                      "ion_steps_per_s": s / dt, "ions_per_s": n / dt,
                                      "one_thread": {"ions": n1, "seconds": dt1, "ion_steps_per_s": s1 / dt1}}}))


def main_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    for _ in range(min(args.warmup, 1)):
        oracle_run(args.config, max(args.oracle_sample // 8, 1024), solver=args.solver)
    tot_steps, tot_t, n_ions, cores = 0, 0.0, 0, 1
    for _ in range(args.steps):
        s, n, dt, cores, cfg = oracle_run(args.config, args.oracle_sample, solver=args.solver)
        tot_steps += s; tot_t += dt; n_ions = n
    v = tot_steps / tot_t
    sample = "first %d ions of config %d (prefix sample; identical ions, Philox counter = ion index), whole path a1-a5 per step" % (n_ions, args.config)
    print(json.dumps({
        "impl": "reference", "metric": "ion-steps/s", "value": v, "unit": "ion-steps/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg%d prefix sample of %d ions" % (args.config, n_ions)},
        "cpu_baseline": {"value": v, "unit": "ion-steps/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "ion-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "ions_per_s": n_ions * args.steps / tot_t}))


def alg_instr(kind, solver):
    """The method's FP64 instructions per ion-step; other solvers: 4 (solver 1, 2) / 1 (Boris) evaluations."""
    alg = ALG_FP64_INSTR_PER_ION_STEP[kind]
    if solver:
        per_eval = (alg - 69.0) / 3.0
        alg = {1: 4 * per_eval + 69.0, 2: 4 * per_eval + 75.0, 3: per_eval + 45.0, 4: per_eval + 45.0}[solver]
    return alg


def measure_case(local, peak_dfma, icfg, ions_override=0, solver=0, opts=(), setup=None, weighted=False, steps=2, warmup=1):
    """One more workload beside the headline: the whole path a1-a5 of BASELINE config `icfg` at full size (nodal field
    resident in HBM), `warmup` untimed steps, then `steps` timed ones with CUDA events around the step and around the trace
    kernel(s), an L2 flush in between, clocks sampled meanwhile.  Own context, so no option leaks into the next case.
    `setup(tg, grid, wl)` loads what the variant needs (loss model, E) after the first load_field."""
    import numpy as np
    import torch
    from paper_2506_15812_b200 import taiga, workloads as wl
    dev = "cuda:%d" % local
    cfg = wl.config(icfg, n_override=ions_override or None)
    grid, nodal = cfg.field_builder()
    nodal_dev = [torch.from_numpy(np.ascontiguousarray(c)).to(dev) for c in nodal]
    tg = taiga.Taiga(local)
    for k, v in opts:
        tg.set_option(k, v)
    tg.load_field(grid, nodal_dev)
    if setup:
        setup(tg, grid, wl)
    ions = taiga.Ions(cfg.n_ions, dev)
    det0 = cfg.detector or cfg.groups[0].detector
    counts = torch.zeros((cfg.n_hist, det0.nw, det0.nu), dtype=torch.int64, device=dev)
    summary = torch.zeros((cfg.n_hist, 6), dtype=torch.int64, device=dev)
    wcounts, wsummary = torch.zeros_like(counts), torch.zeros((cfg.n_hist, 4), dtype=torch.int64, device=dev)
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step():
        marks = [ev() for _ in range(5)]
        marks[0].record()
        tg.load_field(grid, nodal_dev)
        if setup:
            setup(tg, grid, wl)
        counts.zero_(); summary.zero_(); wcounts.zero_(); wsummary.zero_()
        off, spans = 0, []
        for g in cfg.groups:
            v = ions.view(off, off + g.n_ions)
            tg.seed_beam(g.beam, cd, cn, cfg.seed, v, g.first_index, g.group, g.t0)
            spans.append((v, g)); off += g.n_ions
        whole = [(ions, cfg.groups[0], cfg.detector)] if cfg.detector is not None else [(v, g, g.detector) for v, g in spans]
        marks[1].record()
        for v, g, d in whole:
            tg.trace(v, g.beam.charge_C / g.beam.mass_kg, cfg.dt, cfg.max_steps, d, solver)
        marks[2].record()
        for v, g, d in whole:
            tg.detector_histogram(v, d, cfg.n_hist, counts, summary)
        marks[3].record()
        if weighted:
            for v, g, d in whole:
                tg.detector_histogram_weighted(v, d, cfg.n_hist, wcounts, wsummary)
        marks[4].record()
        return marks

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    t_step = t_trace = t_hist = t_whist = 0.0
    for _ in range(steps):
        flush.zero_()
        torch.cuda.synchronize()
        m = step()
        torch.cuda.synchronize()
        t_step += m[0].elapsed_time(m[4]); t_trace += m[1].elapsed_time(m[2]); t_hist += m[2].elapsed_time(m[3]); t_whist += m[3].elapsed_time(m[4])
    sampler.stop_flag = True
    ion_steps = int(ions.steps.to(torch.int64).sum().item())
    ok = int(summary[:, :5].sum().item()) == cfg.n_ions
    t_step, t_trace, t_hist, t_whist = (t / steps for t in (t_step, t_trace, t_hist, t_whist))
    kind = grid.kind
    o = dict(opts)
    f32 = o.get("precision") == 32
    mma = kind != 0 and not f32 and (o.get("mma", -1) == 1 or (o.get("mma", -1) == -1 and kind == 2))
    rate = ion_steps / (t_trace * 1e-3)
    alg = alg_instr(kind, solver)
    out = {"workload": "BASELINE config %d (%s): %d ions, grid %dx%dx%d kind %d, dt=%g, max_steps=%d" % (
               icfg, cfg.name, cfg.n_ions, grid.nR, grid.nZ, grid.nS, kind, cfg.dt, cfg.max_steps),
           "steps": steps, "warmup": warmup, "ms_per_step": t_step, "ion_steps_per_step": ion_steps,
           "trace_kernel": {"ms": t_trace, "launches": len(cfg.groups) if cfg.detector is None else 1,
                            "kernel": "k_trace_mma" if mma else "k_trace"},
           "ion_steps_per_s": ion_steps / (t_step * 1e-3), "ions_per_s": cfg.n_ions / (t_step * 1e-3),
           "trace_ion_steps_per_s": rate, "histogram_ms": t_hist,
           "frac": rate * alg / peak_dfma, "frac_nominal": rate * alg / NOMINAL_FP64_INSTR_PER_S, "alg_fp64_instr_per_ion_step": alg,
           "summary": [int(v) for v in summary.sum(dim=0).tolist()], "invariant_counts_sum_to_n": ok, "clocks": sampler.summary()}
    if weighted:
        out["weighted_histogram_ms"] = t_whist
    if cfg.detector is None:                   # energy scan: per-group share of the steps (the 20 keV group is mostly non-crossers)
        off, per = 0, []
        for g in cfg.groups:
            v = ions.view(off, off + g.n_ions)
            per.append({"energy_eV": g.beam.energy_eV, "ion_steps": int(v.steps.to(torch.int64).sum().item()),
                        "maxsteps_ions": int((v.cell == taiga.CELL_MAXSTEPS).sum().item())})
            off += g.n_ions
        out["groups"] = per
    tg.close()
    del ions, flush, nodal_dev
    torch.cuda.empty_cache()
    return out


def extras(local, peak_dfma, ions_override=0):
    """"configs": the other four BASELINE configs at full size; "variants": the widened kernels on config 2 and the fp32
    evaluation on config 5 (SURVEY.md 8(d) "report per config")."""
    import numpy as np

    def loss(tg, grid, wl):
        psi0, dpsi, ne, te = wl.loss_profile_inputs()
        tg.load_loss(wl.nodal_psi(grid), psi0, dpsi, ne, te, wl.E12_LI)

    def uniform_e(tg, grid, wl):
        tg.set_efield((1.0e4, 0.0, -5.0e3))

    def gridded_e(tg, grid, wl):
        R = np.linspace(grid.Rmin, grid.Rmax, grid.nR)[:, None] * np.ones((1, grid.nZ))
        Z = np.ones((grid.nR, 1)) * np.linspace(grid.Zmin, grid.Zmax, grid.nZ)[None, :]
        tg.load_efield((4.0e4 * np.exp((R - 0.8) / 0.05) - 1.0e4 * 0.56 / R, 6.0e4 * Z, 2.0e4 + 0.0 * R))

    n = ions_override
    configs = {str(i): measure_case(local, peak_dfma, i, n) for i in (1, 3, 4, 5)}
    variants = {
        "cfg2 loss (Eq. 2) + weighted counters": measure_case(local, peak_dfma, 2, n, setup=loss, weighted=True),
        "cfg2 Bezier plane interpolation": measure_case(local, peak_dfma, 2, n, opts=(("plane_interp", 1),)),
        "cfg2 uniform E": measure_case(local, peak_dfma, 2, n, setup=uniform_e),
        "cfg2 gridded E(R,Z)": measure_case(local, peak_dfma, 2, n, setup=gridded_e),
        "cfg2 RK4 (solver 2)": measure_case(local, peak_dfma, 2, n, solver=2),
        "cfg2 Boris-Verlet (solver 3)": measure_case(local, peak_dfma, 2, n, solver=3),
        "cfg5 precision=32": measure_case(local, peak_dfma, 5, n, opts=(("precision", 32),)),
    }
    for k in ("cfg2 loss (Eq. 2) + weighted counters", "cfg2 Bezier plane interpolation", "cfg2 uniform E", "cfg2 gridded E(R,Z)", "cfg5 precision=32"):
        for drop in ("frac", "frac_nominal", "alg_fp64_instr_per_ion_step"):      # no instruction count is claimed for these kernels
            variants[k].pop(drop)
    return configs, variants


def launches_per_step(cfg, kind):
    a1 = 3 + 3 + (1 if kind == 2 else 0)       # 3 second-derivative stencils + 3 assembles [+ phi spline]
    ntrace = 1 if cfg.detector is not None else len(cfg.groups)
    return a1 + len(cfg.groups) + ntrace * (5 + 1) + ntrace      # seeds + (sort 5 + trace 1) + histogram


def main_ours(args):
    import numpy as np
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    from paper_2506_15812_b200 import sharding, workloads as wl
    # weak scaling (default): every rank traces its own cfg.n_ions ions (disjoint Philox counters);
    # strong: the config's ions are split into `world` contiguous index ranges
    cfg = sharding.shard_config(wl.config(args.config, n_override=args.ions or None), rank, world, args.scaling)
    dist = None
    if args.dry_run_ranks:                      # launch / shard logic only: gloo, no CUDA, no library
        import torch.distributed as dist
        if world > 1:
            dist.init_process_group("gloo")
        mine = torch.tensor([rank, local, cfg.groups[0].first_index, cfg.n_ions], dtype=torch.int64)
        allr = [torch.zeros_like(mine) for _ in range(world)]
        if world > 1:
            dist.all_gather(allr, mine)
        else:
            allr = [mine]
        if rank == 0:
            print(json.dumps({"n_gpus": world, "scaling": args.scaling, "dry_run": True,
                              "ranks": [dict(rank=int(a[0]), device="cuda:%d" % int(a[1]), first_index=int(a[2]), n_ions=int(a[3])) for a in allr]}))
        if world > 1:
            dist.destroy_process_group()
        return
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        # rank 0 logs the communicator set-up (transport, NVLS) to stderr, so that a scaling run can be checked against it;
        # stdout stays the one JSON line
        os.environ.setdefault("NCCL_DEBUG", "INFO" if rank == 0 else "WARN")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2506_15812_b200 import taiga
    dev = "cuda:%d" % local
    if args.detector == "gapped":
        if cfg.detector is not None:
            cfg.detector = wl.gapped_detector(cfg.detector)
        for g in cfg.groups:
            if g.detector is not None:
                g.detector = wl.gapped_detector(g.detector)
    grid, nodal = cfg.field_builder()
    nodal_dev = [torch.from_numpy(np.ascontiguousarray(c)).to(dev) for c in nodal]
    nodal_pin = [torch.from_numpy(np.ascontiguousarray(c)).pin_memory() for c in nodal]
    nodal_host = [p.numpy() for p in nodal_pin]                                      # numpy views of the pinned buffers: host pointers for the ABI
    tg = taiga.Taiga(local)
    for kv in args.opt:
        k, v = kv.split("=")
        tg.set_option(k, int(v))
    peak_dfma = tg.fp64_peak(100.0)             # FP64-pipe instructions / s, measured live
    mma_on = grid.kind == 2 and not any(kv.strip() in ("mma=0", "precision=32") for kv in args.opt) or any(kv.strip() == "mma=1" for kv in args.opt)
    mma_on = mma_on and grid.kind != 0
    tg.set_option("stats", 0)                   # no host sync inside taiga_trace while timing
    ions = taiga.Ions(cfg.n_ions, dev)
    det0 = cfg.detector or cfg.groups[0].detector
    counts = torch.zeros((cfg.n_hist, det0.nw, det0.nu), dtype=torch.int64, device=dev)
    summary = torch.zeros((cfg.n_hist, 6), dtype=torch.int64, device=dev)
    counts_pin = torch.zeros(counts.shape, dtype=torch.int64).pin_memory()
    summary_pin = torch.zeros(summary.shape, dtype=torch.int64).pin_memory()
    cd, cn = wl.depth_cdf(), wl.normal_cdf()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    ev = lambda: torch.cuda.Event(enable_timing=True)
    trace_ms, hist_ms = [], []

    def step(host, record=False):
        # e2e: the ABI's own host-buffer path (taiga_coeffs.on_device = 0): the library copies the pinned nodal arrays to
        # the device on its stream and waits for the copy before it returns
        tg.load_field(grid, nodal_host if host else nodal_dev)                           # a1
        counts.zero_(); summary.zero_()
        off, spans = 0, []
        for g in cfg.groups:
            v = ions.view(off, off + g.n_ions)
            tg.seed_beam(g.beam, cd, cn, cfg.seed, v, g.first_index, g.group, g.t0)      # a2
            spans.append((v, g)); off += g.n_ions
        e0, e1 = ev(), ev()
        e0.record()
        if cfg.detector is not None:
            b = cfg.groups[0].beam
            tg.trace(ions, b.charge_C / b.mass_kg, cfg.dt, cfg.max_steps, cfg.detector, args.solver)   # a3 + a4
        else:
            for v, g in spans:
                tg.trace(v, g.beam.charge_C / g.beam.mass_kg, cfg.dt, cfg.max_steps, g.detector, args.solver)
        e1.record()
        if cfg.detector is not None:
            tg.detector_histogram(ions, cfg.detector, cfg.n_hist, counts, summary)       # a5
        else:
            for v, g in spans:
                tg.detector_histogram(v, g.detector, cfg.n_hist, counts, summary)
        e2 = ev(); e2.record()
        sharding.allreduce_counters(dist, counts, summary)                               # exchange step: <= 0.5 MB
        if host:
            counts_pin.copy_(counts, non_blocking=True); summary_pin.copy_(summary, non_blocking=True)
        if record:
            trace_ms.append((e0, e1)); hist_ms.append((e1, e2))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(host):
        for _ in range(max(args.warmup, 3)):
            step(host)
        barrier()
        times = []
        for _ in range(args.steps):
            flush.zero_()                       # L2 flush between timed iterations
            torch.cuda.synchronize()
            if host:
                t0 = time.perf_counter(); step(True); torch.cuda.synchronize(); times.append((time.perf_counter() - t0) * 1e3)
            else:
                a, b = ev(), ev()
                a.record(); step(False, record=True); b.record(); torch.cuda.synchronize()
                times.append(a.elapsed_time(b))
        barrier()
        tot = torch.tensor([sum(times)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(tot, op=dist.ReduceOp.MAX)
        return float(tot.item())

    sampler = ClockSampler(local)
    sampler.start()
    total_ms = timed(False)
    total_ms_e2e = timed(True)
    sampler.stop_flag = True
    ion_steps_rank = int(ions.steps.to(torch.int64).sum().item())
    tsum = torch.tensor([ion_steps_rank, cfg.n_ions], dtype=torch.int64, device=dev)
    if world > 1:
        dist.all_reduce(tsum)
    ion_steps, n_ions = int(tsum[0]), int(tsum[1])
    t_trace = sum(a.elapsed_time(b) for a, b in trace_ms) / len(trace_ms)
    kind = grid.kind
    alg = alg_instr(kind, args.solver)
    achieved = ion_steps_rank * alg / (t_trace * 1e-3)
    traffic = ncu_traffic(args.config, not (args.ions or args.solver or args.opt or args.detector != "config" or world > 1 and args.scaling == "strong"))
    h2d = sum(p.numel() * 8 for p in nodal_pin) + (len(cd) + len(cn)) * 8 * len(cfg.groups) + 4 * (det0.nu + det0.nw) * 8
    d2h = counts.numel() * 8 + summary.numel() * 8
    s_ok = int(summary[:, :5].sum().item()) == n_ions
    out = {
        "metric": "ion-steps/s", "value": ion_steps * args.steps / (total_ms * 1e-3), "unit": "ion-steps/s",
        "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps,
        "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE config %d (%s): %d ions/GPU, grid %dx%dx%d kind %d, dt=%g, max_steps=%d, whole path a1-a5 per step"
                               % (args.config, cfg.name, cfg.n_ions, grid.nR, grid.nZ, grid.nS, kind, cfg.dt, cfg.max_steps)
                               + ("" if not args.solver else ", solver %d" % args.solver),
                   "l2": "256 MiB buffer written between timed iterations (L2 flush)",
                   "ion_steps_per_step": ion_steps, "ions_per_step": n_ions, "invariant_counts_sum_to_n": s_ok},
        "ions_per_s": n_ions * args.steps / (total_ms * 1e-3),
        "trace_kernel": {"ms": t_trace, "ion_steps_per_s": ion_steps_rank / (t_trace * 1e-3)},
        "histogram_kernel": {"ms": sum(a.elapsed_time(b) for a, b in hist_ms) / len(hist_ms), "detector": args.detector,
                             "hits_in_segments": int(summary[:, 0].sum().item()), "hits_in_gaps_or_outside": int(summary[:, 1].sum().item())},
        "e2e": {"value": ion_steps * args.steps / (total_ms_e2e * 1e-3), "unit": "ion-steps/s",
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "ms_per_step": total_ms_e2e / args.steps,
                "timing": "host wall clock around the C-ABI calls; taiga_load_field is given the pinned HOST arrays (on_device = 0: "
                          "its own H2D + wait inside the call), CDF tables and detector edges are host pointers too, counters read back D2H"},
        "gpu_launches": launches_per_step(cfg, kind) * args.steps,
        "roofline": {"bound": "alu", "achieved": 2e-12 * achieved, "peak": 2e-12 * peak_dfma,
                     "unit": "TFLOP/s (FP64 pipe; every FP64 instruction counted as one FMA = 2 flop)",
                     "frac": achieved / peak_dfma,
                     "peak_nominal": 2e-12 * NOMINAL_FP64_INSTR_PER_S, "frac_nominal": achieved / NOMINAL_FP64_INSTR_PER_S,
                     "traffic": traffic[0], "traffic_source": traffic[1],
                     "kernel": "k_trace_mma" if mma_on else "k_trace", "alg_fp64_instr_per_ion_step": alg,
                     "alg": "analytic count of the method's FP64 instructions per ion-step (DESIGN.md section 6), not an executed count",
                     "peak_source": "measured live: register-resident DFMA microkernel, 4 chains with their own operand registers "
                                    "(taiga_measure_fp64_peak); nominal 148 SM x 64 lanes x 1.965 GHz = 18.6e12 instr/s"},
        "clocks": sampler.summary(),
    }
    if mma_on:
        out["roofline"]["dmma_peak"] = 2e-12 * tg.dmma_peak(50.0)
        out["roofline"]["note"] = ("field evaluation on the FP64 tensor pipe (DMMA.8x8x4, same FMA rate as DFMA on B200: dmma_peak); "
                                   "frac counts the method's %d FP64 instructions per ion-step, not the padded tensor work" % int(alg))
    opts = {kv.split("=")[0].strip(): kv.split("=")[1].strip() for kv in args.opt}
    # the kernels that still gather coefficients per lane through L1 (kind 2 with mma=0 / precision=32; kind 1 with the r1 / r2a
    # variants) are reported against the measured L1 delivery rate; the default kernels against the FP64 rate
    gathers = (kind == 2 and not mma_on) or (kind == 1 and not mma_on and opts.get("variant", "0") != "0")
    if gathers and not args.solver:
        f32 = any(kv.strip() == "precision=32" for kv in args.opt)
        l1_peak = tg.l1_gather_peak(50.0, 1)
        l1_bytes = ALG_L1_BYTES_PER_ION_STEP[kind] * (0.5 if f32 else 1.0)
        out["roofline"] = {"bound": "l1", "achieved": 1e-9 * ion_steps_rank * l1_bytes / (t_trace * 1e-3), "peak": 1e-9 * l1_peak,
                           "unit": "GB/s (gathered field coefficients delivered to registers)",
                           "frac": ion_steps_rank * l1_bytes / (t_trace * 1e-3) / l1_peak, "traffic": None, "kernel": "k_trace",
                           "alg_l1_bytes_per_ion_step": l1_bytes, "fp64_frac": achieved / peak_dfma,
                           "peak_source": "measured live: L1-resident 256-bit gather microkernel, all lanes of a warp in one cell "
                                          "(taiga_measure_l1_gather_peak, spread 1: 128 B/clk/SM; 64 with two cells per warp, 32 with four or more)"}
    tg.close()
    default_line = not (args.ions or args.solver or args.opt or args.detector != "config" or args.config != 2)
    if world == 1 and (args.extras == "on" or (args.extras == "auto" and default_line)):
        del ions, flush
        torch.cuda.empty_cache()
        out["configs"], out["variants"] = extras(local, peak_dfma, args.extras_ions)
        out["extras"] = ("configs / variants: each the whole path a1-a5 at %s, 1 warm-up + 2 timed steps (CUDA events, L2 flush between), "
                         "frac against the DFMA rate measured in this run" % ("full size" if not args.extras_ions else "%d ions per group" % args.extras_ions))
    if rank == 0:
        if world == 1:
            s, n, dt, cores, _ = oracle_run(args.config, args.oracle_sample, solver=args.solver)
            s1, n1, dt1, _, _ = oracle_run(args.config, max(args.oracle_sample // 16, 256), nthreads=1, solver=args.solver)
            out["cpu_baseline"] = {"value": s / dt, "unit": "ion-steps/s", "cores": cores, "kind": "oracle",
                                   "ions_per_s": n / dt, "seconds": dt, "value_1thread": s1 / dt1, "seconds_1thread": dt1,
                                   "note": "the oracle is the correctness reference as it stands (-O2, no contraction, 4 field evaluations per step), "
                                           "not a tuned CPU code: the GPU/CPU ratio is not a speed-up claim",
                                   "sample": "first %d ions of config %d (prefix sample, identical ions), whole path a1-a5, OpenMP over ions; "
                                             "value_1thread on the first %d ions" % (n, args.config, n1)}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.csrc_hash:
        print(csrc_hash())
    elif a.oracle_full:
        main_oracle_full(a)
    elif a.impl == "reference":
        main_reference(a)
    else:
        maybe_spawn(a)
        main_ours(a)
