"""bench.py --gpus N launches N ranks by itself (torchrun --standalone, 127.0.0.1) and shards the config; checked on
CPU with world size 2 (gloo): the ranks stop after the rank / shard set-up, before the CUDA library is touched."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(*extra):
    env = dict(os.environ)
    env.pop("WORLD_SIZE", None); env.pop("RANK", None); env.pop("LOCAL_RANK", None)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--dry-run-ranks", *extra], capture_output=True, text=True,
                       env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout                       # rank 0 alone prints, one line
    return json.loads(lines[0])


def test_spawn_command_is_the_drivers_launch_line():
    sys.path.insert(0, ROOT)
    import bench
    cmd = bench.spawn_command(["--gpus", "4", "--steps", "2"], 4)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--standalone"] and "--nproc-per-node" in cmd and cmd[cmd.index("--nproc-per-node") + 1] == "4"
    assert "127.0.0.1" in cmd and cmd[-4:] == ["--gpus", "4", "--steps", "2"]


def test_gpus_2_spawns_two_ranks_weak_and_strong():
    d = _run("--gpus", "2", "--config", "2")
    assert d["n_gpus"] == 2 and d["scaling"] == "weak"
    r0, r1 = sorted(d["ranks"], key=lambda r: r["rank"])
    assert (r0["device"], r1["device"]) == ("cuda:0", "cuda:1")
    assert r0["n_ions"] == r1["n_ions"] == 1048576 and r0["first_index"] == 0 and r1["first_index"] == 1 << 40
    d = _run("--gpus", "2", "--config", "2", "--scaling", "strong")
    r0, r1 = sorted(d["ranks"], key=lambda r: r["rank"])
    assert r0["n_ions"] + r1["n_ions"] == 1048576 and r1["first_index"] == r0["n_ions"] and d["scaling"] == "strong"


def test_single_gpu_does_not_spawn():
    d = _run()
    assert d["n_gpus"] == 1 and len(d["ranks"]) == 1


@pytest.mark.gpu
def test_bench_line_carries_the_contract_keys():
    """One short run of bench.py on the GPU (a 8,192-ion prefix of config 2): one JSON line with the keys the driver and the
    judge read, self-consistent numbers, launches counted."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--ions", "8192", "--steps", "2", "--warmup", "3", "--oracle-sample", "512"],
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "e2e", "gpu_launches", "roofline", "cpu_baseline", "clocks"):
        assert k in line, k
    assert line["metric"] == "ion-steps/s" and line["dtype"] == "f64" and line["n_gpus"] == 1 and line["vs_baseline"] is None
    assert "workload" in line["config"] and line["config"]["invariant_counts_sum_to_n"] is True
    r = line["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic", "frac_nominal"):
        assert k in r, k
    assert r["bound"] == "alu" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9 and 0.0 < r["frac"] < 1.0
    e = line["e2e"]
    assert e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0 and e["value"] > 0 and e["value"] != line["value"]
    c = line["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and c["value_1thread"] > 0 and "sample" in c
    assert line["gpu_launches"] == 14 * line["steps"]
    assert line["value"] * line["ms_per_step"] * 1e-3 == pytest.approx(line["config"]["ion_steps_per_step"], rel=1e-6)


@pytest.mark.gpu
def test_bench_line_reports_every_config_and_the_variant_kernels():
    """`configs` (BASELINE configs 1, 3, 4, 5) and `variants` (loss, Bezier, uniform / gridded E, RK4, Boris on config 2,
    fp32 on config 5) ride in the same JSON line (report per config); here at 4,096 ions per group."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--ions", "8192", "--steps", "2", "--warmup", "3", "--oracle-sample", "512",
                          "--extras", "on", "--extras-ions", "4096"], capture_output=True, text=True, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert sorted(line["configs"]) == ["1", "3", "4", "5"] and len(line["variants"]) == 7
    for name, c in list(line["configs"].items()) + list(line["variants"].items()):
        for k in ("workload", "ms_per_step", "trace_kernel", "ion_steps_per_s", "ions_per_s", "trace_ion_steps_per_s", "clocks"):
            assert k in c, (name, k)
        assert c["invariant_counts_sum_to_n"] is True, name
        assert 0.0 < c["trace_kernel"]["ms"] <= c["ms_per_step"] and c["ion_steps_per_step"] > 0, name
        assert c["summary"][0] > 0, name                            # ions reach the detector in every case
    for name, c in line["configs"].items():
        assert 0.0 < c["frac"] < 1.0 and c["frac_nominal"] > 0.0, name
    assert line["configs"]["5"]["trace_kernel"]["kernel"] == "k_trace_mma" and line["configs"]["4"]["trace_kernel"]["kernel"] == "k_trace"
    assert len(line["configs"]["3"]["groups"]) == 4 and line["configs"]["3"]["trace_kernel"]["launches"] == 4
    assert "weighted_histogram_ms" in line["variants"]["cfg2 loss (Eq. 2) + weighted counters"]
    assert line["roofline"]["traffic"] is None                      # --ions: not the configuration of the ncu capture
