"""Roofline denominators of this machine, measured by the library's own microkernels (csrc/peak.cu):

    python -m paper_2506_15812_b200.peaks [milliseconds per measurement]

FP64 pipe (DFMA instructions / s), FP64 tensor pipe (DMMA.8x8x4, FMA / s), both interleaved (one datapath: the sum does
not exceed either) and the L1 -> register delivery rate of
256-bit gathers for 1 / 2 / 4 / 32 distinct cells per warp.  bench.py takes the first two live in every run.
"""
import json
import sys

from . import taiga


def measure(ms: float = 50.0, device: int = 0) -> dict:
    tg = taiga.Taiga(device)
    out = {"dfma_instr_per_s": tg.fp64_peak(ms), "dmma_fma_per_s": tg.dmma_peak(ms),
           "dfma_plus_dmma_fma_per_s": tg.mixed_fp64_peak(ms),
           "nominal_fp64_instr_per_s": 148 * 64 * 1.965e9,
           "l1_gather_bytes_per_s": {str(k): tg.l1_gather_peak(ms, k) for k in (1, 2, 4, 32)}}
    tg.close()
    return out


if __name__ == "__main__":
    print(json.dumps(measure(float(sys.argv[1]) if len(sys.argv) > 1 else 50.0)))
