"""TEST INFRASTRUCTURE.  Oracle pilot run that freezes the detector centres (reading A10,
SURVEY.md 8(c)): centre = component-wise median (T, Z) of plane-crossing ions, rounded to
0.1 mm.  Calls only oracle/ and the input generators; writes tests/golden/detector_centres.txt.
The values are then copied by hand into workloads.DETECTOR_CENTRES and never changed.

    python oracle/freeze_detector_centres.py [n_pilot_ions_per_group]
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, HERE)
sys.path.insert(0, os.path.dirname(HERE))

import oracle as orc  # noqa: E402
from paper_2506_15812_b200 import workloads as wl  # noqa: E402


def main():
    n_pilot = int(sys.argv[1]) if len(sys.argv) > 1 else 65536
    lines = ["# detector centres (T, Z) [m] from the oracle pilot (A10); "
             "written by oracle/freeze_detector_centres.py %d" % n_pilot,
             "# key  T_centre  Z_centre  n_pilot  n_crossed  steps_min  steps_p50  steps_max"]
    fields = {}
    for i in (1, 2, 3, 4, 5):
        n = {1: 4096, 4: max(n_pilot // 64, 64)}.get(i, n_pilot)
        cfg = wl.config(i, n_override=n)
        key = cfg.field_builder.__name__ + str(i if i == 1 else 0)
        if key not in fields:
            grid, nodal = cfg.field_builder()
            fields[key] = orc.OracleField(grid, nodal)
        res = orc.run_config(cfg, field=fields[key])
        if cfg.detector is not None:            # one shared detector: pool all groups
            sets = [(cfg.name, cfg.detector, res["groups"])]
        else:
            sets = [("%s_%dkeV" % (cfg.name, round(g.beam.energy_eV / 1e3)), g.detector, [r])
                    for g, r in zip(cfg.groups, res["groups"])]
        for name, det, rs in sets:
            u = np.concatenate([r["u"][r["status"] == 0] for r in rs])
            w = np.concatenate([r["w"][r["status"] == 0] for r in rs])
            st = np.concatenate([r["steps"][r["status"] == 0] for r in rs])
            ntot = sum(len(r["status"]) for r in rs)
            T = round((det.origin[1] + float(np.median(u))) * 1e4) / 1e4
            Z = round((det.origin[2] + float(np.median(w))) * 1e4) / 1e4
            lines.append("%s %.4f %.4f %d %d %d %d %d" % (name, T, Z, ntot, len(u), st.min(),
                                                          int(np.median(st)), st.max()))
            print(lines[-1], flush=True)
    out = os.path.join(os.path.dirname(HERE), "tests", "golden", "detector_centres.txt")
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
