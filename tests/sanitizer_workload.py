#!/usr/bin/env python
"""Small runs of the CUDA path for the checked build and for compute-sanitizer:

    AEPID_LIBRARY=paper_2510_24154_b200/libaepid_checked.so python tests/sanitizer_workload.py   (tests/test_gpu_checked_build.py)
    compute-sanitizer --tool memcheck  python tests/sanitizer_workload.py
    compute-sanitizer --tool racecheck python tests/sanitizer_workload.py

(compute-sanitizer is closed on the GPU pool this was developed on, profiles/r02_README.md; the checked build is what ran.)

A C0-shaped photon-only run, a small coupled run with room for only 256 live particles per CTA (the parking / head-room-credit
paths of the scheduler), modes 3 and 4, the collimation stage, the fold, the response post-pass and the analysis kernels.  No
oracle here: the sanitizer checks memory accesses and shared-memory hazards, the parity tests check the numbers."""
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from gen import make_config, head_config                    # noqa: E402
from gen.configs import paper_table1_lut                    # noqa: E402
from paper_2510_24154_b200 import Engine                    # noqa: E402


def run(cfg, n, live=0, tag=""):
    eng = Engine.for_config(cfg, n_batches=4, max_live_per_cta=1024)
    eng.load_config(cfg)
    eng.set_live_limit(live)
    eng.simulate(n, 3)
    r = eng.read_tallies()
    L = r["ledger"]
    bal = abs(L[1] + L[2] + L[3] + L[4] + L[5] - L[0]) / L[0]
    assert L[7] == 0 and bal < 1e-6, (tag, L[7], bal)
    lut = paper_table1_lut()
    sig, tmap = eng.apply_response_lut(lut["lut"], lut["t_min"], lut["t_max"], lut["s_min"], lut["s_max"], -1.0)
    up = eng.upsample(r["epid_mean"], 96, 96)
    eng.gamma_index(up, up * 1.01, 0.3, 0.03, 0.3)
    eng.roi_mean(1.0)
    print("%-28s %7d histories, ledger balance %.1e" % (tag, n, bal), flush=True)
    eng.close()


if __name__ == "__main__":
    n = int(sys.argv[1]) if len(sys.argv) > 1 else 20000
    run(make_config("C0", shrink=4), n, tag="C0 photon-only")
    c1 = make_config("C1", shrink=8)
    run(c1, n, live=256, tag="C1 coupled, live limit 256")
    for mode in (3, 4):
        c1["physics"]["mode"] = mode
        run(c1, n, live=256, tag="C1 mode %d, live limit 256" % mode)
    run(head_config(field=7, shrink=8, n_ps1=20000), 4 * n, tag="C4 field 7, collimation stage")
    print("sanitizer workload done")
