"""Per-phase clocks of the transport kernel (profiling aid; the tables "Per phase" under profiles/).

    python -m paper_2510_24154_b200.phase_clocks [--config C3] [--histories 100000000]

Builds the analysis variant of the library (transport.cu with -DAEPID_PHASE_CLOCK: thread 0 of every CTA reads clock64() around
every phase, counters 10, 11, 16-25 and 27-31 of aepid_read_counters then hold cycles instead of scheduler events), runs one
counting launch of the config and prints, per event class, its share of the phase time, the number of phases and the share of
that time its warps spent inside the phase rather than waiting at the barrier that ends it.  Needs a GPU."""
import argparse
import os
import subprocess
import sys

CODE = r"""
import sys, numpy as np
from gen import make_config
from paper_2510_24154_b200 import Engine
name, n = sys.argv[1], int(float(sys.argv[2]))
cfg = make_config(name)
eng = Engine.for_config(cfg); eng.load_config(cfg)
eng.set_counting(True); eng.simulate(n, cfg["seed"])
c = eng.read_counters().astype(float); eng.close()
tot = c[16:21].sum()
print("%s, %d histories: %d phases, warps busy %.1f %% of the phase time" % (name, n, c[21:26].sum(), 100 * c[10] / c[11]))
for i, k in enumerate(("A source + photon in air", "W Woodcock flights + interactions", "E charged particle in the phantom",
                       "P photon in the EPID", "X charged particle outside the phantom")):
    print("  %-40s %5.1f %% of the time, %7d phases, warps busy %3.0f %%" % (k, 100 * c[16 + i] / tot, c[21 + i], 100 * c[27 + i] / (32 * c[16 + i] + 1)))
"""


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="C3")
    ap.add_argument("--histories", type=float, default=1e8)
    a = ap.parse_args()
    from . import build as b
    lib = b.build_variant("phase_clock", ["-DAEPID_PHASE_CLOCK"])
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, AEPID_LIBRARY=lib, PYTHONPATH=root + os.pathsep + os.environ.get("PYTHONPATH", ""))
    sys.exit(subprocess.call([sys.executable, "-c", CODE, a.config, str(a.histories)], env=env, cwd=root))


if __name__ == "__main__":
    main()
