#!/usr/bin/env python
"""Writes tests/golden/oracle_<case>.npz: high-statistics runs of the CPU oracle (oracle/, nothing else) on the full-size
configs C2, C3 and five fields of C4 (BASELINE.json:configs[2..4]).  The GPU parity tests at full size
(tests/test_gpu_full_size.py) compare the CUDA path with these; tests/test_oracle_goldens.py (no GPU) checks that the
stored numbers still agree with the oracle as it stands and that the seeded inputs have not changed.

    python tests/golden/make_oracle_goldens.py [--procs P] [--only C3,C4_07] [--scale 1.0]

No value in these files comes from the CUDA path.  Inputs: gen.make_config (seeded).  What is stored
per case (raw accumulators of the history-by-history estimator; float64):
  n, seed                 histories [0, n) of that simulation seed
  rb, rb_sum, rb_sq       EPID image re-binned by rb x rb pixels: sum and sum of squares over histories
  ledger, ledger_sq       the six energy channels: sum and sum of squares over histories
  pb, pc_idx, pc_sum, pc_sq   phantom on blocks of pb = (bx, by, bz) voxels, only blocks above 2 % of the maximum: flat
                          block index, sum, sum of squares over histories; pc_shape = block grid
  dd_runs                 depth dose (phantom summed over the two axes across the beam) of K independent sub-runs [K][n_depth]
  counters                the oracle's event counters
  input_sha256            hash of the phantom, source and table arrays the run was made with
"""
import argparse
import hashlib
import multiprocessing as mp
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import oracle                      # noqa: E402
from gen import make_config        # noqa: E402

# case -> (config, field, histories, EPID re-binning, phantom block)
CASES = {
    "C2": ("C2", 0, 200_000_000, 8, (4, 4, 2)),
    "C3": ("C3", 0, 200_000_000, 8, (8, 8, 4)),
    "C4_00": ("C4", 0, 50_000_000, 16, (4, 4, 2)),       # 11.9 cm field
    "C4_04": ("C4", 4, 50_000_000, 8, (4, 4, 2)),        # the smallest field size of the 25 (3.0 cm)
    "C4_07": ("C4", 7, 50_000_000, 8, (4, 4, 2)),        # 4.2 cm
    "C4_17": ("C4", 17, 50_000_000, 16, (4, 4, 2)),      # the largest (18.6 cm)
    "C4_21": ("C4", 21, 50_000_000, 16, (4, 4, 2)),      # 9.4 cm
}
K_SUB = 8


def input_hash(cfg):
    h = hashlib.sha256()
    for grp, keys in (("tables", ("E_grid", "mu_compton", "mu_pe", "mu_pair", "T_grid", "stop_pow", "rad_len")),
                      ("phantom", ("spacing", "origin", "density", "material")),
                      ("epid", ("thickness", "material", "density", "scored")),
                      ("source", ("src_pos", "beam_axes", "E_edges", "E_pdf", "fluence"))):
        for k in keys:
            h.update(np.ascontiguousarray(cfg[grp][k]).tobytes())
    h.update(repr((cfg["epid"]["sid"], cfg["epid"]["nu"], cfg["epid"]["nv"], cfg["epid"]["pitch"], cfg["source"]["f_pitch"],
                   cfg["source"]["f_plane_dist"], sorted(cfg["physics"].items()))).encode())
    return h.hexdigest()


def depth_axes(cfg):
    """Axes of phantom[nz][ny][nx] to sum over for the depth dose: the beam runs along grid y (C2-C4) or z (C0, C1)."""
    return (0, 2) if cfg["source"]["beam_axes"].reshape(3, 3)[2][1] != 0 else (1, 2)


_CFG = None
_OPTS = None


def _work(job):
    first, n = job
    global _ORC
    try:
        o = _ORC
    except NameError:
        o = None
    if o is None:                                  # one oracle context per worker process: the phantom is loaded once
        o = oracle.Oracle(_CFG)
        o.set_options(rebin=_OPTS["rb"], want_phantom_sq=False)
        o.set_phantom_rebin(*_OPTS["pb"])
        globals()["_ORC"] = o
    o.reset()
    o.run(first, n, _OPTS["seed"])
    r = o.read()
    return {"rb_sum": r["rb_sum"], "rb_sq": r["rb_sq"], "pc_sum": r["pc_sum"], "pc_sq": r["pc_sq"], "ledger": r["ledger"],
            "ledger_sq": r["ledger_sq"], "dd": r["phantom_sum"].sum(axis=_OPTS["dd_axes"]), "counters": r["counters"].astype(np.float64)}


def run_case(name, procs, scale):
    global _CFG, _OPTS
    cname, field, n, rb, pb = CASES[name]
    n = int(n * scale)
    cfg = make_config(cname, field=field)
    _CFG, _OPTS = cfg, {"rb": rb, "pb": pb, "seed": cfg["seed"], "dd_axes": depth_axes(cfg)}
    per = n // (K_SUB * procs)
    n = per * K_SUB * procs
    t0 = time.time()
    oracle.build()
    tot, dd_runs = None, []
    with mp.get_context("fork").Pool(procs) as pool:
        for k in range(K_SUB):
            jobs = [((k * procs + j) * per, per) for j in range(procs)]
            parts = pool.map(_work, jobs)
            sub = {key: sum(p[key] for p in parts) for key in parts[0]}
            dd_runs.append(sub["dd"] / (per * procs))
            tot = sub if tot is None else {key: tot[key] + sub[key] for key in tot}
            print("  %s sub-run %d/%d, %.0f s" % (name, k + 1, K_SUB, time.time() - t0), flush=True)
    keep = np.nonzero(tot["pc_sum"].ravel() > 0.02 * tot["pc_sum"].max())[0]
    out = os.path.join(HERE, "oracle_%s.npz" % name)
    np.savez_compressed(out, n=np.int64(n), seed=np.int64(cfg["seed"]), rb=np.int64(rb), rb_sum=tot["rb_sum"], rb_sq=tot["rb_sq"],
                        ledger=tot["ledger"], ledger_sq=tot["ledger_sq"], pb=np.array(pb), pc_shape=np.array(tot["pc_sum"].shape),
                        pc_idx=keep.astype(np.int64), pc_sum=tot["pc_sum"].ravel()[keep], pc_sq=tot["pc_sq"].ravel()[keep],
                        dd_runs=np.array(dd_runs), counters=tot["counters"], input_sha256=np.array(input_hash(cfg)),
                        wall_s=np.float64(time.time() - t0), procs=np.int64(procs))
    print("%s: %d histories in %.0f s (%.3g histories/s on %d processes) -> %s (%d KB)" %
          (name, n, time.time() - t0, n / (time.time() - t0), procs, out, os.path.getsize(out) // 1024), flush=True)


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--procs", type=int, default=max(1, (os.cpu_count() or 2) - 1))
    ap.add_argument("--only", default="")
    ap.add_argument("--scale", type=float, default=1.0, help="multiply every history count (quick trial runs)")
    a = ap.parse_args()
    for case in (a.only.split(",") if a.only else CASES):
        run_case(case, a.procs, a.scale)
