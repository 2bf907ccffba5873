#!/usr/bin/env python
"""Benchmark of the ARCHER-EPID hot path on B200 (contract: see the task statement / DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C1] [--impl ours|reference]

A step = one pass of the whole hot path over one batch of synthetic input:
reset tallies -> simulate(n histories) -> fold the B batches into mean / sigma -> radiological-thickness map
and k(t,s) response correction.  N=1 workload: BASELINE.json configs[1] (C1: 6 MV open field, 30x30x20 cm water at
2.5 mm, 4-layer EPID 512x384, coupled physics, 1e7 histories).  N>1: every rank runs its own block of the global
history range (weak scaling: 1e7 histories per GPU) and one all-reduce of the tally moments per step.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "histories/s on 1 B200; seconds per IMRT field to 1% EPID uncertainty"
UNIT = "histories/s"

# Algorithmic work model of the transport kernel: thread-instructions of the straight-line
# SASS path of each event, times the events per history of the workload (oracle counters, 1e6-history sample).
INSTR_PER_EVENT = {"source": 420, "woodcock": 150, "air": 230, "epid": 170, "interaction": 260,
                   "estep_phantom": 330, "estep_air": 420, "estep_epid": 350}
EVENTS_PER_HISTORY = {
    "C0": {"source": 1, "woodcock": 3.03, "air": 2.00, "epid": 1.39, "interaction": 2.14, "estep_phantom": 0, "estep_air": 0, "estep_epid": 0},
    "C1": {"source": 1, "woodcock": 3.34, "air": 2.01, "epid": 2.50, "interaction": 2.51, "estep_phantom": 9.47, "estep_air": 0.75, "estep_epid": 0.49},
}


# dram__bytes_read.sum + dram__bytes_write.sum of transport_kernel per history, from the committed ncu --set full capture
# (profiles/r01g_README.md: 1.823 GB + 1.676 GB for 1e7 histories of C1); None where no capture exists.
DRAM_BYTES_PER_HISTORY = {"C1": 349.9}


def alg_instr_per_history(name):
    ev = EVENTS_PER_HISTORY.get(name, EVENTS_PER_HISTORY["C1"])
    return float(sum(INSTR_PER_EVENT[k] * v for k, v in ev.items()))


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True); self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def build_cfg(name, field=0, mode=None):
    from gen import make_config
    from gen.configs import paper_table1_lut
    cfg = make_config(name, field=field)
    if mode is not None:
        cfg["physics"]["mode"] = int(mode)      # 2: Class II collisions (Moller delta rays, reading A31)
    if cfg.get("lut") is None:
        cfg["lut"] = paper_table1_lut()          # PAPER.md:157-162 Table 1 as the response LUT (C4 brings its own)
    return cfg


# ------------------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """The oracle as it stands, timed on the host cores; each step is a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cfg = build_cfg(args.config, args.field, args.physics_mode)
    procs = os.cpu_count() or 1
    sample = args.ref_histories
    oracle.build()
    for _ in range(args.warmup):
        oracle.run_sharded(cfg, max(sample // 10, procs), cfg["seed"], procs=procs)
    t = []
    for k in range(args.steps):
        t0 = time.perf_counter()
        raw = oracle.run_sharded(cfg, sample, cfg["seed"], first=k * sample, procs=procs)
        o = oracle.Oracle(cfg)                      # K8 of the step: thickness map + LUT on the sample's image
        dose = raw["epid_sum"] / raw["ledger"][6]
        o.apply_lut(cfg["lut"], dose, o.tmap(), o.field_size())
        t.append(time.perf_counter() - t0)
    ms = 1e3 * float(np.mean(t))
    val = sample / (ms * 1e-3)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "%s (BASELINE.json configs[%s])" % (args.config, args.config[1:]), "histories_per_step": sample,
                       "note": "bounded sample of the workload per step"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": procs, "kind": "oracle",
                             "sample": "%d histories of %s per step, %d processes over disjoint history ranges" % (sample, args.config, procs)},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2510_24154_b200 import Engine, load_library
    from paper_2510_24154_b200 import parallel

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    load_library()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    cfg = build_cfg(args.config, args.field, args.physics_mode)
    n = int(args.histories or cfg["n_histories"])
    n_total = n * world
    seed = cfg["seed"]
    lut = cfg["lut"]
    eng = Engine.for_config(cfg, device=local)
    eng.load_config(cfg)

    # device-resident outputs and LUT (inputs already resident in HBM when the timed region starts)
    f32 = lambda shape: torch.empty(shape, dtype=torch.float32, device=dev)
    outs = {"epid_mean": f32((eng.nv, eng.nu)), "epid_sigma": f32((eng.nv, eng.nu)),
            "phantom_mean": f32((eng.nz, eng.ny, eng.nx)), "phantom_sigma": f32((eng.nz, eng.ny, eng.nx))}
    signal = f32((eng.nv, eng.nu)); tmap = f32((eng.nv, eng.nu))
    lut_d = torch.from_numpy(np.ascontiguousarray(lut["lut"], dtype=np.float32)).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)        # > 126 MB L2

    def step(ev=None):
        first = parallel.shard_histories(n_total, rank, world)[0]
        eng.reset_tallies()
        eng.set_history_offset(first)
        if ev: ev[0].record()
        eng.simulate(n, seed)                                            # K1-K7 scoring
        if ev: ev[1].record()
        if world > 1:                                                    # the one exchange step
            g = parallel.global_tallies(eng)
            dose = g["epid_mean"]
        else:
            eng.read_tallies(out=outs)                                   # K7 fold -> mean / sigma on the device
            dose = outs["epid_mean"]
        eng.apply_response_lut(lut_d, lut["t_min"], lut["t_max"], lut["s_min"], lut["s_max"], -1.0,
                               epid_in=dose, signal_out=signal, tmap_out=tmap)   # K8
    launches_per_step = 1 + (2 if world == 1 else 4) + 2                 # transport, folds (or moments + finalize), tmap + lut

    for _ in range(args.warmup):
        step(); flush.zero_()
    torch.cuda.synchronize()
    if world > 1: dist.barrier()
    sampler = ClockSampler(local)
    if rank == 0: sampler.start()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    torch.cuda.synchronize()
    t_wall = time.perf_counter()
    for k in range(args.steps):
        flush.zero_()                                                    # L2 flush between timed iterations (untimed)
        ev[k][2].record()
        step(ev[k])
        ev[k][3].record()
    torch.cuda.synchronize()
    if world > 1: dist.barrier()
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop() if rank == 0 else None
    step_ms = [e[2].elapsed_time(e[3]) for e in ev]
    kern_ms = [e[0].elapsed_time(e[1]) for e in ev]
    tot = torch.tensor([sum(step_ms), sum(kern_ms)], dtype=torch.float64, device=dev)
    if world > 1: dist.all_reduce(tot, op=dist.ReduceOp.MAX)
    total_ms, kernel_ms = float(tot[0]), float(tot[1])
    ms_per_step = total_ms / args.steps
    value = n_total / (ms_per_step * 1e-3)

    # statistical uncertainty U (reading A19) of the last step, native and re-binned to about 2.5-3 mm
    tall = {k: v.cpu().numpy() for k, v in outs.items()} if world == 1 else None
    unc = None
    if tall is not None:
        b, nb = eng.read_batches()
        def U(r):
            B = b.shape[0]
            rb = b.reshape(B, b.shape[1] // r, r, b.shape[2] // r, r).sum(axis=(2, 4)).astype(np.float64)
            N = nb.sum(); mean = rb.sum(0) / N
            var = (nb[:, None, None] * (rb / np.maximum(nb, 1)[:, None, None] - mean) ** 2).sum(0) / ((B - 1) * N)
            k = mean > 0.5 * mean.max()
            return float(np.sqrt(np.mean(var[k] / mean[k] ** 2)))
        # re-binning factor (reading A19): the common divisor of nu and nv whose pixel comes closest to the paper's 2.5 mm
        pitch_mm = 10.0 * float(cfg["epid"]["pitch"])
        r = min((k for k in range(1, 65) if eng.nu % k == 0 and eng.nv % k == 0), key=lambda k: abs(k * pitch_mm - 2.5))
        un, ur = U(1), U(r)
        unc = {"U_native": un, "U_rebinned": ur, "rebin": r, "pixel_mm_native": pitch_mm, "pixel_mm_rebinned": r * pitch_mm,
               "seconds_to_1pct_native": ms_per_step * 1e-3 * (un / 0.01) ** 2, "seconds_to_1pct_rebinned": ms_per_step * 1e-3 * (ur / 0.01) ** 2}

    # e2e: the same step through the C-ABI with HOST buffers, host<->device copies inside the timed region
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    t, ph, ep, s = cfg["tables"], cfg["phantom"], cfg["epid"], cfg["source"]
    hin = {k: pin(t[k]) for k in ("E_grid", "mu_compton", "mu_pe", "mu_pair", "T_grid", "stop_pow", "rad_len")}
    hin.update(density=pin(ph["density"]), material=pin(ph["material"]), E_edges=pin(s["E_edges"]), E_pdf=pin(s["E_pdf"]),
               fluence=pin(s["fluence"]), lut=pin(np.ascontiguousarray(lut["lut"], dtype=np.float32)))
    hout = {k: torch.empty(v.shape, dtype=torch.float32).pin_memory() for k, v in outs.items()}
    hsig = torch.empty((eng.nv, eng.nu), dtype=torch.float32).pin_memory()
    h2d = sum(v.numel() * v.element_size() for v in hin.values())
    d2h = sum(v.numel() * v.element_size() for v in hout.values()) + hsig.numel() * 4

    def e2e_step():
        eng.init_materials(hin["E_grid"], hin["mu_compton"], hin["mu_pe"], hin["mu_pair"], hin["T_grid"], hin["stop_pow"], hin["rad_len"])
        eng.set_class2(t["electrons_per_gram"])                          # [n_mat] floats, input of physics mode 2
        eng.load_phantom(ph["spacing"], ph["origin"], hin["density"], hin["material"])
        eng.load_epid_layers(ep["thickness"], ep["material"], ep["density"], ep["scored"], ep["sid"], ep["nu"], ep["nv"], ep["pitch"])
        eng.load_source(s["src_pos"], s["beam_axes"], hin["E_edges"], hin["E_pdf"], s["f_pitch"], s["f_plane_dist"], hin["fluence"])
        eng.set_history_offset(parallel.shard_histories(n_total, rank, world)[0])
        eng.simulate(n, seed)
        eng.read_tallies(out=hout)
        eng.apply_response_lut(hin["lut"], lut["t_min"], lut["t_max"], lut["s_min"], lut["s_max"], -1.0, epid_in=None,
                               signal_out=hsig, tmap_out=None, want_tmap=False)
    e2e_step()
    torch.cuda.synchronize()
    if world > 1: dist.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2e_steps = 1 if args.profile else max(1, min(args.steps, 5))
    e0.record()
    for _ in range(e2e_steps):
        e2e_step()
    e1.record(); torch.cuda.synchronize()
    e2e_ms = torch.tensor([e0.elapsed_time(e1) / e2e_steps], dtype=torch.float64, device=dev)
    if world > 1: dist.all_reduce(e2e_ms, op=dist.ReduceOp.MAX)
    e2e_val = n_total / (float(e2e_ms[0]) * 1e-3)

    if rank != 0:
        if world > 1: dist.destroy_process_group()
        return

    # roofline of the dominant kernel (transport): issue-bound, DESIGN.md "Roofline"
    peaks, which = measured_peaks()
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    peak_ginstr = sm_count * 4 * 32 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e9
    alg = alg_instr_per_history(args.config)
    achieved = alg * n / (kernel_ms / args.steps * 1e-3) / 1e9
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_ginstr, "unit": "Gthread-instr/s", "frac": achieved / peak_ginstr,
                "traffic": DRAM_BYTES_PER_HISTORY.get(args.config) and DRAM_BYTES_PER_HISTORY[args.config] * n, "kernel": "transport_kernel", "kernel_ms_per_launch": kernel_ms / args.steps,
                "alg_thread_instr_per_history": alg, "peak_source": "%s sm_max_mhz x %d SMs x 4 schedulers x 32 lanes" % (which, sm_count),
                "hbm_gbs_peak": peaks.get("hbm_gbs")}

    # CPU baseline: the oracle as it stands on the host cores, bounded sample
    import oracle
    procs = os.cpu_count() or 1
    oracle.build()
    oracle.run_sharded(cfg, procs * 100, seed, procs=procs)              # fork / page-in warm-up
    ns = 10_000 if args.profile else args.cpu_sample
    t0 = time.perf_counter()
    oracle.run_sharded(cfg, ns, seed, procs=procs)
    dt = time.perf_counter() - t0
    cpu = {"value": ns / dt, "unit": UNIT, "cores": procs, "kind": "oracle",
           "sample": "first %d histories of %s, %d processes over disjoint history ranges (%.1f s wall)" % (ns, args.config, procs, dt)}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": "%s (BASELINE.json configs[%s])%s" % (args.config, args.config[1:], " field %d" % args.field if args.config == "C4" else ""), "histories_per_gpu_per_step": n,
                       "n_batches": eng.n_batches, "physics_mode": int(cfg["physics"]["mode"]), "l2": "flushed between timed steps (256 MiB write)",
                       "parallelism": "history-range sharding x%d, one all-reduce of tally moments per step" % world if world > 1 else "single GPU"},
            "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": float(e2e_ms[0])},
            "gpu_launches": launches_per_step * args.steps,
            "uncertainty": unc, "wall_s_timed_region": t_wall,
            "context": {"paper": "~90 s per 1e9-history IMRT field on 1x RTX 3090 (PAPER.md:127, 202), ~1.1e7 histories/s, fuller physics"}}
    print(json.dumps(line))
    if world > 1: dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C1", choices=["C0", "C1", "C2", "C3", "C4"])
    ap.add_argument("--physics-mode", type=int, default=None, choices=[0, 1, 2, 3], help="override the physics mode (2: Class II collisions, 3: + bremsstrahlung)")
    ap.add_argument("--field", type=int, default=0, help="which of C4's 25 IMRT fields (seeds per reading A23)")
    ap.add_argument("--histories", type=int, default=0, help="histories per GPU per step (default: the config's)")
    ap.add_argument("--cpu-sample", type=int, default=1_000_000, help="oracle histories timed for cpu_baseline")
    ap.add_argument("--ref-histories", type=int, default=400_000, help="oracle histories per step of --impl reference")
    ap.add_argument("--profile", action="store_true", help="short run for ncu: one e2e step, tiny cpu_baseline sample (numbers are not bench values)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
