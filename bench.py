#!/usr/bin/env python
"""Benchmark of the ARCHER-EPID hot path on B200 (contract: see the task statement / DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--impl ours|reference]

A step = one pass of the whole hot path over one batch of synthetic input:
reset tallies -> simulate(n histories) -> fold the B batches into mean / sigma -> radiological-thickness map
and k(t,s) response correction.  N=1 workload: BASELINE.json configs[3] (C3: 9-segment IMRT field on the
512 x 512 x 200 synthetic patient, 4-layer EPID 1024 x 768, coupled physics, 1e9 histories: the config the metric's
"seconds per IMRT field to 1 %" is quoted on and the largest single-GPU one).  N>1: every rank runs its own block of
the global history range (weak scaling: the config's histories per GPU) and one all-reduce of the tally moments per step.
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

# Algorithmic work model of the transport kernel (from SURVEY.md 8(d) "Algorithmic work per unit"):
# thread-instructions the METHOD needs per event, the middle of the survey's ranges (150-250 per photon flight, 120-200
# per electron step) plus what it implies for the two event kinds the survey gives no range for (a Klein-Nishina /
# photoelectric / pair interaction with its Philox block; the source sample: one Philox block, two table searches, one
# direction).  These are NOT this kernel's instruction counts: those are measured by ncu (profiles/) and reported beside.
ALG_UNIT_COST = {"flight": 200.0, "electron_step": 160.0, "interaction": 200.0, "source": 150.0}


def events_per_history(counters, n):
    """Event mix of the workload from the library's own counters (aepid_read_counters) of an untimed counting launch."""
    c = [float(x) for x in counters]
    return {"flight": (c[0] + c[1] + c[2]) / n, "electron_step": (c[6] + c[7] + c[8]) / n, "interaction": (c[3] + c[4] + c[5]) / n,
            "source": 1.0, "woodcock_flights": c[0] / n, "air_flights": c[1] / n, "epid_flights": c[2] / n,
            "esteps_phantom": c[6] / n, "esteps_air": c[7] / n, "esteps_epid": c[8] / n, "kn_trials": c[12] / n, "charged_tracks": c[14] / n}


def alg_instr_per_history(ev):
    return float(sum(ALG_UNIT_COST[k] * ev[k] for k in ALG_UNIT_COST))


# ncu captures committed under profiles/ (one `ncu --set full` launch of transport_kernel per config, never a bench value):
# dram__bytes_read.sum + dram__bytes_write.sum per history, executed warp-instructions per history, active lanes per
# warp-instruction, issue-slot utilisation.  None where no capture of the current kernel exists.
NCU_CAPTURES = {}
try:
    import csv as _csv
    with open(os.path.join(ROOT, "profiles", "ncu_transport_summary.csv")) as _f:
        for _r in _csv.DictReader(_f):
            NCU_CAPTURES[_r["key"]] = {k: (float(v) if k not in ("key", "report") else v) for k, v in _r.items()}
except Exception:
    pass


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


def build_cfg(name, field=0, mode=None, collimator=False):
    from gen import make_config, head_config
    from gen.configs import paper_table1_lut
    if collimator and name != "C4":
        raise SystemExit("--collimator goes with --config C4 (the field's apertures become jaws and leaves)")
    cfg = head_config(field=field) if collimator else make_config(name, field=field)   # NEXT-3: Phase Space 1 + jaws / MLC instead of the fluence map
    if mode is not None:
        cfg["physics"]["mode"] = int(mode)      # 2: Class II collisions (Moller delta rays, reading A31)
        if int(mode) == 4:
            cfg["physics"]["f_E"] = 0.2         # reading A38: the multi-voxel step loses 20 % of the energy (as in the parity tests)
    if cfg.get("lut") is None:
        cfg["lut"] = paper_table1_lut()          # PAPER.md:157-162 Table 1 as the response LUT (C4 brings its own)
    return cfg


# ------------------------------------------------------------------------------------------------ reference arm
_REF = {}


def _ref_init(cfg):
    import oracle
    o = oracle.Oracle(cfg)                          # one context per worker: the phantom is loaded once, outside the timed region
    o.set_options(want_phantom_sq=False)
    _REF["o"] = o


def _ref_run(job):
    first, n, seed = job
    o = _REF["o"]
    o.reset(); o.run(first, n, seed)
    r = o.read()
    return r["epid_sum"], r["ledger"]


def run_reference(args):
    """The oracle as it stands, timed on the host cores; each step is a bounded sample of the workload: P worker processes
    (contexts and phantom loaded before the timed region) transport disjoint history ranges, the parent adds the images.
    The K8 post-pass of the oracle (exact Siddon thickness map + LUT) is timed once, outside the steps, and reported."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import multiprocessing as mp
    import oracle
    cfg = build_cfg(args.config, args.field, args.physics_mode, args.collimator)
    procs = os.cpu_count() or 1
    sample = args.ref_histories or {"C0": 8_000_000, "C1": 4_000_000, "C2": 2_000_000}.get(args.config, 1_000_000)   # a few seconds per step
    oracle.build()
    per = max(sample // procs, 1); sample = per * procs
    with mp.get_context("fork").Pool(procs, initializer=_ref_init, initargs=(cfg,)) as pool:
        jobs = lambda k: [((k * procs + j) * per, per, cfg["seed"]) for j in range(procs)]
        for w in range(args.warmup):
            pool.map(_ref_run, [(f, max(n // 10, 1), sd) for f, n, sd in jobs(w)])
        t = []
        for k in range(args.steps):
            t0 = time.perf_counter()
            parts = pool.map(_ref_run, jobs(k))
            img = sum(p[0] for p in parts); n_run = sum(p[1][6] for p in parts)
            dose = img / n_run
            t.append(time.perf_counter() - t0)
    t0 = time.perf_counter()
    if not args.skip_ref_postpass:
        o = oracle.Oracle(cfg)
        o.apply_lut(cfg["lut"], dose, o.tmap(), o.field_size())
    t_post = time.perf_counter() - t0
    ms = 1e3 * float(np.mean(t))
    val = sample / (ms * 1e-3)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args), "histories_per_step": sample,
                       "note": "bounded sample of the workload per step; transport only (worker contexts persist across steps); "
                               "K8 post-pass of the oracle timed once: %.2f s" % t_post},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": procs, "kind": "oracle",
                             "sample": "%d histories of %s per step, %d persistent processes over disjoint history ranges" % (sample, args.config, procs),
                             "postpass_s_once": t_post},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_name(args):
    desc = {"C0": "photon-only toy", "C1": "6 MV open field on a water slab", "C2": "IMRT-like field on the heterogeneous thorax phantom",
            "C3": "9-segment IMRT field on the 512x512x200 synthetic patient, EPID 1024x768, 1e9 histories",
            "C4": "batch of 25 IMRT fields on the thorax phantom + response LUT"}[args.config]
    return "%s (BASELINE.json configs[%s]: %s)%s%s" % (args.config, args.config[1:], desc, " field %d" % args.field if args.config == "C4" else "",
                                                     " through the collimation stage (one history = one Phase Space 1 particle)" if args.collimator else "")


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

    cfg = build_cfg(args.config, args.field, args.physics_mode, args.collimator)
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
    first = parallel.shard_histories(n_total, rank, world)[0]

    def step(ev=None):
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
        if ev: ev[2].record()
        eng.apply_response_lut(lut_d, lut["t_min"], lut["t_max"], lut["s_min"], lut["s_max"], -1.0,
                               epid_in=dose, signal_out=signal, tmap_out=tmap)   # K8
    n_launch_transport = (n + (1 << 31) - 1) >> 31                       # aepid_simulate splits at 2^31 histories per launch
    launches_per_step = n_launch_transport + (2 if world == 1 else 4) + 2   # transport, folds (or moments + finalize), tmap + lut

    for _ in range(args.warmup):
        step(); flush.zero_()
    torch.cuda.synchronize()
    if world > 1: dist.barrier()
    sampler = ClockSampler(local)
    if rank == 0: sampler.start()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    torch.cuda.synchronize()
    t_wall = time.perf_counter()
    for k in range(args.steps):
        flush.zero_()                                                    # L2 flush between timed iterations (untimed)
        ev[k][3].record()
        step(ev[k])
        ev[k][4].record()
    torch.cuda.synchronize()
    if world > 1: dist.barrier()
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop() if rank == 0 else None
    step_ms = [e[3].elapsed_time(e[4]) for e in ev]
    kern_ms = [e[0].elapsed_time(e[1]) for e in ev]
    fold_ms = [e[1].elapsed_time(e[2]) for e in ev]
    post_ms = [e[2].elapsed_time(e[4]) for e in ev]
    tot = torch.tensor([sum(step_ms), sum(kern_ms), sum(fold_ms), sum(post_ms)], dtype=torch.float64, device=dev)
    if world > 1: dist.all_reduce(tot, op=dist.ReduceOp.MAX)
    total_ms, kernel_ms = float(tot[0]), float(tot[1])
    ms_per_step = total_ms / args.steps
    value = n_total / (ms_per_step * 1e-3)
    eng.synchronize()                                                    # raises if the transport kernel flagged an internal error (ledger[7])

    # statistical uncertainty U (reading A19) of the last step, native and re-binned towards the paper's 2.5 mm pixel
    unc = None
    if world == 1:
        b, nb = eng.read_batches()
        def U(r):
            B = b.shape[0]
            nv_, nu_ = (b.shape[1] // r) * r, (b.shape[2] // r) * r      # crop symmetrically to a multiple of r (6 does not divide 1024)
            o1, o2 = (b.shape[1] - nv_) // 2, (b.shape[2] - nu_) // 2
            rb = b[:, o1:o1 + nv_, o2:o2 + nu_].reshape(B, nv_ // r, r, nu_ // r, r).sum(axis=(2, 4)).astype(np.float64)
            N = nb.sum(); mean = rb.sum(0) / N
            var = (nb[:, None, None] * (rb / np.maximum(nb, 1)[:, None, None] - mean) ** 2).sum(0) / ((B - 1) * N)
            k = mean > 0.5 * mean.max()
            return float(np.sqrt(np.mean(var[k] / mean[k] ** 2)))
        pitch_mm = 10.0 * float(cfg["epid"]["pitch"])
        r_div = min((k for k in range(1, 65) if eng.nu % k == 0 and eng.nv % k == 0), key=lambda k: abs(k * pitch_mm - 2.5))
        r_near = max(1, int(round(2.5 / pitch_mm)))                      # the factor whose pixel is closest to 2.5 mm, image cropped
        un, ud, ur = U(1), U(r_div), U(r_near)
        t1 = lambda u: ms_per_step * 1e-3 * (u / 0.01) ** 2
        unc = {"U_native": un, "pixel_mm_native": pitch_mm,
               "U_rebinned": ur, "rebin": r_near, "pixel_mm_rebinned": r_near * pitch_mm,
               "rebinned_note": "%d x %d native pixels = %.3f mm, the factor closest to the paper's 2.5 mm (PAPER.md:110); the image is cropped by %d / %d "
                                "pixels to a multiple of it" % (r_near, r_near, r_near * pitch_mm, eng.nu % r_near, eng.nv % r_near),
               "U_rebinned_divisor": ud, "rebin_divisor": r_div, "pixel_mm_rebinned_divisor": r_div * pitch_mm,
               "seconds_to_1pct_native": t1(un), "seconds_to_1pct_rebinned": t1(ur), "seconds_to_1pct_rebinned_divisor": t1(ud),
               "seconds_per_field": ms_per_step * 1e-3}

    head = None
    if cfg.get("ps1") is not None and world == 1:
        hs = eng.read_head()
        head = {"ps2_particles_per_history": hs[0] / n, "ps2_particles_per_s": hs[0] / (ms_per_step * 1e-3), "ps2_energy_per_history_MeV": hs[1] / n,
                "absorbed_in_head_per_history_MeV": hs[2] / n, "note": "one history = one Phase Space 1 particle (synthetic, DESIGN.md A35); the paper counts Phase Space 2 particles (PAPER.md:100)"}
    # event mix of the workload: one untimed counting launch (instrumented instantiation of the same kernel)
    n_cnt = int(min(n, 20_000_000))
    eng.reset_tallies(); eng.set_history_offset(first); eng.set_counting(True)
    eng.simulate(n_cnt, seed)
    counters = eng.read_counters()
    eng.set_counting(False); eng.reset_tallies()
    evmix = events_per_history(counters, n_cnt)

    # e2e: the same step through the C-ABI with HOST buffers, host<->device copies inside the timed region
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    t, ph, ep, s = cfg["tables"], cfg["phantom"], cfg["epid"], cfg["source"]
    hin = {k: pin(t[k]) for k in ("E_grid", "mu_compton", "mu_pe", "mu_pair", "T_grid", "stop_pow", "rad_len")}
    hin.update(density=pin(ph["density"]), material=pin(ph["material"]), E_edges=pin(s["E_edges"]), E_pdf=pin(s["E_pdf"]),
               fluence=pin(s["fluence"]), lut=pin(np.ascontiguousarray(lut["lut"], dtype=np.float32)))
    if cfg.get("ps1") is not None:
        hin["ps1"] = pin(cfg["ps1"]["records"])
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
        if cfg.get("ps1") is not None:                                   # collimation stage: Phase Space 1 table and the jaws / leaves
            eng.load_phase_space_source(hin["ps1"], cfg["ps1"]["plane"])
            eng.load_collimator(cfg["collimator"])
        eng.set_history_offset(first)
        eng.simulate(n, seed)
        eng.read_tallies(out=hout)                                       # host outputs: synchronises and checks the kernel's error flags
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
    alg = alg_instr_per_history(evmix)
    k_ms = kernel_ms / args.steps
    achieved = alg * n / (k_ms * 1e-3) / 1e9
    cap = NCU_CAPTURES.get("%s_mode%d" % (args.config, int(cfg["physics"]["mode"])))
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_ginstr, "unit": "Gthread-instr/s", "frac": achieved / peak_ginstr,
                "traffic": (cap["dram_bytes_per_history"] * n) if cap else None,
                "kernel": "transport_kernel", "kernel_ms_per_launch": k_ms / n_launch_transport, "launches_per_step": n_launch_transport,
                "kernel_share_of_step": kernel_ms / total_ms,
                "alg_thread_instr_per_history": alg, "alg_unit_cost": ALG_UNIT_COST,
                "events_per_history": evmix, "events_from": "aepid_read_counters after an untimed counting launch of %d histories of this workload" % n_cnt,
                "how": "frac = sum_k alg_unit_cost[k] * events_per_history[k] * histories / kernel time / peak; peak = %s sm_max_mhz x %d SMs x 4 schedulers x 32 lanes" % (which, sm_count),
                "ncu": cap, "hbm_gbs_peak": peaks.get("hbm_gbs"),
                "hbm_frac": (cap["dram_bytes_per_history"] * n / (k_ms * 1e-3) / 1e9 / float(peaks.get("hbm_gbs", 6549.4))) if cap else None,
                # north_star's second candidate, "the instruction count at the SM issue peak", with the EXECUTED count of the ncu
                # capture (warp-instructions per history x active lanes) at this run's rate: what the kernel issues, not what the method needs
                "executed_thread_instr_per_history": (cap["warp_instr_per_history"] * cap["lanes_per_warp_instr"]) if cap else None,
                "executed_frac": (cap["warp_instr_per_history"] * cap["lanes_per_warp_instr"] * n / (k_ms * 1e-3) / 1e9 / peak_ginstr) if cap else None}
    per_kernel = {"transport_ms": k_ms, "fold_ms": float(tot[2]) / args.steps, "tmap_and_lut_ms": float(tot[3]) / args.steps,
                  "note": "CUDA events on the launching stream; fold = the two fold_kernel launches of aepid_read_tallies (EPID, phantom), "
                          "tmap_and_lut = tmap_kernel + apply_lut_kernel of aepid_apply_response_lut"}

    # CPU baseline: the oracle as it stands on the host cores, bounded sample; all cores, then one thread
    import oracle
    procs = os.cpu_count() or 1
    oracle.build()
    ns = 10_000 if args.profile else (args.cpu_sample or {"C0": 120_000_000, "C1": 60_000_000, "C2": 40_000_000, "C4": 40_000_000}.get(args.config, 30_000_000))   # 10-30 s of host time
    wk = _OraclePool(cfg, procs)
    wk.run(procs * 50, seed, 0)                                          # page-in warm-up
    t0 = time.perf_counter(); wk.run(ns, seed, 0); dt = time.perf_counter() - t0
    wk.close()
    n1 = max(ns // (4 * procs), 1000)
    w1 = _OraclePool(cfg, 1); w1.run(100, seed, 0)
    t0 = time.perf_counter(); w1.run(n1, seed, 0); dt1 = time.perf_counter() - t0
    w1.close()
    cpu = {"value": ns / dt, "unit": UNIT, "cores": procs, "kind": "oracle",
           "sample": "first %d histories of %s, %d processes over disjoint history ranges, contexts loaded beforehand (%.1f s wall)" % (ns, args.config, procs, dt),
           "single_thread": {"value": n1 / dt1, "unit": UNIT, "cores": 1, "sample": "first %d histories, one process (%.1f s)" % (n1, dt1)}}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(args), "histories_per_gpu_per_step": n,
                       "n_batches": eng.n_batches, "physics_mode": int(cfg["physics"]["mode"]), "l2": "flushed between timed steps (256 MiB write)",
                       "parallelism": "history-range sharding x%d, one all-reduce of tally moments per step" % world if world > 1 else "single GPU"},
            "clocks": clocks, "roofline": roofline, "per_kernel": per_kernel, "cpu_baseline": cpu,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": float(e2e_ms[0])},
            "gpu_launches": launches_per_step * args.steps,
            "uncertainty": unc, "collimation_stage": head, "wall_s_timed_region": t_wall,
            "context": {"paper": "~90 s per 1e9-history IMRT field on 1x RTX 3090 (PAPER.md:127, 202), ~1.1e7 histories/s, fuller physics"}}
    print(json.dumps(line))
    if world > 1: dist.destroy_process_group()


class _OraclePool:
    """P oracle worker processes with their contexts (phantom, tables) loaded once; run() times transport only."""

    def __init__(self, cfg, procs):
        import multiprocessing as mp
        self.procs = procs
        self.pool = mp.get_context("fork").Pool(procs, initializer=_ref_init, initargs=(cfg,))
        self.pool.map(_ref_run, [(0, 1, 0)] * procs)                     # make sure every worker has built its context

    def run(self, n, seed, first):
        per = max(n // self.procs, 1)
        return self.pool.map(_ref_run, [(first + j * per, per, seed) for j in range(self.procs)])

    def close(self):
        self.pool.close(); self.pool.join()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C3", choices=["C0", "C1", "C2", "C3", "C4"])
    ap.add_argument("--physics-mode", type=int, default=None, choices=[0, 1, 2, 3, 4], help="override the physics mode (2: Class II collisions, 3: + bremsstrahlung, 4: multi-voxel steps with a random hinge)")
    ap.add_argument("--field", type=int, default=0, help="which of C4's 25 IMRT fields (seeds per reading A23)")
    ap.add_argument("--collimator", action="store_true", help="C4 only: collimation stage (synthetic Phase Space 1, jaws, MLC) in place of the fluence map")
    ap.add_argument("--histories", type=int, default=0, help="histories per GPU per step (default: the config's)")
    ap.add_argument("--cpu-sample", type=int, default=0, help="oracle histories timed for cpu_baseline (default: by config, 10-30 s of host time)")
    ap.add_argument("--ref-histories", type=int, default=0, help="oracle histories per step of --impl reference (default: by config)")
    ap.add_argument("--skip-ref-postpass", action="store_true", help="--impl reference: do not time the oracle's K8 post-pass")
    ap.add_argument("--profile", action="store_true", help="short run for ncu: one e2e step, tiny cpu_baseline sample (numbers are not bench values)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
