#!/usr/bin/env python
"""bench.py — timesteps/s and site-updates/s of the pseudo-spectral SPDE step on B200.

    python bench.py --gpus N --steps K --warmup W [--workload modelb_1024] [--inner 500]
    python bench.py --impl reference ...            # the CPU oracle, timed on the host cores

One bench "step" is one call pss_step(inner): `inner` consecutive time steps of the whole hot path
(k_rows + k_update per time step, or all of them inside one persistent p2d::k_persist2d launch at 1024^2 fp32) on the workload's lattice.  The state of a time stepper is consumed by
the next time step, so inside one bench step the working set is as warm as the workload makes it; BETWEEN
timed bench steps L2 is flushed (a 256 MiB buffer is written), so every timed step starts cold.

value      = timesteps/s with the state resident in HBM (sum over ranks; N > 1 runs independent replicas,
             different seeds, no collective: "replicas only", DESIGN.md section Multi-GPU)
e2e        = the same through the public API with HOST buffers: pss_set_field(host) -> pss_step(inner) ->
             pss_get_field(host) inside the timed region
roofline   = dominant kernel (by device time, from pss_profile_step's per-launch CUDA events): algorithmic
             bytes per launch / mean launch duration against MEASURED_PEAKS.json's HBM copy bandwidth
cpu_baseline = the oracle as it stands on the host cores, bounded sample
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2405_02410_b200 import replicas, workloads as wl  # noqa: E402

FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md "FALLBACK"


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.lines = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "25"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_rate(cfg, prec, budget_s, max_steps):
    """timesteps/s of the CPU oracle on a bounded sample: 1 warm-up step, then steps until budget_s."""
    from oracle import opss
    o, _ = wl.build(opss, cfg, prec=prec)
    o.step(1)
    n, t0 = 0, time.perf_counter()
    while True:
        o.step(1)
        n += 1
        el = time.perf_counter() - t0
        if el >= budget_s or n >= max_steps:
            break
    cores = int(os.environ.get("OMP_NUM_THREADS", "0")) or (os.cpu_count() or 1)
    return n / el, n, el, cores


def bench_config(args, cfg, R):
    """the `config` object of the JSON line: the workload, identical for the CUDA arm and the reference arm"""
    return {"workload": args.workload, "lattice": list(cfg["n"]), "precision": args.prec,
            "timesteps_per_bench_step": int(min(args.inner, 250) if cfg["model"] == "nematic" else args.inner),
            "replicas_per_gpu": int(R),
            "parallelism": "replicas only (independent realisations; value counts replica time steps)",
            "l2": "flushed between timed bench steps (256 MiB written); inside a bench step the "
                  "time stepper reuses its own state, as the workload does"}


def run_reference(args, cfg, rank, world):
    """--impl reference: the CPU oracle as it stands on the host cores, same workload/metric/unit.  One bench step is
    a bounded sample of oracle time steps (ref_budget / steps seconds, at least one time step)."""
    if rank != 0:
        return
    from oracle import opss
    o, _ = wl.build(opss, cfg, prec=args.prec)
    for _ in range(max(1, args.warmup)):
        o.step(1)
    sites = int(np.prod(cfg["n"]))
    per_step_budget = args.ref_budget / max(1, args.steps)
    total_steps, total_t = 0, 0.0
    for _ in range(args.steps):
        n, t0 = 0, time.perf_counter()
        while True:
            o.step(1)
            n += 1
            el = time.perf_counter() - t0
            if el >= per_step_budget:
                break
        total_steps += n
        total_t += el
    cores = int(os.environ.get("OMP_NUM_THREADS", "0")) or (os.cpu_count() or 1)
    v = total_steps / total_t
    line = {
        "impl": "reference", "metric": "timesteps/s", "value": v, "unit": "timesteps/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total_t / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "site_updates_per_s": v * sites,
        "config": bench_config(args, cfg, 1),
        "note": "CPU oracle (oracle/opss.cpp) as it stands; each bench step is a bounded sample of oracle time steps "
                "of the workload that config names",
        "cpu_baseline": {"value": v, "unit": "timesteps/s", "cores": cores, "kind": "oracle",
                         "sample": "%d oracle time steps of %s in %.1f s" % (total_steps, args.workload, total_t)},
        "e2e": {"value": v, "unit": "timesteps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--inner", type=int, default=500, help="time steps per bench step (one pss_step call)")
    ap.add_argument("--workload", default="modelb_1024")
    ap.add_argument("--prec", default="f32")
    ap.add_argument("--impl", default="pss", choices=["pss", "reference"])
    ap.add_argument("--ref-budget", type=float, default=20.0, help="seconds of oracle work for the reference arm")
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of oracle work for cpu_baseline")
    ap.add_argument("--replicas", type=int, default=1,
                    help="ensemble: R independent realisations stepped in the same launches (value counts replica-steps)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-compare", action="store_true", help="skip the cuFFT+cuRAND comparison step (2D Model B only)")
    ap.add_argument("--no-secondary", action="store_true",
                    help="skip the short timed legs of the other BASELINE configs that the default (headline) run appends under `secondary`")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = wl.make_config(args.workload)

    if args.impl == "reference":
        run_reference(args, cfg, rank, world)
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    import paper_2405_02410_b200 as pss

    # replicas only: every rank advances its own realisation (seed + rank), no data-path collective
    cfg_r = replicas.rank_config(cfg, rank)
    R = max(1, args.replicas)
    cfg_r["seed"] = cfg["seed"] + rank * R          # replica r of rank k is the realisation seed + k*R + r
    g, ids = wl.build(pss, cfg_r, prec=args.prec, device="cuda:%d" % local_rank, set_ic=False, replicas=R)
    dyn_names = list(cfg["ic"].keys())
    sites = int(np.prod(cfg["n"]))
    rsize = 4 if args.prec == "f32" else 8
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    ics = [wl.initial_conditions(dict(cfg_r, seed=cfg_r["seed"] + r), g.rdtype) for r in range(R)]

    def reset_state():
        for r in range(R):
            g.select_replica(r)
            for name, arr in ics[r].items():
                g.set_field(ids[name], arr)

    reset_state()

    # nematic (A20): the literal parameters blow up after ~400 steps -> re-seed before every bench step
    reseed = cfg["model"] == "nematic"
    inner = min(args.inner, 250) if reseed else args.inner

    # clocks / throttle reasons are sampled from before the warm-up (same kernels, same load) to the end of the timed region
    sampler = ClockSampler(local_rank) if rank == 0 else None
    for _ in range(max(args.warmup, 0)):
        if reseed:
            reset_state()
        g.step(inner)
    barrier()

    launches0 = g.launch_count
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    launches_timed = 0
    for i in range(args.steps):
        if reseed:
            reset_state()
        flush.fill_(i & 0xff)  # L2 flush between timed steps (not timed)
        l0 = g.launch_count
        ev[i][0].record(stream)
        g.step(inner)
        ev[i][1].record(stream)
        launches_timed += g.launch_count - l0
    barrier()
    ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(ms))
    clocks = sampler.stop() if sampler else None
    # the state the TIMED steps ended on (the e2e leg below reloads the initial condition, so its output says nothing
    # about the long run)
    g.select_replica(0)
    timed_finite = all(bool(np.isfinite(g.get_field_fourier(ids[n_]).view(g.rdtype)).all()) for n_ in dyn_names)

    # ---- e2e: host buffers through the public API, copies inside the timed region ----
    host_in = [{name: torch.from_numpy(arr).pin_memory() for name, arr in ics[r].items()} for r in range(R)]
    host_out = [{name: torch.empty_like(t).pin_memory() for name, t in host_in[r].items()} for r in range(R)]
    e2e_steps = max(2, min(args.steps, 5))

    def e2e_once():
        for r in range(R):
            g.select_replica(r)
            for name in dyn_names:
                g.set_field(ids[name], host_in[r][name].numpy())
        g.step(inner)
        for r in range(R):
            g.select_replica(r)
            for name in dyn_names:
                g.get_field(ids[name], out=host_out[r][name].numpy())

    e2e_once()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_once()
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0
    finite = all(bool(np.isfinite(host_out[r][n].numpy()).all()) for r in range(R) for n in dyn_names)

    # ---- per-kernel device times (CUDA events around every launch) for the roofline of the dominant kernel ----
    if reseed:
        reset_state()
    prof_n = min(200, inner)
    prof = g.profile_step(prof_n)
    barrier()

    # max over ranks of the timed totals; sum of units
    (total_ms, e2e_s), steps_all = replicas.reduce_timings([total_ms, e2e_s], args.steps * inner * R, device=dev)
    value = steps_all / (total_ms * 1e-3)
    e2e_value = world * e2e_steps * inner * R / e2e_s

    if rank == 0:
        peak, peak_src = measured_peak()
        S = sites * rsize
        b_alg = g.model_bytes_per_step(True)
        b_model = g.model_bytes_per_step(False)
        step_ms = total_ms / (args.steps * inner)   # one launch sequence advances all R replicas by one time step
        # dominant kernel by share of device time
        shares = {k: v[0] * v[1] for k, v in prof.items() if v[1] > 0}
        dom = max(shares, key=shares.get)
        dom_ms = prof[dom][0]
        dom_name = (g.fused_kernel_name or dom) if dom == "k_fused2d" else dom   # which persistent kernel ran
        P = g  # algorithmic bytes per launch of each kernel family
        # the persistent kernel's launches are cut at the Hermitian-projection period (pss_hermitian_period()) and run one
        # replica each: time steps one launch advances = prof_n * R / launches
        fused_steps = prof_n * R / max(1, prof["k_fused2d"][1])
        kb = kernel_bytes(cfg, S * R, g, fused_steps / R)
        roof_kernel = dom_name
        if kb[dom] is None:
            # several rounds of the two step kernels per time step (product-defined intermediate fields): the library
            # reports algorithmic bytes per STEP only (pss_model_bytes_per_step sums the rounds), so the roofline entry is
            # the whole step's launch sequence, not one kernel with an invented share of the bytes
            roof_kernel = "k_rows+k_update (all rounds of one time step)"
            kb[dom] = b_alg
            dom_ms = step_ms
        ach = kb[dom] / (dom_ms * 1e-3) / 1e9
        line = {
            "metric": "timesteps/s", "value": value, "unit": "timesteps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": args.prec, "data": "synthetic",
            "site_updates_per_s": value * sites, "us_per_timestep": step_ms * 1e3, "us_per_replica_timestep": step_ms * 1e3 / R,
            "config": bench_config(args, cfg, R),
            "final_state_finite": bool(finite and timed_finite), "timed_state_finite": timed_finite,
            "gpu_launches": int(launches_timed),
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "timesteps/s",
                    "h2d_bytes_per_step": len(dyn_names) * S * R, "d2h_bytes_per_step": len(dyn_names) * S * R,
                    "note": "pss_set_field(host) + pss_step(%d) + pss_get_field(host) per bench step" % inner},
            "roofline": {"bound": "hbm", "kernel": roof_kernel, "achieved": ach, "peak": peak, "unit": "GB/s",
                         "frac": ach / peak, "traffic": (ncu_traffic(args.workload, dom_name) or {}).get("dram_bytes_per_launch"),
                         "traffic_capture": ncu_traffic(args.workload, dom_name), "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": kb[dom], "launch_ms": dom_ms,
                         "timesteps_per_launch": fused_steps if dom == "k_fused2d" else 1,
                         "kernel_ms": {(dom_name if k == dom else k): v[0] for k, v in prof.items() if v[1] > 0},
                         "kernel_share": {(dom_name if k == dom else k): shares[k] / sum(shares.values()) for k in shares}},
            "roofline_step": {"B_alg_bytes": b_alg, "B_model_bytes": b_model,
                              "achieved_alg_GBs": b_alg / (step_ms * 1e-3) / 1e9,
                              "frac_alg": b_alg / (step_ms * 1e-3) / 1e9 / peak,
                              "frac_model": b_model / (step_ms * 1e-3) / 1e9 / peak,
                              "frac_alg_of_8TBs": b_alg / (step_ms * 1e-3) / 1e9 / 8000.0},
        }
        # secondary reading: the kernels are issue-bound, so also report the issue-slot fraction of the dominant kernel
        # (ncu smsp__inst_executed.sum of the committed capture / its step count, against 4 schedulers x SMs x clock)
        tr = line["roofline"]["traffic_capture"]
        if tr:
            nsm = torch.cuda.get_device_properties(dev).multi_processor_count
            mhz = (clocks or {}).get("sm_mhz") or 1965.0
            wi_step = R * tr["warp_instr_per_launch"] / tr["timesteps_per_launch"]  # the capture ran one replica
            t_dom = dom_ms * 1e-3 * (prof["k_fused2d"][1] / prof_n if dom == "k_fused2d" else 1)   # dominant kernel's time per time step
            line["roofline"]["issue"] = {"bound": "alu", "unit": "warp-instr/s", "achieved": wi_step / t_dom,
                                         "peak": 4.0 * nsm * mhz * 1e6, "frac": wi_step / t_dom / (4.0 * nsm * mhz * 1e6),
                                         "note": "instruction-issue slots: 4 schedulers per SM x 1 warp-instr per clock"}
            # `frac` above is BASELINE.json's target metric: ALGORITHMIC bytes against the HBM peak.  What the kernel really
            # pulls from DRAM (the committed ncu capture) can be far less when the working set stays in L2: say so, and name
            # the resource that is actually closest to its ceiling.
            dram_step = R * tr["dram_bytes_per_launch"] / tr["timesteps_per_launch"]
            dram_frac = dram_step / t_dom / 1e9 / peak
            line["roofline"]["frac_meaning"] = "algorithmic bytes per launch / launch time / measured HBM peak (BASELINE.json target metric)"
            line["roofline"]["dram_frac_measured"] = dram_frac
            line["roofline"]["limiter"] = ("issue slots / L2 round trips (working set L2-resident: measured DRAM traffic is %.1f%% of the algorithmic bytes)"
                                           % (100.0 * dram_step / b_alg)
                                           if line["roofline"]["issue"]["frac"] > dram_frac else "hbm")
        if not args.no_cpu_baseline and world == 1:
            r, n, el, cores = oracle_rate(cfg, args.prec, args.cpu_budget, 10 ** 6)
            line["cpu_baseline"] = {"value": r, "unit": "timesteps/s", "cores": cores, "kind": "oracle",
                                    "sample": "%d oracle time steps of %s after 1 warm-up step, %.1f s" % (n, args.workload, el)}
        if not args.no_compare and world == 1 and cfg["model"] == "model_b" and len(cfg["n"]) == 2 and args.prec == "f32":
            line["cufft_curand_comparison"] = cufft_compare(cfg)
        if not args.no_secondary and world == 1 and R == 1 and args.workload == "modelb_1024" and args.prec == "f32":
            del g
            line["secondary"] = secondary_legs(pss, torch, dev, stream, flush, peak)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


SECONDARY = ("sweep_4096", "kpz_4096", "modelb_256c", "nematic_1024", "modelb_128")


def secondary_legs(pss, torch, dev, stream, flush, peak):
    """Short timed legs of the other BASELINE.json configs, so that the driver's own run clocks more than the headline:
    per workload 3 warm-up calls and 3 timed calls of pss_step(20) (60 timed time steps), CUDA events on the launching
    stream, L2 flushed before every timed call, state resident in HBM; fp32, one replica, no oracle leg.
    frac_alg = B_alg (pss_model_bytes_per_step, pruned) / time per time step / measured HBM peak."""
    out = {}
    for name in SECONDARY:
        try:
            c = wl.make_config(name)
            s, ids = wl.build(pss, c, prec="f32", device=str(dev))
            inner, calls = 20, 3
            for _ in range(3):
                s.step(inner)
            if c["model"] == "nematic":   # A20: the literal parameters blow up after ~400 steps; 60 + 60 stay well inside
                for nm, arr in wl.initial_conditions(c, s.rdtype).items():
                    s.set_field(ids[nm], arr)
                s.step(inner)
            torch.cuda.synchronize(dev)
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(calls)]
            for i in range(calls):
                flush.fill_(i + 1)
                ev[i][0].record(stream)
                s.step(inner)
                ev[i][1].record(stream)
            torch.cuda.synchronize(dev)
            us = 1e3 * sum(a.elapsed_time(b) for a, b in ev) / (calls * inner)
            b_alg = s.model_bytes_per_step(True)
            fin = bool(np.isfinite(s.get_field(ids[list(c["ic"].keys())[0]])).all())
            out[name] = {"us_per_timestep": us, "frac_alg": b_alg / (us * 1e-6) / 1e9 / peak, "B_alg_bytes": b_alg,
                         "lattice": list(c["n"]), "timed_timesteps": calls * inner, "kernel": s.fused_kernel_name or "k_rows+k_update",
                         "final_state_finite": fin}
            del s
        except Exception as e:  # a secondary leg never takes the headline line down with it
            out[name] = {"unavailable": repr(e)[:200]}
    return out


def cufft_compare(cfg):
    """The same 2D Model-B step built the way the paper describes its GPU path (cuFFT for every transform, cuRAND
    noise, one pointwise kernel per arrow; compare/cufft_modelb.cu), timed with CUDA events on
    this GPU.  A comparison baseline only (north_star); the product never loads it."""
    import ctypes
    try:
        from compare import build as compare_build
        lib = ctypes.CDLL(compare_build.build())
        us = ctypes.c_double(0.0)
        pr = cfg["params"]
        nsteps = 200 if cfg["n"][0] <= 2048 else 30
        rc = lib.cmp_cufft_modelb(int(cfg["n"][0]), int(cfg["n"][1]), ctypes.c_double(float(cfg["dx"])),
                                  ctypes.c_double(cfg["dt"]), ctypes.c_double(pr["a"]), ctypes.c_double(pr["b"]),
                                  ctypes.c_double(pr["k"]), ctypes.c_double(pr["D"]), nsteps, 20, ctypes.byref(us))
        if rc != 0:
            return {"unavailable": "cmp_cufft_modelb returned %d" % rc}
        return {"us_per_timestep": us.value, "timesteps_per_s": 1e6 / us.value, "timed_steps": nsteps,
                "what": "mask copy, cufftExecC2R, cube, cufftExecR2C, curandGenerateNormal, cufftExecR2C, Eq. 18 kernel"}
    except Exception as e:  # the comparison is optional context, never a reason to fail the bench
        return {"unavailable": repr(e)[:200]}


def kernel_bytes(cfg, S, g, steps_per_fused_launch):
    """algorithmic bytes per launch of each kernel family (pruned count, SURVEY.md 8(d) / DESIGN.md).
    k_fused2d runs every step of a pss_step(n) call in ONE launch: its bytes per launch are n * B_alg."""
    total = g.model_bytes_per_step(True)
    ndim = len(cfg["n"])
    model = cfg["model"]
    # factor kept-fractions and counts follow from the term list; derive the split from the totals:
    # rows   : sum_f c_f (read) + ngrp (write)
    # update : ngrp (read) + 2 ndyn + sum_f c_f^(ndim-1) (write)
    table = {"model_b": (1, 1, [0.5]), "kpz": (1, 1, [2 / 3.0] * ndim),
             "nematic": (2, 2, [0.5, 0.5] + [2 / 3.0] * 7), "diffusion": (1, 0, [])}
    if model not in table:  # several rounds of the two kernels (product-defined intermediate fields): no per-kernel split
        return {"k_rows": None, "k_update": None, "k_mid": None, "k_fused2d": total * steps_per_fused_launch}
    ndyn, ngrp, cs = table[model]
    rows = S * (sum(cs) + ngrp)
    upd = S * (ngrp + 2 * ndyn + sum(c ** (ndim - 1) for c in cs))
    mid = 0.0
    if ndim == 3:
        mid = (total - rows - upd) / 2.0  # two k_mid launches per step (forward on groups, inverse on factors)
    return {"k_rows": rows, "k_update": upd, "k_mid": mid, "k_fused2d": total * steps_per_fused_launch}


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload` from the committed
    ncu --set full capture (profiles/ncu_traffic.csv), or None.  For k_fused2d one launch of that capture ran
    `timesteps_per_launch` time steps (the working set is L2-resident: DRAM traffic is mostly the first touch)."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    try:
        with open(p) as f:
            for ln in f.read().splitlines()[1:]:
                w, k, b, n, wi, src = ln.split(",")
                if w == workload and k == kernel:
                    return {"dram_bytes_per_launch": int(b), "timesteps_per_launch": int(n),
                            "warp_instr_per_launch": int(wi), "source": src}
    except Exception:
        pass
    return None


if __name__ == "__main__":
    main()
