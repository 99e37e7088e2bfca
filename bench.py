#!/usr/bin/env python
"""bench.py -- zone-updates/s of the hydro hot path on BASELINE.json config 5 (512^3).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..5]

A "step" is one whole pass of the hot path over the workload: one SSP-RK2 step =
estimate_dt + 2 x (fill_ghosts + advance_stage) on every zone of the synthetic state.
Prints ONE JSON line (rank 0).  See DESIGN.md sec. 7 for every field.

  value      whole-job zone-updates/s with the state resident in HBM (CUDA events on the launch
             stream, max over ranks).  N > 1 = N independent replicas (the
             path named by north_star is single-GPU, "replicas only"), so scaling = "weak".
  e2e        same metric through the C-ABI call that takes HOST buffers (hydro_run_host):
             H2D of the state + step + D2H inside the timed region.
  roofline   dominant kernel class: algorithmic bytes per launch / its mean launch duration
             (CUDA event pairs recorded by the library around every launch of the timed region).
  cpu_baseline  the CPU oracle, as it stands, timed on this box's host cores on a bounded
             sample of the same recipe.
--impl reference times only the oracle (there is no reference implementation to install).
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

import numpy as np  # noqa: E402

from paper_2007_05218_b200 import workloads as W  # noqa: E402

METRIC = "zone-updates/sec per RK2 step (FP64)"
UNIT = "zone-updates/s"


# ----------------------------------------------------------------------------- helpers
def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def algorithmic_bytes(wl, ns_groups, steps, split_ghosts, fuse_dt, xmarch=False, one_launch=0):
    """Algorithmic HBM bytes per launch of each kernel class: what the kernel
    split must move -- every input once with the 3-zone PPM halo along the sweep direction, every
    output once.  Returns {class: mean bytes per launch over the launches of `steps` steps issued
    by ONE hydro_step call}."""
    nb, nvar, nflux, ns, ng = wl.nb, wl.nvar, wl.nflux, wl.nspec, wl.ng
    Z = wl.zones
    halo = [(nb[d] + 6) / nb[d] for d in range(3)]
    face = [(nb[d] + 1) / nb[d] for d in range(3)]
    nt = wl.nt
    ghost_zones = wl.nboxes * (nt[0] * nt[1] * nt[2] - nb[0] * nb[1] * nb[2])
    row_zones = wl.nboxes * (nt[2] * nt[1] - nb[2] * nb[1]) * nt[0]          # zones of the ghost rows
    xend = (2 * ng / nb[0]) if split_ghosts else 0.0                          # x images per valid zone
    out = {}
    full = 2 * nvar * 8 * ghost_zones
    rows = 2 * nvar * 8 * row_zones
    if split_ghosts:      # one full fill of the caller's state (two launches: x ends, ghost rows), then ghost-row copies
        out["fill_ghosts"] = (full + (2 * steps - 1) * rows) / (2 * steps + 1)
    else:
        out["fill_ghosts"] = full
    out["estimate_dt"] = 5 * 8 * Z
    out["sweep_x"] = Z * ((nvar - 1) * 8 * halo[0] + nflux * 8)
    if xmarch:
        # marching x kernels (march_x.cuh): rows are read in 4-zone steps -4 .. nb0+3; the hydro launch writes
        # F_rho,x (rows of nb0+4), every species launch reads it and rho again.  Mean over the 1 + groups launches.
        hx, fx = (nb[0] + 8) / nb[0], (nb[0] + 4) / nb[0]
        per = [5 * 8 * hx + 5 * 8 + 8 * fx] + [(1 + g) * 8 * hx + 8 * fx + g * 8 for g in ns_groups]
        out["sweep_x"] = Z * float(np.mean(per))
    out["hydro_y"] = Z * (5 * 8 * halo[1] + 2 * 5 * 8 + 8 * face[1])
    # z hydro: 6 state rows with halo (ring), Lacc read, 6 components written (+ their x images),
    # F_rho written; stage 1 also reads U0 (mean over the two stages)
    out["hydro_z"] = Z * (6 * 8 * halo[2] + 5 * 8 + 6 * 8 * (1 + xend) + 8 * face[2] + 0.5 * 5 * 8)
    if wl.params.get("flatten"):
        # k_flatten reads (rho, m_x, m_y, m_z, rho e) with one ghost layer more than it writes; every sweep
        # kernel reads the coefficient row of its zones (with the march halo)
        ext = np.prod([(nb[d] + 2) / nb[d] for d in range(3)])
        out["flatten"] = Z * (5 * 8 * np.prod([(nb[d] + 8) / nb[d] for d in range(3)]) + 8 * ext)
        out["sweep_x"] += Z * 8 * halo[0]
        out["hydro_y"] += Z * 8 * halo[1]
        out["hydro_z"] += Z * 8 * halo[2]
    ev = bool(wl.params.get("evolve_eint"))
    fl = bool(wl.params.get("flatten"))
    if ev:
        # O11: three more accumulator slots: flux of rho*e and div(u_face) go through x (written), y (read and
        # written) and z (read; the z hydro kernel also writes the final div u and rho*E - K); the energy launch
        # of each direction is a one-"species" sweep over (rho, rho*e) that is timed with the species class
        out["sweep_x"] += Z * 2 * 8
        out["hydro_y"] += Z * 2 * 8
        out["hydro_z"] += Z * (8 + 2 * 8)
    if ns or ev:
        groups = list(ns_groups)
        sy = [Z * ((1 + g) * 8 * halo[1] + 8 * face[1] + 2 * g * 8 + (8 * halo[1] if fl else 0)) for g in groups]
        sz = [Z * ((1 + g) * 8 * halo[2] + 8 * face[2] + g * 8 + g * 8 * (1 + xend) + 0.5 * g * 8 + (8 * halo[2] if fl else 0))
              for g in groups]
        if ev:
            sy.append(Z * (2 * 8 * halo[1] + 8 * face[1] + 2 * 8 + (8 * halo[1] if fl else 0)))
            sz.append(Z * (2 * 8 * halo[2] + 8 * face[2] + 4 * 8 + 8 * (1 + xend) + 0.5 * 8 + (8 * halo[2] if fl else 0)))
        out["species_y"] = float(np.mean(sy))
        out["species_z"] = float(np.mean(sz))
        # all groups in one launch (hydro_query 5): the launch reads rho (with its halo) and F_rho once, not once per group
        shared = [Z * (8 * halo[d] + 8 * face[d]) for d in (1, 2)]
        n_sp = len(groups)            # the O11 energy launch stays a launch of its own
        if one_launch & 1 and n_sp >= 2:
            out["species_y"] = (float(np.sum(sy[:n_sp])) - (n_sp - 1) * shared[0] + float(np.sum(sy[n_sp:]))) / (1 + len(sy) - n_sp)
        if one_launch & 2 and n_sp >= 2:
            out["species_z"] = (float(np.sum(sz[:n_sp])) - (n_sp - 1) * shared[1] + float(np.sum(sz[n_sp:]))) / (1 + len(sz) - n_sp)
    return out


def reduce_max(x, world, device="cpu"):
    """Max over ranks of a per-rank scalar (the device-timed ms of the timed region): the contract's
    max-over-ranks rule.  gloo (CPU tensors) in the tests, nccl (device tensors) in the bench."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(zones, steps, ms_total, world):
    """Whole-job zone-updates/s of `world` independent replicas (replicas only)."""
    return world * zones * steps / (ms_total * 1e-3)


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.stop_flag = index, [], False

    def run(self):
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5)
                f = [x.strip() for x in out.stdout.strip().split(",")]
                if len(f) >= 6:
                    self.samples.append(f)
            except Exception:
                pass
            time.sleep(0.1)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(s[0]) for s in self.samples)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(s[2 + i].lower().startswith("active") for s in self.samples)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.samples[0][1]), "reasons": reasons,
                "samples": len(sm)}


def host_info():
    model = "unknown"
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"cpu_model": model, "nproc": os.cpu_count()}


def oracle_sample(steps, warmup, n=256, threads=None):
    """The oracle, as it stands, on a bounded sample of the config-5 recipe: the n^3 instance of the
    same index-based generator (13 species, periodic, CFL 0.4) in 64^3 boxes, on `threads` host threads
    (None = all the cores OpenMP sees; the loop over boxes is the only parallel loop)."""
    from oracle import oracle_binding as O
    nb = 64 if n >= 256 else 32           # at least 64 boxes: the loop over boxes is what keeps the cores busy
    wl = W.config(5, ndom=(n, n, n), nbox=(nb, nb, nb))
    U0 = W.initial_state(wl, threads=8)
    U1 = np.zeros_like(U0)
    p = O.make_params(wl.params)
    all_threads = O.max_threads()
    if "TORCHELASTIC_RUN_ID" in os.environ:      # torchrun sets OMP_NUM_THREADS=1 for its ranks; rank 0 alone works here
        all_threads = max(all_threads, len(os.sched_getaffinity(0)))
    O.set_threads(threads or all_threads)
    used = min(threads or all_threads, wl.nboxes)
    for _ in range(warmup):
        O.step(p, U0, U1)
    t0 = time.perf_counter()
    for _ in range(steps):
        O.step(p, U0, U1)
    el = time.perf_counter() - t0
    O.set_threads(all_threads)
    return {"value": wl.zones * steps / el, "unit": UNIT, "cores": used, "cores_available": all_threads, "kind": "oracle",
            "sample": f"config-5 recipe at {n}^3 (13 species, {wl.nboxes} boxes of {nb}^3), {steps} RK2 steps, "
                      f"{used} of {all_threads} thread(s) over boxes, {el:.1f} s"}, el / steps * 1e3, wl


def workload_config(wl, n_cfg):
    p = wl.params
    return {"workload": f"BASELINE.json configs[{n_cfg - 1}] ({wl.name}): {'x'.join(map(str, p['ndom']))} zones in "
                        f"{wl.nboxes} boxes of {'x'.join(map(str, p['nbox']))}, {wl.ng} ghost zones, "
                        f"{wl.nspec} passive species (NVAR={wl.nvar}), gamma={p['gamma']:.6g}, cfl={p['cfl']}",
            "zones": wl.zones, "state_gb": round(wl.state_bytes / 1e9, 3),
            "l2_policy": "inputs_larger_than_l2 (every kernel streams >= 1 GB; no flush needed)"}


# ----------------------------------------------------------------------------- reference arm
def run_reference(args, rank):
    """There is no reference implementation (paper text only): this arm times the CPU oracle, as it stands, on
    this box's host cores.  `config` is the workload of our arm (the metric is a rate per zone); a STEP of this
    arm is one RK2 step of a BOUNDED SAMPLE of it -- the 256^3 instance of the same index-based recipe in 64^3 boxes
    (one eighth of the zones, about 6 s on 16 cores), or the 128^3 instance in 32^3 boxes when more than 24 steps are
    asked for; 64 boxes either way, so every core has work -- and `config.zones`, `config.sample`,
    `cpu_baseline.sample` and `ms_per_step` describe that sample, so that K + W steps end within a few minutes."""
    if rank != 0:
        return
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    n = 256 if steps + warmup <= 24 else 128
    cb, ms, wl = oracle_sample(steps, warmup, n=n)
    cb.update(host_info())
    cfg = workload_config(W.config(args.config), args.config)
    cfg["l2_policy"] = "n/a (host)"
    cfg["full_workload_zones"] = cfg["zones"]
    cfg["zones"] = wl.zones                      # what a step of THIS arm advances
    cfg["state_gb"] = round(wl.state_bytes / 1e9, 3)
    cfg["sample"] = {"workload": workload_config(wl, args.config)["workload"], "zones": wl.zones,
                     "state_gb": round(wl.state_bytes / 1e9, 3),
                     "why": "the oracle needs about 50 s per RK2 step of the 512^3 state on 16 cores; its rate per zone "
                            "does not depend on the zone count"}
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": cfg, "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "note": "no reference implementation exists (paper text only): this arm is the CPU oracle; ms_per_step is the "
                    "time of one step of config.sample, not of the 512^3 state"}
    print(json.dumps(line), flush=True)


def run_ctu(args, wl, h, host, t_gen, barrier, local_rank, world, dev):
    """--ctu: the CTU update O12.  A step = one hydro_ctu_step step: estimate_dt, ghost fill,
    ONE flux evaluation (6 Riemann solves per zone) and update.  First CUDA path of the row: its kernels keep the traced
    states and fluxes in HBM, so the roofline object is the whole step's measured-by-model bytes, not a tuned kernel's."""
    import torch
    per_box = 12 * wl.nflux * int(np.prod(wl.nt)) * 8
    nb = max(1, min(wl.nboxes, int(60e9 // per_box)))
    h.hydro_ctu_step(max(1, args.warmup), batch_boxes=nb)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    n0 = h.hydro_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(h.stream)
    h.hydro_ctu_step(args.steps, batch_boxes=nb)
    e1.record(h.stream)
    barrier()
    ms_total = reduce_max(e0.elapsed_time(e1), world, dev)
    launches = h.hydro_launch_count() - n0
    sampler.stop_flag = True
    sampler.join(timeout=10)
    peak, peak_src = measured_peaks()
    Z, nq, nvar = wl.zones, wl.nflux, wl.nvar
    # bytes per zone of one step with every intermediate array in HBM: trace reads the state
    # 3 x 5 zones deep and writes 2*NQ*3; first fluxes read 2*NQ*3, write NQ*3; final fluxes read 2*NQ*3 + 4*NQ*3,
    # write NQ*3; update reads 2*NQ*3 + NVAR, writes NVAR
    alg = Z * 8 * (3 * nvar + 6 * nq + 6 * nq + 3 * nq + 6 * nq + 12 * nq + 3 * nq + 6 * nq + 2 * nvar)
    ms_step = ms_total / args.steps
    if int(os.environ.get("RANK", "0")) == 0:
        cfg = workload_config(wl, args.config)
        cfg.update({"integrator": "CTU (O12): PPM + characteristic tracing + 6-solve transverse corrections, one update per step",
                    "batch_boxes": nb, "replicas": world,
                    "call": f"hydro_ctu_step(h, scratch, {nb} boxes per batch, {args.steps} steps) -- one C-ABI call"})
        line = {"metric": METRIC.replace("RK2", "CTU"), "value": job_value(Z, args.steps, ms_total, world), "unit": UNIT,
                "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
                "roofline": {"bound": "hbm", "kernel": "whole CTU step (first CUDA path, intermediates in HBM)",
                             "achieved": alg / 1e9 / (ms_step * 1e-3), "peak": peak, "unit": "GB/s",
                             "frac": alg / 1e9 / (ms_step * 1e-3) / peak, "traffic": None, "peak_source": peak_src,
                             "alg_bytes_per_zone_update": alg / Z},
                "cpu_baseline": None, "e2e": None, "gpu_launches": int(launches), "clocks": sampler.summary()}
        print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- our arm
def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2007_05218_b200 import binding as B
    from paper_2007_05218_b200 import build as build_mod

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the hydro path has no CPU fallback)")
    build_mod.build()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    wl = W.config(args.config)
    if args.flatten:
        wl.params["flatten"] = 1
    if args.evolve:
        wl.params["evolve_eint"] = 1
    # ---- synthetic input, generated on the host, resident in pinned memory -------------
    t0 = time.perf_counter()
    pinned = True
    try:
        host = torch.empty(wl.state_shape, dtype=torch.float64, pin_memory=True)
    except RuntimeError:
        host, pinned = torch.empty(wl.state_shape, dtype=torch.float64), False
    W.initial_state(wl, out=host.numpy(), threads=min(32, os.cpu_count() or 1))
    t_gen = time.perf_counter() - t0

    h = B.Hydro(wl.params, device=dev)
    h.U0.copy_(host.reshape(-1), non_blocking=True)
    torch.cuda.synchronize(dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    if args.ctu:
        return run_ctu(args, wl, h, host, t_gen, barrier, local_rank, world, dev)
    h.hydro_step(args.warmup, want_dt=False)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = h.hydro_launch_count()
    ns_max, split_ghosts, fuse_dt = h.hydro_query(3), bool(h.hydro_query(1)), bool(h.hydro_query(2))
    xmarch = bool(h.hydro_query(4))
    xchunk = bool(h.hydro_query(6))
    one_launch = max(0, h.hydro_query(5))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(h.stream)
    h.hydro_step(args.steps, want_dt=False)          # K whole RK2 steps, one C-ABI call; no per-launch events here
    e1.record(h.stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = h.hydro_launch_count() - launches0
    # per-class launch durations: the same call once more, with the library's event pairs around every launch
    h.hydro_profile(1)
    h.hydro_step(args.steps, want_dt=False)
    prof = h.hydro_profile_read()
    h.hydro_profile(0)
    sampler.stop_flag = True
    sampler.join(timeout=10)
    dt_last = h.hydro_estimate_dt()
    totals = h.hydro_conserved_totals(0)
    ms_total = reduce_max(ms_total, world, dev)
    ms_step = ms_total / args.steps
    value = job_value(wl.zones, args.steps, ms_total, world)

    # ---- roofline of the dominant kernel class ------------------------------------------
    peak, peak_src = measured_peaks()
    ngroups = max(1, -(-wl.nspec // ns_max)) if wl.nspec else 0
    groups = [wl.nspec // ngroups + (1 if i < wl.nspec % ngroups else 0) for i in range(ngroups)] if ngroups else []
    alg = algorithmic_bytes(wl, groups, args.steps, split_ghosts, fuse_dt, xmarch, one_launch)
    kernels = {}
    tot_ms = sum(v[0] for v in prof.values())
    for k, (ms, cnt) in prof.items():
        if cnt and k in alg:
            kernels[k] = {"ms_per_launch": ms / cnt, "launches_per_step": cnt / args.steps,
                          "share_of_step": ms / tot_ms, "alg_gb_per_launch": alg[k] / 1e9,
                          "gbs": alg[k] / 1e9 / (ms / cnt * 1e-3), "frac": alg[k] / 1e9 / (ms / cnt * 1e-3) / peak}
    # The dominant kernel is chosen by kernel FUNCTION, not by class: a class of hydro_profile_read can bundle several
    # template instances (the z sweeps exist per RK stage, the z species sweep also per group size; the x and y sweeps
    # are one function each for both stages), and a bundle must not outrank the largest single kernel.
    ndistinct = max(1, len(set(groups)))
    functions = {"sweep_x": 1 if not xmarch else 1 + ndistinct, "hydro_y": 1, "hydro_z": 2,
                 "species_y": 1 if (one_launch & 1 and ngroups >= 2 and max(groups) >= 2) else ndistinct,
                 "species_z": 2 * (1 if (one_launch & 2 and ngroups >= 2 and max(groups) >= 2) else ndistinct)}
    for k, v in kernels.items():
        v["functions"] = functions.get(k, 1)
        v["ms_per_step_of_one_function"] = v["ms_per_launch"] * v["launches_per_step"] / v["functions"]
    dom = max(kernels, key=lambda k: kernels[k]["ms_per_step_of_one_function"])
    step_alg = sum(alg[k] * kernels[k]["launches_per_step"] for k in kernels)
    roofline = {"bound": "hbm", "kernel": dom, "chosen_by": "largest time per step of a single kernel function",
                "achieved": kernels[dom]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": kernels[dom]["frac"], "traffic": None, "peak_source": peak_src,
                "whole_step": {"alg_bytes_per_zone_update": step_alg / wl.zones,
                               "gbs": step_alg / 1e9 / (ms_step * 1e-3),
                               "frac": step_alg / 1e9 / (ms_step * 1e-3) / peak,
                               "frac_of_nominal_8000": step_alg / 1e9 / (ms_step * 1e-3) / 8000.0}}
    # ncu figures of the committed capture (profiles/traffic.json, written by paper_2007_05218_b200.ncu_summary):
    # DRAM bytes and instruction counts per launch of every class.  They are used ONLY while the capture's hash
    # (kernel sources, hydro_api.cu, build flags, run-time switches) equals that of this run; with the live launch durations they give
    # traffic_ratio (measured / algorithmic bytes) and the second roofline: FP64 pipe and issue slots.
    from paper_2007_05218_b200 import ncu_summary
    tr = os.path.join(ROOT, "profiles", "traffic.json")
    fp64 = B.hydro_probe_fp64()                               # measured FP64 instr/s of this GPU, now
    clocks = sampler.summary()
    sm_hz = (clocks.get("sm_mhz") or 1965.0) * 1e6            # median SM clock sampled under load
    capture = "none"
    if os.path.exists(tr) and not (args.flatten or args.evolve):
        try:
            t = json.load(open(tr)).get(wl.name, {})
            if t.get("source_sha256") == ncu_summary.source_sha():
                capture = "profiles/traffic.json (kernel sources, hydro_api.cu, build flags and run-time switches match)"
                for k, v in kernels.items():
                    c = t["classes"].get(k)
                    if not c:
                        continue
                    sec = v["ms_per_launch"] * 1e-3
                    v["traffic"] = c["dram_bytes"]
                    v["traffic_ratio"] = c["dram_bytes"] / alg[k]
                    v["fp64_pipe_frac"] = c["fp64_warp_instr"] * 32 / sec / fp64["dfma"]
                    v["issue_slot_frac"] = c["warp_instr"] / sec / (148 * 4 * sm_hz)
            else:
                capture = "profiles/traffic.json is from other sources, flags or switches (hash differs): not used"
        except Exception as e:                                  # a malformed file must not kill the bench line
            capture = f"profiles/traffic.json unreadable ({type(e).__name__})"
    roofline["traffic"] = kernels[dom].get("traffic")
    roofline["traffic_ratio"] = kernels[dom].get("traffic_ratio")
    roofline["ncu_capture"] = capture
    roofline["alu"] = {"fp64_peak_instr_per_s": fp64["dfma"],
                       "fp64_peak_source": "hydro_probe_fp64 (libhydro_probe_b200: independent DFMA chains), this run",
                       "issue_peak_warp_instr_per_s": 148 * 4 * sm_hz,
                       "issue_peak_source": "148 SMs x 4 schedulers x the median SM clock sampled during the run",
                       "fp64_pipe_frac": kernels[dom].get("fp64_pipe_frac"), "issue_slot_frac": kernels[dom].get("issue_slot_frac")}
    isf = kernels[dom].get("issue_slot_frac")
    if isf is not None and isf > kernels[dom]["frac"]:
        # the dominant class is bound by instruction issue / the FP64 pipe, not by HBM: say so (the HBM figures stay)
        roofline["bound_note"] = (f"{dom} issues {isf:.2f} of the SM issue slots and keeps the FP64 pipe "
                                  f"{kernels[dom].get('fp64_pipe_frac'):.2f} busy while moving {kernels[dom]['frac']:.2f} of the "
                                  "HBM peak: ALU/issue-bound (DESIGN.md sec. 5)")

    # ---- e2e: the same K steps through the C-ABI call that takes HOST buffers ------------------
    # hydro_run_host(params, U_host, K): allocate, H2D of the whole state, K steps, D2H of the whole state, free --
    # all inside the timed region.  PCIe moves 2 x 24.5 GB per call, so the per-step cost is the call's divided by K.
    del h
    torch.cuda.empty_cache()
    e2e = None
    if not args.no_e2e:
        p = B.make_params(wl.params)
        B.hydro_run_host(p, host, 1)                            # warm-up (first touch of the pinned pages)
        barrier()
        t0 = time.perf_counter()
        B.hydro_run_host(p, host, args.steps)
        torch.cuda.synchronize(dev)
        el = time.perf_counter() - t0
        el = reduce_max(el, world, dev)
        e2e = {"value": job_value(wl.zones, args.steps, el * 1e3, world), "unit": UNIT,
               "h2d_bytes_per_step": wl.state_bytes / args.steps, "d2h_bytes_per_step": wl.state_bytes / args.steps,
               "h2d_bytes_per_call": wl.state_bytes, "d2h_bytes_per_call": wl.state_bytes,
               "steps": args.steps, "seconds_per_call": el, "pinned_host": pinned,
               "api": f"hydro_run_host(params, U_host, {args.steps}) -- one call: cudaMalloc, H2D, {args.steps} steps, D2H, cudaFree"}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu_baseline, _, _ = oracle_sample(3, 0)      # about 18 s of host work on all cores
        one, _, _ = oracle_sample(1, 0, n=128, threads=1)   # about 8 s on one core
        cpu_baseline["one_core"] = {"value": one["value"], "unit": UNIT, "sample": one["sample"]}
        cpu_baseline.update(host_info())

    if rank == 0:
        cfg = workload_config(wl, args.config)
        cfg.update({"replicas": world, "host_generation_s": round(t_gen, 1), "species_groups_yz": groups,
                    "flatten": bool(wl.params.get("flatten", 0)), "evolve_eint": bool(wl.params.get("evolve_eint", 0)), "split_ghost_fill": split_ghosts, "dt_fused_in_z_sweep": fuse_dt, "x_sweep": "marching (march_x.cuh)" if xmarch else ("chunk-lane (sweep_xc.cuh)" if xchunk else "one zone per lane (sweep_x.cuh)"), "species_groups_in_one_launch": {"y": bool(one_launch & 1), "z": bool(one_launch & 2)},
                    "call": f"hydro_step(h, {args.steps}) -- one C-ABI call for the K timed steps",
                    "fmad": open(B.LIB_PATH + ".flags").read() if os.path.exists(B.LIB_PATH + ".flags") else "?"})
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
                "zone_stages_per_s": 2 * value, "roofline": roofline, "kernels": kernels,
                "cpu_baseline": cpu_baseline, "e2e": e2e, "gpu_launches": int(launches),
                "clocks": clocks, "dt_last": dt_last, "total_mass": totals[0]}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def dry_run(args, rank, world, local_rank):
    """--dry-run: everything about the launch that needs no GPU.  Every rank joins a gloo process group, the ranks
    are gathered and the per-rank times go through the same reduce_max / job_value as the timed run; rank 0 prints
    the line's skeleton (no value is a measurement)."""
    import torch
    import torch.distributed as dist
    if world > 1:
        dist.init_process_group("gloo")
    seen = [rank]
    if world > 1:
        t = torch.zeros(world, dtype=torch.int64)
        t[rank] = local_rank + 1
        dist.all_reduce(t)
        seen = [r for r in range(world) if t[r] > 0]
    ms = reduce_max(1.0 + rank, world)
    wl = W.config(args.config)
    if rank == 0:
        print(json.dumps({"dry_run": True, "impl": args.impl, "metric": METRIC, "value": None, "unit": UNIT, "n_gpus": world,
                          "ranks": seen, "steps": args.steps, "warmup": args.warmup, "ms_per_step": None,
                          "max_over_ranks_check_ms": ms, "replica_aggregate_check": job_value(wl.zones, 1, 1e3, world) / wl.zones,
                          "higher_is_better": True, "scaling": "weak", "dtype": "f64", "data": "synthetic",
                          "config": workload_config(wl, args.config)}), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--flatten", action="store_true", help="switch the optional shock flattening O10 on")
    ap.add_argument("--evolve", action="store_true", help="switch the optional evolved rho*e O11 on")
    ap.add_argument("--ctu", action="store_true", help="time the CTU update O12 (hydro_ctu_step) instead of the RK2 path")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--dry-run", action="store_true",
                    help="launch check without CUDA: start the ranks, form the process group over gloo, print the line's skeleton")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # a plain `python bench.py --gpus N`: nobody has started the ranks, so start them here -- one process per
        # GPU under torch.distributed.run, exactly the launch the driver uses -- and hand back its exit code
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
        raise SystemExit(subprocess.run(cmd).returncode)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.dry_run:
        return dry_run(args, rank, world, local_rank)
    if args.impl == "reference":
        run_reference(args, rank)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
