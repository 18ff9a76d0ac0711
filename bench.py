#!/usr/bin/env python
"""bench.py -- advection grid-points/sec and achieved HBM GB/s on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload config1|config2|config3] [--xchunk X] [--group G]

A "step" is one pass of the hot path over one batch of synthetic fields:
  config1 (default, the configuration BASELINE.json's metric is quoted on):
      256x256x128 fp64, one fused u/v/w momentum call;
  config2 / config3: 512x512x256, momentum + 10 batched scalars (a1 + a2),
      fp64 / fp32 (a4).
`value` is interior grid points advected per second with inputs resident in
HBM; `e2e` is the same metric through monc_adv_step_async with PINNED HOST
buffers (H2D of the fields, kernels, D2H of the tendencies inside the timed
region).  Prints ONE JSON line (rank 0).

--impl reference times the CPU oracle (oracle/, fp64, single thread) on the
same workload: each step is one full oracle pass over the first `--ref-planes`
x planes of the workload.
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

# algorithmic bytes per interior point: every input read
# once, every output written once
BYTES_PER_PT = {"momentum": {"f64": 48, "f32": 24}}


def scalar_bytes_per_pt(nq, dtype):
    es = 8 if dtype == "f64" else 4
    return 3 * es + 2 * es * nq  # wind once + q in + sq out


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region: NVML polled from a
    thread every few ms (the timed region of config1 is milliseconds long, too
    short for `nvidia-smi -lms`); falls back to the recipe's nvidia-smi line."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0, period_s=0.004):
        self.rows, self.proc, self.index, self.period = [], None, index, period_s
        self.sm, self.reasons, self.mx, self.power = [], set(), None, []
        self._stop = threading.Event()
        self._thr = None
        self._nvml = None

    def _physical_index(self):
        vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
        try:
            return int(vis.split(",")[self.index]) if vis else self.index
        except Exception:
            return self.index

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self._physical_index())
            self.mx = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            bits = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown,
                    "hw_thermal_slowdown": nv.nvmlClocksEventReasonHwThermalSlowdown,
                    "sw_thermal_slowdown": nv.nvmlClocksEventReasonSwThermalSlowdown,
                    "sw_power_cap": nv.nvmlClocksEventReasonSwPowerCap}

            def poll():
                while not self._stop.is_set():
                    try:
                        self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                        r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                        for name, b in bits.items():
                            if r & b:
                                self.reasons.add(name)
                        self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                    except Exception:
                        pass
                    self._stop.wait(self.period)

            self._nvml = nv
            self._thr = threading.Thread(target=poll, daemon=True)
            self._thr.start()
            return
        except Exception:
            self._nvml = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-i", str(self._physical_index()), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self._nvml is not None:
            self._stop.set()
            self._thr.join(timeout=1.0)
            return {"sm_mhz": float(np.median(self.sm)) if self.sm else None,
                    "sm_min_mhz": float(np.min(self.sm)) if self.sm else None, "sm_max_mhz": self.mx,
                    "power_w_max": float(np.max(self.power)) if self.power else None,
                    "samples": len(self.sm), "reasons": sorted(self.reasons), "source": "nvml"}
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown",
                                "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx,
                "samples": len(sm), "reasons": sorted(reasons), "source": "nvidia-smi"}


def workload_cfg(name):
    from paper_2009_12850_b200 import synth
    return synth.CONFIGS[{"config1": 1, "config2": 2, "config3": 3, "config4": 4}[name]]


# ncu `dram__bytes_read.sum + dram__bytes_write.sum` per launch of the dominant
# kernel, from the committed `--set full` captures under profiles/ (bytes).  Keyed
# by (workload, kernel family); valid for the library's default launch plan only.
NCU_TRAFFIC = {
    ("config1", "tma_momentum"): (358.1e6, "profiles/r01_config1_tma_momentum_f64.md"),
    ("config2", "tma_scalars"): (12814.3e6, "profiles/r01_config2_tma_scalars_f64.md"),
    ("config3", "tma_scalars"): (6206.1e6, "profiles/r01_config3_tma_f32.md"),
    ("config2", "tma_fused"): (14273.8e6, "profiles/r01_config2_tma_fused.md"),
    ("config3", "tma_fused"): (7077.1e6, "profiles/r01_config3_tma_fused.md"),
}


# ---------------------------------------------------------------------------
# reference arm: the CPU oracle as it stands
# ---------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import dataclasses
    import oracle
    from paper_2009_12850_b200 import synth
    cfg = workload_cfg(args.workload)
    sub = dataclasses.replace(cfg, nx=min(cfg.nx, args.ref_planes))
    g = synth.grid(cfg.nz)
    P = oracle.Problem(sub.nx, sub.ny, sub.nz, sub.halo, synth.DX, synth.DY,
                       g["dz"], g["dzn"], g["rho"], g["rhon"])
    names = ["u", "v", "w"] + synth.field_names(sub)
    H = [synth.field(sub, n) for n in names]
    outs = tuple(np.zeros(P.shape) for _ in range(3))
    sq = np.zeros(P.shape)

    def step():
        P.momentum(H[0], H[1], H[2], nthreads=1, out=outs)
        for q in H[3:]:
            P.scalar(H[0], H[1], H[2], q, nthreads=1, out=sq)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    val = sub.points * args.steps / dt / 1e9
    sample = (f"oracle (fp64, 1 thread) on the first {sub.nx} of {cfg.nx} x-planes of {args.workload}"
              f" ({sub.points} pts/step, {len(names)} fields)")
    print(json.dumps({
        "impl": "reference", "metric": "advection grid-points/sec", "value": val, "unit": "Gpts/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "nx": cfg.nx, "ny": cfg.ny, "nz": cfg.nz,
                   "nq": cfg.nq, "halo": cfg.halo},
        "cpu_baseline": {"value": val, "unit": "Gpts/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "Gpts/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2009_12850_b200 import binding, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg = workload_cfg(args.workload)
    g = synth.grid(cfg.nz)
    L = binding.MoncAdv(cfg.nx, cfg.ny, cfg.nz, cfg.halo, synth.DX, synth.DY,
                        g["dz"], g["dzn"], g["rho"], g["rhon"], dtype=cfg.dtype)
    L.set_tuning(xchunk=args.xchunk, group=args.group, stages=args.stages, tile_y=args.tile_y,
                 warps=args.warps, split=args.split)
    if args.variant:
        L.set_variant(args.variant)
    if args.no_pdl:
        L.set_pdl(False)
    if args.form != "flux":
        L.set_form(args.form)
    tdt = L.torch_dtype
    # weak scaling: every rank advects its own subdomain of the config's size
    # ("replicas only" until the halo-exchange row of SURVEY.md 8(f) is built);
    # rank-keyed seed so ranks do not share data
    import dataclasses
    from paper_2009_12850_b200 import dist as pdist
    names = ["u", "v", "w"] + synth.field_names(cfg)
    if args.halo_exchange:
        # one periodic global domain of world * nx planes, x-slab per rank; the halo
        # swap runs inside every timed step
        gcfg = dataclasses.replace(cfg, nx=world * cfg.nx)
        H = []
        for n in names:
            f = pdist.local_from_global(synth.interior_field(gcfg, n), cfg.halo, world, rank)
            H.append(pdist.fill_halo_y_periodic(f, cfg.halo).numpy())
    else:
        rcfg = cfg if rank == 0 else dataclasses.replace(cfg, seed_cid=1000 + rank)
        H = [synth.field(rcfg, n) for n in names]
    nf = len(names)
    field_bytes = cfg.elems * (8 if cfg.dtype == "f64" else 4)
    # rotate between buffer sets so that no step finds its inputs in L2
    nsets = max(2, min(4, int(np.ceil(3 * 126e6 / (2 * nf * field_bytes))) + 1))
    sets = []
    for s in range(nsets):
        ins = [torch.from_numpy(a).to("cuda", dtype=tdt) for a in H]
        outs = [torch.zeros(L.shape, device="cuda", dtype=tdt) for _ in names]
        sets.append((ins, outs))
    st = torch.cuda.Stream()

    def step(s):
        ins, outs = sets[s % nsets]
        if args.halo_exchange:
            pdist.exchange_halo_x(ins, cfg.halo)
        L.momentum(ins[0], ins[1], ins[2], outs[0], outs[1], outs[2], stream=st)
        if nf > 3:
            L.scalars(ins[3:], outs[3:], stream=st)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    with torch.cuda.stream(st):
        for s in range(args.warmup):
            step(s)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    n0 = L.launch_count()
    # Events are recorded on the launch stream.  Momentum-only workloads: one event
    # every `grp` launches (an event between two launches costs ~1 us of stream time
    # and defeats the programmatic dependent launch of back-to-back kernels), so the
    # mean launch duration is (event span) / grp.  With scalars: one event between
    # the two kernels of a step as well.
    split = nf > 3 or args.halo_exchange
    grp = 1 if split else max(1, min(args.event_every, args.steps))
    marks = []  # (kind, event)
    with torch.cuda.stream(st):
        e0 = torch.cuda.Event(enable_timing=True)
        e0.record(st)
        marks.append(("start", e0))
        for s in range(args.steps):
            ins, outs = sets[(args.warmup + s) % nsets]
            if args.halo_exchange:
                pdist.exchange_halo_x(ins, cfg.halo)
                e = torch.cuda.Event(enable_timing=True); e.record(st); marks.append(("swap", e))
            L.momentum(ins[0], ins[1], ins[2], outs[0], outs[1], outs[2], stream=st)
            if split or (s + 1) % grp == 0 or s + 1 == args.steps:
                e = torch.cuda.Event(enable_timing=True); e.record(st); marks.append(("mom", e))
            if nf > 3:
                L.scalars(ins[3:], outs[3:], stream=st)
                e = torch.cuda.Event(enable_timing=True); e.record(st); marks.append(("sca", e))
    barrier()
    launches = L.launch_count() - n0
    plan = L.describe_plan()
    total_ms = marks[0][1].elapsed_time(marks[-1][1])
    span = {"swap": 0.0, "mom": 0.0, "sca": 0.0}
    best = {"swap": 1e30, "mom": 1e30, "sca": 1e30}
    done = 0
    for (k0_, a), (k1_, b) in zip(marks[:-1], marks[1:]):
        ms = a.elapsed_time(b)
        span[k1_] += ms
        n_in = 1
        if k1_ == "mom" and not split:
            n_in = min(grp, args.steps - done)
            done += n_in
        best[k1_] = min(best[k1_], ms / n_in)
    mom_avg, sca_avg, swap_avg = (span[k] / args.steps for k in ("mom", "sca", "swap"))
    if world > 1:
        t = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    value = world * cfg.points * args.steps / (total_ms * 1e-3) / 1e9

    # ---- the same step through monc_adv_tendencies (one fused launch where it fits):
    # supplementary; `value` above stays the two north_star calls
    fused = None
    if nf > 3 and not args.halo_exchange:
        fsteps = args.steps
        # the board's power controller averages over ~1 s: let it settle so
        # this loop starts from the same state as the two-call loop above did
        barrier()
        time.sleep(2.0)
        n1 = L.launch_count()
        with torch.cuda.stream(st):
            for s in range(3):
                ins, outs = sets[s % nsets]
                L.tendencies(ins[0], ins[1], ins[2], outs[0], outs[1], outs[2], ins[3:], outs[3:], stream=st)
            f0 = torch.cuda.Event(enable_timing=True); f0.record(st)
            for s in range(fsteps):
                ins, outs = sets[(3 + s) % nsets]
                L.tendencies(ins[0], ins[1], ins[2], outs[0], outs[1], outs[2], ins[3:], outs[3:], stream=st)
            f1 = torch.cuda.Event(enable_timing=True); f1.record(st)
        barrier()
        ftot = f0.elapsed_time(f1)
        if world > 1:
            t = torch.tensor([ftot], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ftot = float(t.item())
        fms = ftot / fsteps
        es_ = 8 if cfg.dtype == "f64" else 4
        fb_ = (6 + 2 * cfg.nq) * es_ * cfg.points  # u, v, w read once; 3 + nq outputs; nq scalars read
        fused = {"call": "monc_adv_tendencies", "ms_per_step": fms, "value": world * cfg.points / (fms * 1e-3) / 1e9,
                 "unit": "Gpts/s", "algorithmic_bytes_per_step": fb_, "algorithmic_GBs": fb_ / (fms * 1e-3) / 1e9,
                 "steps": fsteps, "launches": (L.launch_count() - n1) * fsteps // (fsteps + 3),
                 "launches_per_step": (L.launch_count() - n1) / (fsteps + 3),
                 "launch_plan": L.describe_plan()}

    clocks = sampler.stop() if rank == 0 else None

    # ---- end to end through the host-buffer entry point (a3)
    hin = [torch.empty(L.shape, dtype=tdt, pin_memory=True) for _ in names]
    for t_, a in zip(hin, H):
        t_.copy_(torch.from_numpy(a))
    hout = [torch.zeros(L.shape, dtype=tdt, pin_memory=True) for _ in names]
    L.set_chunks(args.chunks)

    enqueue_s = [0.0]

    def e2e_step():
        te = time.perf_counter()
        L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
        enqueue_s[0] += time.perf_counter() - te  # the host is free from here
        L.step_wait()

    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    for _ in range(2):
        e2e_step()
    barrier()
    enqueue_s[0] = 0.0
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    enqueue_ms = enqueue_s[0] / e2e_steps * 1e3
    phase = L.step_times_ms()
    # the same step with copies and kernels serialised on one stream: its phases are
    # the "alone" times of the overlap ratio
    L.set_overlap(False)
    e2e_step()
    torch.cuda.synchronize()
    serial = L.step_times_ms()
    L.set_overlap(True)
    if world > 1:
        t = torch.tensor([e2e_s], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    es = 8 if cfg.dtype == "f64" else 4
    plane_b = (cfg.ny + 2 * cfg.halo) * cfg.nz * es
    h2d_b = nf * (cfg.nx + 2) * plane_b
    d2h_b = nf * cfg.points * es
    e2e_val = world * cfg.points * e2e_steps / e2e_s / 1e9

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel
    peak, peak_src = peaks()
    mom_b = BYTES_PER_PT["momentum"][cfg.dtype] * cfg.points
    sca_b = scalar_bytes_per_pt(cfg.nq, cfg.dtype) * cfg.points if cfg.nq else 0
    if sca_b and sca_avg > mom_avg:
        kern, kb, kms = "scalars", sca_b, sca_avg
    else:
        kern, kb, kms = "momentum", mom_b, mom_avg
    fam = {"": "tma", "auto": "tma", "tma": "tma", "march": "march", "generic": "generic"}[args.variant]
    tsuf = "double" if cfg.dtype == "f64" else "float"
    achieved = kb / (kms * 1e-3) / 1e9
    traffic, traffic_src = args.traffic, "--traffic"
    tuned = any((args.xchunk, args.group, args.stages, args.tile_y, args.warps, args.split)) or args.form != "flux"
    if traffic is None and not tuned:
        traffic, traffic_src = NCU_TRAFFIC.get((args.workload, f"{fam}_{kern}"), (None, None))
    roofline = {"bound": "hbm", "kernel": f"{fam}_{kern}<{tsuf}>", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": kb, "avg_launch_ms": kms,
                "best_launch_ms": best["mom" if kern == "momentum" else "sca"],
                "launches_per_event": grp if kern == "momentum" else 1,
                "frac_of_nominal_8TBs": achieved / 8000.0,
                # BASELINE.json's "achieved HBM GB/s from ncu": the profiled DRAM bytes of
                # one launch over this run's measured launch time
                "ncu_dram_GBs": (traffic / (kms * 1e-3) / 1e9) if traffic else None}
    two_calls = {"value": value, "ms_per_step": total_ms / args.steps, "gpu_launches": launches,
                 "dominant_kernel_roofline": dict(roofline)}
    ms_per_step = total_ms / args.steps
    if fused is not None and not args.two_calls:
        # the whole step through monc_adv_tendencies is the headline; its kernel the roofline's
        value, ms_per_step, launches, plan = fused["value"], fused["ms_per_step"], fused["launches"], fused["launch_plan"]
        if "tma_fused" in plan:
            ach = fused["algorithmic_bytes_per_step"] / (fused["ms_per_step"] * 1e-3) / 1e9
            traffic, traffic_src = args.traffic, "--traffic"
            if traffic is None and not tuned:
                traffic, traffic_src = NCU_TRAFFIC.get((args.workload, "tma_fused"), (None, None))
            roofline = {"bound": "hbm", "kernel": f"tma_scalars<{tsuf}, MOM=1> (fused momentum + scalars)",
                        "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": traffic,
                        "traffic_source": traffic_src, "peak_source": peak_src,
                        "algorithmic_bytes_per_launch": fused["algorithmic_bytes_per_step"],
                        "avg_launch_ms": fused["ms_per_step"], "launches_per_event": fused["steps"],
                        "frac_of_nominal_8TBs": ach / 8000.0,
                        "ncu_dram_GBs": (traffic / (fused["ms_per_step"] * 1e-3) / 1e9) if traffic else None}
    kernels = {"momentum_ms": mom_avg, "momentum_GBs": mom_b / (mom_avg * 1e-3) / 1e9}
    if args.halo_exchange:
        kernels["halo_swap_ms"] = swap_avg
    if sca_b:
        kernels.update({"scalars_ms": sca_avg, "scalars_GBs": sca_b / (sca_avg * 1e-3) / 1e9})

    # ---- the oracle beside it: bounded sample on this box's host cores
    cpu = cpu_baseline(cfg, args)

    out = {
        "metric": "advection grid-points/sec", "value": value, "unit": "Gpts/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype,
        "data": "synthetic",
        "config": {"workload": args.workload, "nx": cfg.nx, "ny": cfg.ny, "nz": cfg.nz,
                   "halo": cfg.halo, "nq": cfg.nq, "fields_per_step": nf,
                   "l2": f"rotating {nsets} buffer sets ({nsets * 2 * nf * field_bytes / 1e6:.0f} MB) > 126 MB L2",
                   "parallelism": ("x-slab decomposition, halo swap every step" if args.halo_exchange
                                   else ("replicas only" if world > 1 else "1 GPU")),
                   "variant": args.variant or "auto", "xchunk": args.xchunk, "group": args.group,
                   "stages": args.stages, "tile_y": args.tile_y, "warps": args.warps,
                   "split": args.split, "pdl": not args.no_pdl, "form": args.form,
                   "step_call": ("monc_adv_tendencies" if (fused is not None and not args.two_calls)
                                 else ("monc_adv_momentum + monc_adv_scalars" if nf > 3 else "monc_adv_momentum")),
                   "launch_plan": plan},
        "roofline": roofline, "kernels": kernels, "fused_step": fused,
        "two_call_step": two_calls if fused is not None else None, "cpu_baseline": cpu,
        "e2e": {"value": e2e_val, "unit": "Gpts/s", "h2d_bytes_per_step": h2d_b,
                "d2h_bytes_per_step": d2h_b, "steps": e2e_steps, "ms_per_step": e2e_s / e2e_steps * 1e3,
                "host_enqueue_ms_per_step": enqueue_ms,
                "h2d_GBs": h2d_b / (phase["h2d"] * 1e-3) / 1e9, "d2h_GBs": d2h_b / (phase["d2h"] * 1e-3) / 1e9,
                "phase_ms": phase, "chunks": args.chunks, "serial_phase_ms": serial,
                "overlap_ratio": (serial["h2d"] + serial["kernels"] + serial["d2h"]) / phase["total"],
                "timing": "host wall clock around step_async + step_wait, pinned host buffers"},
        "gpu_launches": launches, "clocks": clocks,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------
# config4: the paper's hybrid asynchronous step as the step
# ---------------------------------------------------------------------------
def run_hybrid(args):
    """1024x1024x160 fp64, 3 momentum + 4 scalars in PINNED HOST memory; a step is
    monc_adv_step_async (8 x-slab chunks H2D -> kernels -> D2H on three streams)
    + monc_adv_step_wait.  Fields are perturbed on the host between steps
    (BASELINE.json configs[4]), outside the timed region: the time of a step is
    the library's device-event span first copy -> last copy, summed over steps."""
    import torch
    from paper_2009_12850_b200 import binding, synth
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("config4 is a single-GPU workload (one host link)")
    torch.cuda.set_device(0)
    cfg = workload_cfg("config4")
    g = synth.grid(cfg.nz)
    L = binding.MoncAdv(cfg.nx, cfg.ny, cfg.nz, cfg.halo, synth.DX, synth.DY,
                        g["dz"], g["dzn"], g["rho"], g["rhon"], dtype=cfg.dtype)
    L.set_chunks(args.chunks)
    names = ["u", "v", "w"] + synth.field_names(cfg)
    nf = len(names)
    hin = []
    for n in names:
        t = torch.empty(L.shape, dtype=L.torch_dtype, pin_memory=True)
        t.copy_(torch.from_numpy(synth.field(cfg, n)))
        hin.append(t)
    hout = [torch.zeros(L.shape, dtype=L.torch_dtype, pin_memory=True) for _ in names]

    def step():
        L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
        L.step_inputs_consumed()
        L.step_wait()
        return L.step_times_ms()

    for _ in range(max(1, min(args.warmup, 3))):
        step()
    sampler = ClockSampler(0, period_s=0.05)
    sampler.start()
    n0 = L.launch_count()
    phases = []
    for s_ in range(args.steps):
        if not args.no_perturb:
            for n, t in zip(names, hin):
                synth.perturb(cfg, n, t.numpy(), s_ + 1)
        phases.append(step())
    launches = L.launch_count() - n0
    clocks = sampler.stop()
    L.set_overlap(False)
    serial = step()
    L.set_overlap(True)
    plan = L.describe_plan()
    tot_ms = float(np.sum([p_["total"] for p_ in phases]))
    es = 8
    plane_b = (cfg.ny + 2 * cfg.halo) * cfg.nz * es
    h2d_b = nf * (cfg.nx + 2) * plane_b
    d2h_b = nf * cfg.points * es
    value = cfg.points * args.steps / (tot_ms * 1e-3) / 1e9
    med = {k: float(np.median([p_[k] for p_ in phases])) for k in phases[0]}
    peak, peak_src = peaks()
    kb = (BYTES_PER_PT["momentum"]["f64"] + scalar_bytes_per_pt(cfg.nq, "f64")) * cfg.points
    ach = kb / (serial["kernels"] * 1e-3) / 1e9
    e2e = {"value": value, "unit": "Gpts/s", "h2d_bytes_per_step": h2d_b, "d2h_bytes_per_step": d2h_b,
           "steps": args.steps, "ms_per_step": tot_ms / args.steps, "chunks": args.chunks,
           "h2d_GBs": h2d_b / (med["h2d"] * 1e-3) / 1e9, "d2h_GBs": d2h_b / (med["d2h"] * 1e-3) / 1e9,
           "link_alone_GBs": {"h2d": h2d_b / (serial["h2d"] * 1e-3) / 1e9,
                              "d2h": d2h_b / (serial["d2h"] * 1e-3) / 1e9},
           "phase_ms_median": med, "serial_phase_ms": serial,
           "overlap_ratio": (serial["h2d"] + serial["kernels"] + serial["d2h"]) / med["total"]}
    print(json.dumps({
        "metric": "advection grid-points/sec", "value": value, "unit": "Gpts/s", "n_gpus": 1,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config4", "nx": cfg.nx, "ny": cfg.ny, "nz": cfg.nz, "halo": cfg.halo,
                   "nq": cfg.nq, "fields_per_step": nf, "chunks": args.chunks,
                   "perturbed_each_step": not args.no_perturb,
                   "l2": f"inputs stream from pinned host memory ({h2d_b / 1e9:.2f} GB per step) > 126 MB L2",
                   "timing": "device events inside the library, first H2D -> last D2H, summed over steps",
                   "launch_plan": plan},
        "roofline": {"bound": "hbm", "kernel": "tma_momentum<double> + tma_scalars<double> per chunk",
                     "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None,
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": kb,
                     "avg_launch_ms": serial["kernels"],
                     "note": "kernel time = sum over the 8 chunks, copies not overlapping; the step itself is host-link bound"},
        "cpu_baseline": cpu_baseline(cfg, args), "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
    }))


def cpu_baseline(cfg, args):
    import dataclasses
    import oracle
    from paper_2009_12850_b200 import synth
    sub = dataclasses.replace(cfg, nx=min(cfg.nx, args.ref_planes))
    g = synth.grid(cfg.nz)
    P = oracle.Problem(sub.nx, sub.ny, sub.nz, sub.halo, synth.DX, synth.DY,
                       g["dz"], g["dzn"], g["rho"], g["rhon"])
    names = ["u", "v", "w"] + synth.field_names(sub)
    H = [synth.field(sub, n) for n in names]
    outs = tuple(np.zeros(P.shape) for _ in range(3))
    sq = np.zeros(P.shape)
    reps, t0 = 0, time.perf_counter()
    while True:
        P.momentum(H[0], H[1], H[2], nthreads=1, out=outs)
        for q in H[3:]:
            P.scalar(H[0], H[1], H[2], q, nthreads=1, out=sq)
        reps += 1
        dt = time.perf_counter() - t0
        if dt > args.cpu_seconds:
            break
    # the same loops threaded over (i, j) on every host core
    nthr = oracle.max_threads()
    reps_all, t1 = 0, time.perf_counter()
    while True:
        P.momentum(H[0], H[1], H[2], nthreads=nthr, out=outs)
        for q in H[3:]:
            P.scalar(H[0], H[1], H[2], q, nthreads=nthr, out=sq)
        reps_all += 1
        dt_all = time.perf_counter() - t1
        if dt_all > args.cpu_seconds / 3:
            break
    return {"value": sub.points * reps / dt / 1e9, "unit": "Gpts/s", "cores": 1, "kind": "oracle",
            "sample": f"{reps} oracle passes (fp64, 1 thread) over the first {sub.nx} of {cfg.nx}"
                      f" x-planes of {args.workload}, {len(names)} fields, {dt:.1f} s",
            "all_cores": {"value": sub.points * reps_all / dt_all / 1e9, "unit": "Gpts/s", "cores": nthr,
                          "sample": f"{reps_all} passes of the same sample, {dt_all:.1f} s"},
            "host_cores_available": len(os.sched_getaffinity(0))}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config1", choices=["config1", "config2", "config3", "config4"])
    ap.add_argument("--xchunk", type=int, default=0)
    ap.add_argument("--group", type=int, default=0)
    ap.add_argument("--stages", type=int, default=0)
    ap.add_argument("--tile-y", type=int, default=0)
    ap.add_argument("--warps", type=int, default=0)
    ap.add_argument("--split", type=int, default=0)
    ap.add_argument("--variant", default="", choices=["", "auto", "generic", "march", "tma"])
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--event-every", type=int, default=10,
                    help="momentum-only workloads: launches between two timing events")
    ap.add_argument("--no-pdl", action="store_true", help="plain stream order between kernels")
    ap.add_argument("--two-calls", action="store_true",
                    help="headline = monc_adv_momentum + monc_adv_scalars instead of monc_adv_tendencies")
    ap.add_argument("--form", default="flux", choices=["flux", "pw_skew"],
                    help="flux form (default, BASELINE.json) or the Piacsek-Williams skew form (DESIGN.md R4)")
    ap.add_argument("--ref-planes", type=int, default=64)
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--halo-exchange", action="store_true",
                    help="N ranks advect x-slabs of ONE periodic domain of N*nx planes and swap halos over NCCL every step"
                         " (default: independent replicas, no data-path collective)")
    ap.add_argument("--chunks", type=int, default=8, help="x-slab chunks per hybrid step (BASELINE.json config 4: 8)")
    ap.add_argument("--no-perturb", action="store_true", help="config4: keep the fields fixed between steps")
    ap.add_argument("--traffic", type=float, default=None,
                    help="ncu dram bytes per launch of the dominant kernel, if known")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = {"config1": 1000, "config2": 100, "config3": 200, "config4": 10}[args.workload]
        if args.impl == "reference":
            args.steps = 5
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    elif args.workload == "config4":
        run_hybrid(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
