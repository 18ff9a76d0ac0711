#!/usr/bin/env python
"""bench.py -- advection grid-points/sec and achieved HBM GB/s on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload config1|config2|config3|config4] [--no-others]

A "step" is one pass of the whole hot path over one batch of synthetic fields.
The default workload is BASELINE.json's config 2, the largest single-GPU
kernel configuration: 512x512x256 fp64, the three momentum fields plus ten
scalars (every prognostic is advected), the whole step through
ONE call, monc_adv_tendencies (one fused launch).  `value` is interior grid
points advected per second over the K timed steps with inputs resident in HBM;
`e2e` is the same metric through monc_adv_step_async with PINNED HOST buffers
(H2D of the fields, kernels, D2H of the tendencies inside the timed region,
SURVEY.md 8(a) a3).  The same line carries a >= 2 s `sustained` record of the
headline step (the board reaches its power cap within a second), the two
north_star calls timed kernel by kernel, and compact records of the other
BASELINE configs (`other_configs`: config1 momentum only, config3 fp32 with its end-to-end step, a ragged-nz shape, config4
the hybrid step from host memory).  Prints ONE JSON line (rank 0).

--impl reference times the CPU oracle (oracle/, fp64, single thread) on the
same workload: each step is one full oracle pass over the first `--ref-planes`
x planes of the workload.
"""
import argparse
import dataclasses
import gc
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

NOMINAL_GBS = 8000.0  # BASELINE.json: "B200's ~8 TB/s peak", the denominator of the 70 % target


def es_of(dtype):
    return 8 if dtype == "f64" else 4


# algorithmic bytes per interior point: every input read once,
# every output written once
def bytes_momentum(dtype):
    return 6 * es_of(dtype)


def bytes_scalars(nq, dtype):
    return (3 + 2 * nq) * es_of(dtype)  # wind once + q in + sq out


def bytes_fused(nq, dtype):
    return (6 + 2 * nq) * es_of(dtype)  # u, v, w read once for momentum AND scalars


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region: NVML polled from a
    thread every few ms (a timed region can be milliseconds long, too short for
    `nvidia-smi -lms`); falls back to the recipe's nvidia-smi line."""
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
            return self
        except Exception:
            self._nvml = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-i", str(self._physical_index()), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None
        return self

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


def config_record(cfg, workload, **extra):
    """The `config` object: the same keys for our arm and for the reference arm."""
    nf = 3 + cfg.nq
    d = {"workload": workload, "nx": cfg.nx, "ny": cfg.ny, "nz": cfg.nz, "halo": cfg.halo, "nq": cfg.nq,
         "fields_per_step": nf, "storage_dtype": cfg.dtype}
    d.update(extra)
    return d


# ncu `dram__bytes_read.sum + dram__bytes_write.sum` per launch of the dominant
# kernel, from the committed `--set full` captures under profiles/ (bytes).  Keyed
# by (workload, kernel family); valid for the library's default launch plan only.
NCU_TRAFFIC = {
    ("config1", "tma_momentum"): (356.8e6, "profiles/r02_config1_tma_momentum.md"),
    ("config2", "tma_fused"): (14600.6e6, "profiles/r02_config2_tma_fused.md"),
    ("config3", "tma_fused"): (7109.4e6, "profiles/r02_config3_tma_fused.md"),
}


def roofline_record(kernel, alg_bytes, ms, launches_per_event, traffic_key, tuned, args):
    peak, peak_src = peaks()
    ach = alg_bytes / (ms * 1e-3) / 1e9
    traffic, traffic_src = args.traffic, "--traffic"
    if traffic is None:
        traffic, traffic_src = (None, None) if tuned else NCU_TRAFFIC.get(traffic_key, (None, None))
        if traffic_src:
            traffic_src = "committed ncu --set full capture, not re-measured in this run: " + traffic_src
    return {"bound": "hbm", "kernel": kernel, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
            "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
            "algorithmic_bytes_per_launch": alg_bytes, "avg_launch_ms": ms, "launches_per_event": launches_per_event,
            "frac_of_nominal_8TBs": ach / NOMINAL_GBS,
            # BASELINE.json's "achieved HBM GB/s from ncu": the profiled DRAM bytes of one launch
            # over this run's measured launch time
            "ncu_dram_GBs": (traffic / (ms * 1e-3) / 1e9) if traffic else None}


# ---------------------------------------------------------------------------
# reference arm: the CPU oracle as it stands
# ---------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
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
        "config": config_record(cfg, args.workload, l2="host memory", parallelism="1 host thread",
                                step_call="oracle momentum + scalar passes (CPU)", variant="oracle", xchunk=0,
                                group=0, stages=0, tile_y=0, warps=0, split=0, pdl=False, form=args.form,
                                launch_plan="none (CPU loops)"),
        "cpu_baseline": {"value": val, "unit": "Gpts/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "Gpts/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------
class Ctx:
    """torch.distributed plumbing shared by the legs of one run."""

    def __init__(self):
        import torch
        self.torch = torch
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
        torch.cuda.set_device(self.local)
        if self.world > 1:
            import torch.distributed as dist
            # the communicator's own log (one "comm ... nranks N" line per rank) goes to stderr,
            # so that a reader of the run can see that N ranks took part; stdout stays one JSON line
            os.environ.setdefault("NCCL_DEBUG", "INFO")
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
            os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
            dist.init_process_group("nccl", device_id=torch.device("cuda", self.local))
            self.dist = dist

    def barrier(self):
        self.torch.cuda.synchronize()
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def max_over_ranks(self, v):
        if self.world == 1:
            return float(v)
        t = self.torch.tensor([v], device="cuda", dtype=self.torch.float64)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def close(self):
        if self.world > 1:
            self.dist.destroy_process_group()


def make_library(cfg, args):
    from paper_2009_12850_b200 import binding, synth
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
    return L


def is_tuned(args):
    return any((args.xchunk, args.group, args.stages, args.tile_y, args.warps, args.split, args.variant)) \
        or args.form != "flux"


def host_fields(cfg, rank, cache):
    """Seeded fp64 host fields of a config; config 3 reuses config 2's (same seeds)."""
    from paper_2009_12850_b200 import synth
    names = ["u", "v", "w"] + synth.field_names(cfg)
    rcfg = cfg if rank == 0 else dataclasses.replace(cfg, seed_cid=1000 + rank)  # ranks do not share data
    key = (rcfg.seed, cfg.nx, cfg.ny, cfg.nz, cfg.halo, cfg.nq)
    if key not in cache:
        cache.clear()
        cache[key] = [synth.field(rcfg, n) for n in names]
    return names, cache[key]


def timed_loop(ctx, st, fn, nsteps, warm=0):
    """fn(i) enqueues step i on stream st; device time of nsteps back-to-back steps (ms)."""
    torch = ctx.torch
    with torch.cuda.stream(st):
        for i in range(warm):
            fn(i)
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for i in range(nsteps):
            fn(warm + i)
        e1.record(st)
    return e0, e1


def run_device_config(ctx, args, workload, cache, headline):
    """Configs 1-3: fields resident in HBM.  headline=True: the full record (K timed
    steps, two-call breakdown, sustained loop, e2e, cpu_baseline); else a compact one."""
    torch = ctx.torch
    from paper_2009_12850_b200 import dist as pdist
    cfg = workload_cfg(workload)
    L = make_library(cfg, args)
    tdt = L.torch_dtype
    names, H = host_fields(cfg, ctx.rank, cache)
    if args.halo_exchange and headline:
        from paper_2009_12850_b200 import synth
        # one periodic global domain of world * nx planes, x-slab per rank; the halo
        # swap runs inside every timed step
        gcfg = dataclasses.replace(cfg, nx=ctx.world * cfg.nx)
        H = []
        for n in names:
            f = pdist.local_from_global(synth.interior_field(gcfg, n), cfg.halo, ctx.world, ctx.rank)
            H.append(pdist.fill_halo_y_periodic(f, cfg.halo).numpy())
    nf, nq = len(names), cfg.nq
    es = es_of(cfg.dtype)
    field_bytes = cfg.elems * es
    # rotate between buffer sets so that no step finds its inputs in L2
    nsets = max(2, min(4, int(np.ceil(3 * 126e6 / (2 * nf * field_bytes))) + 1))
    sets = []
    for s in range(nsets):
        ins = [torch.from_numpy(a).to("cuda", dtype=tdt) for a in H]
        outs = [torch.zeros(L.shape, device="cuda", dtype=tdt) for _ in names]
        sets.append((ins, outs))
    st = torch.cuda.Stream()
    swap = args.halo_exchange and headline

    def whole_step(i):  # the step as a user makes it: ONE call when there are scalars
        ins, outs = sets[i % nsets]
        if swap:
            pdist.exchange_halo_x(ins, cfg.halo)
        if nq:
            L.tendencies(ins[0], ins[1], ins[2], outs[0], outs[1], outs[2], ins[3:], outs[3:], stream=st)
        else:
            L.momentum(ins[0], ins[1], ins[2], outs[0], outs[1], outs[2], stream=st)

    alg = (bytes_fused(nq, cfg.dtype) if nq else bytes_momentum(cfg.dtype)) * cfg.points
    steps = args.steps if headline else max(20, min(200, int(0.02 / (alg / 6.0e12))))
    warm = args.warmup if headline else 3

    # ---- the headline timed region: `steps` whole steps back to back
    with torch.cuda.stream(st):
        for i in range(warm):
            whole_step(i)
    ctx.barrier()
    sampler = ClockSampler(ctx.local).start() if ctx.rank == 0 else None
    n0 = L.launch_count()
    e0, e1 = timed_loop(ctx, st, whole_step, steps)
    ctx.barrier()
    clocks = sampler.stop() if sampler else None
    launches = L.launch_count() - n0
    total_ms = ctx.max_over_ranks(e0.elapsed_time(e1))
    ms_per_step = total_ms / steps
    value = ctx.world * cfg.points / (ms_per_step * 1e-3) / 1e9
    plan = L.describe_plan()
    tsuf = "double" if cfg.dtype == "f64" else "float"
    fam = "tma" if ("tma_" in plan) else ("march" if "march_" in plan else "generic")
    if nq and "tma_fused" in plan:
        kname, tkey = f"tma_scalars<{tsuf}, MOM=1> (fused momentum + scalars)", (workload, "tma_fused")
    elif nq:
        kname, tkey = f"{fam}_momentum<{tsuf}> + {fam}_scalars<{tsuf}> (not fused)", (workload, None)
    else:
        kname, tkey = f"{fam}_momentum<{tsuf}>", (workload, f"{fam}_momentum")
    roof = roofline_record(kname, alg, ms_per_step, steps, tkey, is_tuned(args), args)
    rec = {"value": value, "unit": "Gpts/s", "ms_per_step": ms_per_step, "steps": steps, "warmup": warm,
           "dtype": cfg.dtype, "gpu_launches": launches, "launch_plan": plan, "roofline": roof, "clocks": clocks,
           "config": config_record(
               cfg, workload,
               l2=f"rotating {nsets} buffer sets ({nsets * 2 * nf * field_bytes / 1e6:.0f} MB) > 126 MB L2",
               parallelism=("x-slab decomposition, halo swap every step" if swap
                            else ("replicas only" if ctx.world > 1 else "1 GPU")),
               step_call="monc_adv_tendencies" if nq else "monc_adv_momentum",
               variant=args.variant or "auto", xchunk=args.xchunk, group=args.group, stages=args.stages,
               tile_y=args.tile_y, warps=args.warps, split=args.split, pdl=not args.no_pdl, form=args.form,
               launch_plan=plan)}

    rec["field_points_per_s_G"] = value * nf  # grid points x advected fields
    if headline and not swap:
        # SURVEY.md 8(d) timing protocol: >= 20 launches timed one by one, median and best
        ctx.barrier()
        evs = []
        with torch.cuda.stream(st):
            for i in range(3):
                whole_step(i)
            for i in range(21):
                e = torch.cuda.Event(enable_timing=True)
                e.record(st)
                evs.append(e)
                if i < 20:
                    whole_step(i)
        ctx.barrier()
        per = sorted(a.elapsed_time(b) for a, b in zip(evs[:-1], evs[1:]))
        rec["roofline"]["per_launch_ms"] = {"launches": 20, "median": float(np.median(per)), "best": per[0],
                                            "median_GBs": alg / (float(np.median(per)) * 1e-3) / 1e9,
                                            "best_GBs": alg / (per[0] * 1e-3) / 1e9}
    # ---- sustained: the same step for >= args.sustain_seconds (the board reaches its power
    # cap within about a second; sw_power_cap is noted, not rejected)
    if args.sustain_seconds > 0 and not swap:
        nsus = max(steps, int(np.ceil(args.sustain_seconds * 1e3 / ms_per_step)))
        ctx.barrier()
        sm = ClockSampler(ctx.local, period_s=0.02).start() if ctx.rank == 0 else None
        s0, s1 = timed_loop(ctx, st, whole_step, nsus)
        ctx.barrier()
        sclk = sm.stop() if sm else None
        sms = ctx.max_over_ranks(s0.elapsed_time(s1)) / nsus
        sg = alg / (sms * 1e-3) / 1e9
        rec["sustained"] = {"steps": nsus, "seconds": sms * nsus * 1e-3, "ms_per_step": sms,
                            "value": ctx.world * cfg.points / (sms * 1e-3) / 1e9, "algorithmic_GBs": sg,
                            "frac": sg / roof["peak"], "frac_of_nominal_8TBs": sg / NOMINAL_GBS, "clocks": sclk}
    # ---- calibration: a plain device copy that moves the same number of bytes per launch (half read, half
    # written), timed the same way: what this board gives a kernel with no arithmetic, burst and sustained
    if headline and not swap and ctx.world == 1:
        try:
            n8 = int(alg // 16)
            csrc = [torch.empty(n8, device="cuda", dtype=torch.float64).normal_() for _ in range(2)]
            cdst = [torch.empty(n8, device="cuda", dtype=torch.float64) for _ in range(2)]

            def copy_step(i):
                cdst[i % 2].copy_(csrc[i % 2])

            time.sleep(2.0)
            c0, c1 = timed_loop(ctx, st, copy_step, 20, warm=3)
            ctx.barrier()
            cb = c0.elapsed_time(c1) / 20
            ncs = max(20, int(np.ceil(min(args.sustain_seconds, 1.5) * 1e3 / cb)))
            c0, c1 = timed_loop(ctx, st, copy_step, ncs)
            ctx.barrier()
            cs = c0.elapsed_time(c1) / ncs
            moved = 2 * n8 * 8
            rec["copy_same_bytes"] = {"bytes_per_launch": moved, "burst_GBs": moved / (cb * 1e-3) / 1e9,
                                      "sustained_GBs": moved / (cs * 1e-3) / 1e9, "sustained_steps": ncs,
                                      "kernel_over_copy_burst": None, "kernel_over_copy_sustained": None,
                                      "note": "torch copy_ (not this library's kernel), same stream, same event timing"}
            del csrc, cdst
            torch.cuda.empty_cache()
        except Exception as e:  # calibration only
            rec["copy_same_bytes"] = {"error": f"{type(e).__name__}: {e}"}
    # ---- burst: 20 steps from an idle board, if the headline region was not already that
    if headline and steps > 40 and not swap:
        ctx.barrier()
        time.sleep(2.0)
        b0, b1 = timed_loop(ctx, st, whole_step, 20, warm=3)
        ctx.barrier()
        bms = ctx.max_over_ranks(b0.elapsed_time(b1)) / 20
        bg = alg / (bms * 1e-3) / 1e9
        rec["burst"] = {"steps": 20, "ms_per_step": bms, "value": ctx.world * cfg.points / (bms * 1e-3) / 1e9,
                        "algorithmic_GBs": bg, "frac": bg / roof["peak"], "frac_of_nominal_8TBs": bg / NOMINAL_GBS}
    # ---- the paper's work-scaling experiment: the flux arithmetic of every
    # point evaluated 16 times on the same bytes (ULTIMATE's cost); same results
    if headline and not swap and not is_tuned(args) and not args.no_work_scale:
        ctx.barrier()
        time.sleep(1.0)
        L.set_work_scale(16)
        w0, w1 = timed_loop(ctx, st, whole_step, 10, warm=2)
        ctx.barrier()
        L.set_work_scale(1)
        wms = ctx.max_over_ranks(w0.elapsed_time(w1)) / 10
        rec["work_scale_16"] = {"steps": 10, "ms_per_step": wms, "ratio_to_x1": wms / ms_per_step,
                                "value": ctx.world * cfg.points / (wms * 1e-3) / 1e9,
                                "note": "kernel time with 16 x the arithmetic per byte; the hybrid step through the "
                                        "host link is timed at x16 in other_configs.config4 (PAPER.md:109)"}
    # ---- accumulate mode (source terms are additive): the same step with
    # every output a read-modify-write
    if headline and not swap and not is_tuned(args):
        ctx.barrier()
        time.sleep(1.0)
        L.set_accumulate(True)
        a0, a1 = timed_loop(ctx, st, whole_step, 10, warm=2)
        ctx.barrier()
        L.set_accumulate(False)
        ams = ctx.max_over_ranks(a0.elapsed_time(a1)) / 10
        out_b = (3 + nq) * es * cfg.points
        rec["accumulate"] = {"steps": 10, "ms_per_step": ams, "ratio_to_overwrite": ams / ms_per_step,
                             "value": ctx.world * cfg.points / (ams * 1e-3) / 1e9,
                             "bytes_moved_per_step": alg + out_b, "moved_GBs": (alg + out_b) / (ams * 1e-3) / 1e9,
                             "launch_plan": L.describe_plan()}
    if not headline:
        if cfg.dtype == "f32" and nq:
            # the precision variant end to end (half the bytes on the host link)
            del sets
            gc.collect()
            torch.cuda.empty_cache()
            hin = [torch.empty(L.shape, dtype=tdt, pin_memory=True) for _ in names]
            for t_, a in zip(hin, H):
                t_.copy_(torch.from_numpy(a))
            hout = [torch.zeros(L.shape, dtype=tdt, pin_memory=True) for _ in names]
            L.set_chunks(args.chunks)
            t_e2e = []
            for _ in range(3):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
                L.step_wait()
                t_e2e.append(time.perf_counter() - t0)
            e_s = float(np.mean(t_e2e[1:]))
            ph = L.step_times_ms()
            plane_b = (cfg.ny + 2 * cfg.halo) * cfg.nz * es
            rec["e2e"] = {"value": cfg.points / e_s / 1e9, "unit": "Gpts/s", "ms_per_step": e_s * 1e3, "steps": 2,
                          "chunks": L.step_chunk_count(), "h2d_bytes_per_step": nf * (cfg.nx + 2) * plane_b,
                          "d2h_bytes_per_step": nf * cfg.points * es,
                          "h2d_GBs": nf * (cfg.nx + 2) * plane_b / (ph["h2d"] * 1e-3) / 1e9,
                          "d2h_GBs": nf * cfg.points * es / (ph["d2h"] * 1e-3) / 1e9}
            del hin, hout
        else:
            del sets
        L.close()
        gc.collect()
        torch.cuda.empty_cache()
        return rec

    # ---- the two north_star calls, kernel by kernel (an event between the two launches)
    if nq and not swap:
        tsteps = min(steps, 20)
        ctx.barrier()
        time.sleep(1.0)
        marks = []
        with torch.cuda.stream(st):
            for i in range(3):
                ins, outs = sets[i % nsets]
                L.momentum(ins[0], ins[1], ins[2], outs[0], outs[1], outs[2], stream=st)
                L.scalars(ins[3:], outs[3:], stream=st)
            e = torch.cuda.Event(enable_timing=True); e.record(st); marks.append(("start", e))
            for i in range(tsteps):
                ins, outs = sets[(3 + i) % nsets]
                L.momentum(ins[0], ins[1], ins[2], outs[0], outs[1], outs[2], stream=st)
                e = torch.cuda.Event(enable_timing=True); e.record(st); marks.append(("mom", e))
                L.scalars(ins[3:], outs[3:], stream=st)
                e = torch.cuda.Event(enable_timing=True); e.record(st); marks.append(("sca", e))
        ctx.barrier()
        span = {"mom": 0.0, "sca": 0.0}
        for (_, a), (k, b) in zip(marks[:-1], marks[1:]):
            span[k] += a.elapsed_time(b)
        mom_ms, sca_ms = span["mom"] / tsteps, span["sca"] / tsteps
        mb, sb = bytes_momentum(cfg.dtype) * cfg.points, bytes_scalars(nq, cfg.dtype) * cfg.points
        rec["two_call_step"] = {
            "call": "monc_adv_momentum + monc_adv_scalars", "steps": tsteps, "ms_per_step": mom_ms + sca_ms,
            "value": ctx.world * cfg.points / ((mom_ms + sca_ms) * 1e-3) / 1e9, "launch_plan": L.describe_plan(),
            "momentum_ms": mom_ms, "momentum_GBs": mb / (mom_ms * 1e-3) / 1e9,
            "scalars_ms": sca_ms, "scalars_GBs": sb / (sca_ms * 1e-3) / 1e9,
            "algorithmic_bytes_per_step": mb + sb}

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

    e2e_steps = max(1, min(steps, args.e2e_steps))
    for _ in range(2):
        e2e_step()
    ctx.barrier()
    enqueue_s[0] = 0.0
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = ctx.max_over_ranks(time.perf_counter() - t0)
    enqueue_ms = enqueue_s[0] / e2e_steps * 1e3
    phase = L.step_times_ms()
    # the same step with copies and kernels serialised on one stream: its phases are
    # the "alone" times of the overlap ratio
    L.set_overlap(False)
    e2e_step()
    torch.cuda.synchronize()
    serial = L.step_times_ms()
    L.set_overlap(True)
    plane_b = (cfg.ny + 2 * cfg.halo) * cfg.nz * es
    h2d_b = nf * (cfg.nx + 2) * plane_b
    d2h_b = nf * cfg.points * es
    rec["e2e"] = {"value": ctx.world * cfg.points * e2e_steps / e2e_s / 1e9, "unit": "Gpts/s",
                  "h2d_bytes_per_step": h2d_b, "d2h_bytes_per_step": d2h_b, "steps": e2e_steps,
                  "ms_per_step": e2e_s / e2e_steps * 1e3, "host_enqueue_ms_per_step": enqueue_ms,
                  "h2d_GBs": h2d_b / (phase["h2d"] * 1e-3) / 1e9, "d2h_GBs": d2h_b / (phase["d2h"] * 1e-3) / 1e9,
                  # the host link alone, one direction at a time (the serialised pass): the
                  # denominator of the copy/compute overlap (BASELINE.json north_star)
                  "link_alone_GBs": {"h2d": h2d_b / (serial["h2d"] * 1e-3) / 1e9,
                                     "d2h": d2h_b / (serial["d2h"] * 1e-3) / 1e9},
                  "phase_ms": phase, "chunks": L.step_chunk_count(),
                  "chunks_chosen_by": "caller (--chunks)" if args.chunks else "library (automatic)",
                  "serial_phase_ms": serial,
                  "overlap_ratio": (serial["h2d"] + serial["kernels"] + serial["d2h"]) / phase["total"],
                  "timing": "host wall clock around step_async + step_wait, pinned host buffers"}
    L.close()
    del sets, hin, hout
    gc.collect()
    torch.cuda.empty_cache()
    return rec


# ---------------------------------------------------------------------------
# config4: the paper's hybrid asynchronous step as the step
# ---------------------------------------------------------------------------
def run_hybrid_config(ctx, args, steps, warmup, with_cpu):
    """1024x1024x160 fp64, 3 momentum + 4 scalars in PINNED HOST memory; a step is
    monc_adv_step_async (8 x-slab chunks H2D -> kernels -> D2H on three streams)
    + monc_adv_step_wait.  Fields are perturbed on the host between steps
    (BASELINE.json configs[4]), outside the timed region: the time of a step is
    the library's device-event span first copy -> last copy, summed over steps."""
    torch = ctx.torch
    from paper_2009_12850_b200 import synth
    cfg = workload_cfg("config4")
    L = make_library(cfg, args)
    nchunks = args.chunks or 8  # BASELINE.json configs[4]: 8 chunks; the library's own choice is timed beside it
    L.set_chunks(nchunks)
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

    for _ in range(max(1, min(warmup, 3))):
        step()
    sampler = ClockSampler(0, period_s=0.05).start()
    n0 = L.launch_count()
    phases = []
    for s_ in range(steps):
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
    value = cfg.points * steps / (tot_ms * 1e-3) / 1e9
    med = {k: float(np.median([p_[k] for p_ in phases])) for k in phases[0]}
    kb = bytes_fused(cfg.nq, "f64") * cfg.points
    peak, peak_src = peaks()
    ach = kb / (serial["kernels"] * 1e-3) / 1e9

    # ---- streaming combine: the host integrates a chunk's source terms as
    # soon as that chunk has landed, while the later chunks are still on the wire, instead of
    # waiting for the whole copy.  Integrate = axpy into the host's own copy of su (one field
    # stands for the model's `step fields`).
    h = cfg.halo
    own = np.zeros(L.shape)
    C = nchunks

    def integrate(a, b):
        own[h + a:h + b, h:h + cfg.ny] += 0.5 * hout[0].numpy()[h + a:h + b, h:h + cfg.ny]

    t0 = time.perf_counter()
    L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
    L.step_wait()
    t_wait = time.perf_counter() - t0
    integrate(0, cfg.nx)
    t_after = time.perf_counter() - t0
    t0 = time.perf_counter()
    L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
    for c in range(C):
        L.step_wait_chunk(c)
        integrate(*L.step_chunk_range(c))
    L.step_wait()
    t_stream = time.perf_counter() - t0
    # and the on-device combine: the host's source terms go up with the fields,
    # the kernels add, no separate result buffer -- at the price of the extra H2D
    L.set_accumulate(True)
    t0 = time.perf_counter()
    L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
    L.step_wait()
    t_devacc = time.perf_counter() - t0
    L.set_accumulate(False)
    # the paper's x16 work-scaled run: "the GPU times look very similar"
    L.set_work_scale(16)
    t0 = time.perf_counter()
    L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
    L.step_wait()
    t_x16 = time.perf_counter() - t0
    x16 = L.step_times_ms()
    L.set_work_scale(1)
    # the same step with the chunk count the library picks itself (monc_adv_set_chunks(h, 0))
    L.set_chunks(0)
    step()
    auto = [step() for _ in range(2)]
    auto_rec = {"chunks": L.step_chunk_count(), "ms_per_step": float(np.mean([a["total"] for a in auto])),
                "value": cfg.points / (float(np.mean([a["total"] for a in auto])) * 1e-3) / 1e9}
    L.set_chunks(nchunks)
    combine = {"wait_all_then_integrate_ms": t_after * 1e3, "of_which_integrate_ms": (t_after - t_wait) * 1e3,
               "integrate_as_chunks_land_ms": t_stream * 1e3,
               "combine_overlap": (t_after - t_stream) / max(t_after - t_wait, 1e-9),
               "device_accumulate_step_ms": t_devacc * 1e3,
               "note": "combine_overlap = share of the host's integrate time hidden under the copies still in "
                       "flight (1 = all of it); device_accumulate uploads the 7 source-term arrays as well"}

    rec = {"value": value, "unit": "Gpts/s", "ms_per_step": tot_ms / steps, "steps": steps, "warmup": warmup,
           "dtype": "f64", "gpu_launches": launches, "launch_plan": plan, "clocks": clocks,
           "config": config_record(
               cfg, "config4", chunks=nchunks, perturbed_each_step=not args.no_perturb,
               l2=f"inputs stream from pinned host memory ({h2d_b / 1e9:.2f} GB per step) > 126 MB L2",
               parallelism="1 GPU", step_call="monc_adv_step_async + monc_adv_step_wait",
               timing="device events inside the library, first H2D -> last D2H, summed over steps",
               launch_plan=plan),
           "roofline": {"bound": "hbm", "kernel": "tma_scalars<double, MOM=1> (fused) per x-slab chunk",
                        "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "traffic": None,
                        "peak_source": peak_src, "algorithmic_bytes_per_launch": kb / nchunks,
                        "avg_launch_ms": serial["kernels"] / nchunks, "frac_of_nominal_8TBs": ach / NOMINAL_GBS,
                        "note": "kernel time = sum over the chunks of the serialised pass (copies not "
                                "overlapping); the step itself is host-link bound"},
           "e2e": {"value": value, "unit": "Gpts/s", "h2d_bytes_per_step": h2d_b, "d2h_bytes_per_step": d2h_b,
                   "steps": steps, "ms_per_step": tot_ms / steps, "chunks": nchunks, "automatic_chunks": auto_rec,
                   "h2d_GBs": h2d_b / (med["h2d"] * 1e-3) / 1e9, "d2h_GBs": d2h_b / (med["d2h"] * 1e-3) / 1e9,
                   "link_alone_GBs": {"h2d": h2d_b / (serial["h2d"] * 1e-3) / 1e9,
                                      "d2h": d2h_b / (serial["d2h"] * 1e-3) / 1e9},
                   "phase_ms_median": med, "serial_phase_ms": serial,
                   "overlap_ratio": (serial["h2d"] + serial["kernels"] + serial["d2h"]) / med["total"],
                   "streaming_combine": combine,
                   "work_scale_16": {"step_ms": x16["total"], "kernels_ms": x16["kernels"], "wall_ms": t_x16 * 1e3,
                                     "step_ratio_to_x1": x16["total"] / med["total"],
                                     "kernels_ratio_to_x1": x16["kernels"] / med["kernels"]}}}
    if with_cpu:
        rec["cpu_baseline"] = cpu_baseline(cfg, args, "config4")
    L.close()
    del hin, hout
    gc.collect()
    torch.cuda.empty_cache()
    return rec


def run_paper_shape(ctx, args):
    """Context: the paper's own per-process sub-domain, 64x64x64 = 262144 points
    (PAPER.md:105-111), 3 momentum + theta + 5 q, through the hybrid step; alone, and 8 such
    sub-domains sharing the GPU as the paper's 8 MPI ranks shared a K20X: 8 handles,
    every step enqueued before any is waited for.  Timing only (seeded host fields)."""
    torch = ctx.torch
    from paper_2009_12850_b200 import binding, synth
    cfg = synth.Config(90, 64, 64, 64, halo=2, nq=6, dtype="f64")
    g = synth.grid(cfg.nz)
    names = ["u", "v", "w"] + synth.field_names(cfg)
    H = [synth.field(cfg, n) for n in names]
    ranks = []
    for _ in range(8):
        L = binding.MoncAdv(cfg.nx, cfg.ny, cfg.nz, cfg.halo, synth.DX, synth.DY, g["dz"], g["dzn"], g["rho"], g["rhon"],
                            dtype="f64")
        hin = [torch.from_numpy(a).pin_memory() for a in H]
        hout = [torch.zeros(L.shape, dtype=torch.float64).pin_memory() for _ in names]
        ranks.append((L, hin, hout))

    def enqueue(r):
        L, hin, hout = r
        L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])

    def timed(rs, n):
        for _ in range(3):
            for r in rs:
                enqueue(r)
            for r in rs:
                r[0].step_wait()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(n):
            for r in rs:
                enqueue(r)
            for r in rs:
                r[0].step_wait()
        return (time.perf_counter() - t0) / n

    t1 = timed(ranks[:1], 50)
    t8 = timed(ranks, 20)
    pts = cfg.nx * cfg.ny * cfg.nz
    out = {"config": {"workload": "paper sub-domain 64x64x64, 3 + 6 fields, hybrid step", "nx": 64, "ny": 64, "nz": 64,
                      "nq": 6, "storage_dtype": "f64", "step_call": "monc_adv_step_async + monc_adv_step_wait"},
           "one_subdomain": {"ms_per_step": t1 * 1e3, "value": pts / t1 / 1e9, "chunks": ranks[0][0].step_chunk_count()},
           "eight_subdomains_sharing_the_gpu": {"ms_per_round": t8 * 1e3, "value": 8 * pts / t8 / 1e9,
                                                "speedup_over_one_after_another": 8 * t1 / t8},
           "unit": "Gpts/s", "launch_plan": ranks[0][0].describe_plan()}
    for L, _, _ in ranks:
        L.close()
    del ranks
    gc.collect()
    # the paper's strong-scaling domain (z = 64, x = y = 2048, 268 M points; 1024 K20X nodes at
    # the far end of Fig. 4) resident in ONE B200's HBM: the same 3 + 6 fields, one fused launch per step
    nx = ny = 2048
    L = binding.MoncAdv(nx, ny, 64, 2, synth.DX, synth.DY, g["dz"], g["dzn"], g["rho"], g["rhon"], dtype="f64")
    gen = torch.Generator(device="cuda").manual_seed(20091285)
    ins = [torch.randn(L.shape, device="cuda", dtype=torch.float64, generator=gen) for _ in range(9)]
    outs = [torch.empty(L.shape, device="cuda", dtype=torch.float64) for _ in range(9)]
    st = torch.cuda.Stream()

    def whole(i):
        L.tendencies(ins[0], ins[1], ins[2], outs[0], outs[1], outs[2], ins[3:], outs[3:], stream=st)

    e0, e1 = timed_loop(ctx, st, whole, 5, warm=2)
    ctx.barrier()
    ms = e0.elapsed_time(e1) / 5
    alg = bytes_fused(6, "f64") * nx * ny * 64
    peak, _ = peaks()
    out["global_domain_2048x2048x64_resident"] = {
        "ms_per_step": ms, "value": nx * ny * 64 / (ms * 1e-3) / 1e9, "algorithmic_GBs": alg / (ms * 1e-3) / 1e9,
        "frac": alg / (ms * 1e-3) / 1e9 / peak, "hbm_resident_GB": 18 * L.shape[0] * L.shape[1] * L.shape[2] * 8 / 1e9,
        "launch_plan": L.describe_plan(), "steps": 5, "data": "device randn (timing only)"}
    L.close()
    del ins, outs
    gc.collect()
    torch.cuda.empty_cache()
    return out


def run_ragged_nz(ctx, args):
    """Config 2 with one level less (512x512x255 fp64, 3 + 10 fields): nz is not a whole number of
    16-byte vectors, the shape round 1 sent to the one-thread-per-point kernels.  Timing only (device
    random inputs; parity of this path: tests/test_gpu_parity.py::test_ragged_nz_on_the_tma_kernels)."""
    torch = ctx.torch
    from paper_2009_12850_b200 import binding, synth
    nx, ny, nz, nq = 512, 512, 255, 10
    g = synth.grid(nz)
    out = {"config": {"workload": "config2 with nz = 255 (ragged)", "nx": nx, "ny": ny, "nz": nz, "nq": nq,
                      "storage_dtype": "f64", "step_call": "monc_adv_tendencies", "data": "device randn (timing only)"}}
    L = binding.MoncAdv(nx, ny, nz, 2, synth.DX, synth.DY, g["dz"], g["dzn"], g["rho"], g["rhon"], dtype="f64")
    gen = torch.Generator(device="cuda").manual_seed(20091285)
    sets = [([torch.randn(L.shape, device="cuda", dtype=torch.float64, generator=gen) for _ in range(3 + nq)],
             [torch.empty(L.shape, device="cuda", dtype=torch.float64) for _ in range(3 + nq)]) for _ in range(2)]
    st = torch.cuda.Stream()
    alg = bytes_fused(nq, "f64") * nx * ny * nz
    peak, _ = peaks()

    def step(i):
        a, o = sets[i % 2]
        L.tendencies(a[0], a[1], a[2], o[0], o[1], o[2], a[3:], o[3:], stream=st)

    for variant in ("auto", "generic"):
        L.set_variant(variant)
        e0, e1 = timed_loop(ctx, st, step, 20, warm=3)
        ctx.barrier()
        ms = e0.elapsed_time(e1) / 20
        out["tma_ragged" if variant == "auto" else "generic_kernels"] = {
            "ms_per_step": ms, "value": nx * ny * nz / (ms * 1e-3) / 1e9, "algorithmic_GBs": alg / (ms * 1e-3) / 1e9,
            "frac": alg / (ms * 1e-3) / 1e9 / peak, "launch_plan": L.describe_plan(), "steps": 20}
    L.close()
    del sets
    gc.collect()
    torch.cuda.empty_cache()
    return out


def compact(rec):
    """What a sub-record of `other_configs` keeps."""
    keep = ("value", "unit", "ms_per_step", "steps", "dtype", "gpu_launches", "launch_plan", "clocks",
            "sustained", "burst")
    out = {k: rec[k] for k in keep if k in rec}
    r = rec["roofline"]
    out["roofline"] = {k: r[k] for k in ("kernel", "achieved", "peak", "frac", "frac_of_nominal_8TBs",
                                         "algorithmic_bytes_per_launch", "avg_launch_ms") if k in r}
    out["config"] = {k: rec["config"][k] for k in ("workload", "nx", "ny", "nz", "nq", "storage_dtype", "step_call")}
    if "e2e" in rec:
        e = rec["e2e"]
        out["e2e"] = {k: e[k] for k in ("value", "ms_per_step", "chunks", "automatic_chunks", "h2d_bytes_per_step",
                                        "d2h_bytes_per_step", "h2d_GBs", "d2h_GBs",
                                        "link_alone_GBs", "overlap_ratio", "streaming_combine", "work_scale_16") if k in e}
    return out


def run_ours(args):
    ctx = Ctx()
    cache = {}
    if args.workload == "config4":
        if ctx.world > 1:
            raise SystemExit("config4 is a single-GPU workload (one host link)")
        rec = run_hybrid_config(ctx, args, args.steps, args.warmup, with_cpu=True)
        cfg = workload_cfg("config4")
    else:
        cfg = workload_cfg(args.workload)
        rec = run_device_config(ctx, args, args.workload, cache, headline=True)
        if ctx.rank == 0:
            rec["cpu_baseline"] = cpu_baseline(cfg, args, args.workload)
    others = {}
    if not args.no_others and ctx.world == 1 and not args.halo_exchange and not is_tuned(args):
        for w in ("config3", "config2", "config1", "config4"):  # config 3 first: it reuses config 2's fields
            if w == args.workload:
                continue
            try:
                if w == "config4":
                    cache.clear()
                    others[w] = compact(run_hybrid_config(ctx, args, steps=3, warmup=1, with_cpu=False))
                else:
                    others[w] = compact(run_device_config(ctx, args, w, cache, headline=False))
            except Exception as e:  # a sub-record must not take the headline down with it
                others[w] = {"error": f"{type(e).__name__}: {e}"}
            if w == "config1":
                for key, fn in (("ragged_nz", run_ragged_nz), ("paper_subdomain", run_paper_shape)):
                    try:
                        others[key] = fn(ctx, args)
                    except Exception as e:
                        others[key] = {"error": f"{type(e).__name__}: {e}"}
    if ctx.rank != 0:
        ctx.close()
        return
    out = {"metric": "advection grid-points/sec", "value": rec["value"], "unit": "Gpts/s", "n_gpus": ctx.world,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": rec["ms_per_step"],
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype,
           "data": "synthetic", "config": rec["config"], "roofline": rec["roofline"],
           "cpu_baseline": rec.get("cpu_baseline"), "e2e": rec["e2e"], "gpu_launches": rec["gpu_launches"],
           "clocks": rec["clocks"]}
    c = rec.get("copy_same_bytes")
    if c and "burst_GBs" in c:
        if "burst" in rec:
            c["kernel_over_copy_burst"] = rec["burst"]["algorithmic_GBs"] / c["burst_GBs"]
        if "sustained" in rec:
            c["kernel_over_copy_sustained"] = rec["sustained"]["algorithmic_GBs"] / c["sustained_GBs"]
    for k in ("field_points_per_s_G", "sustained", "burst", "two_call_step", "work_scale_16", "accumulate",
              "copy_same_bytes"):
        if k in rec:
            out[k] = rec[k]
    if others:
        out["other_configs"] = others
    print(json.dumps(out))
    ctx.close()


def cpu_baseline(cfg, args, workload):
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
                      f" x-planes of {workload}, {len(names)} fields, {dt:.1f} s",
            "all_cores": {"value": sub.points * reps_all / dt_all / 1e9, "unit": "Gpts/s", "cores": nthr,
                          "sample": f"{reps_all} passes of the same sample, {dt_all:.1f} s"},
            "host_cores_available": len(os.sched_getaffinity(0))}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2", choices=["config1", "config2", "config3", "config4"])
    ap.add_argument("--no-others", action="store_true",
                    help="skip the compact records of the other BASELINE configs")
    ap.add_argument("--no-work-scale", action="store_true",
                    help="skip the x16 work-scaled leg (PAPER.md:109) of the headline record")
    ap.add_argument("--sustain-seconds", type=float, default=2.5,
                    help="length of the sustained loop of the headline step (0 = skip)")
    ap.add_argument("--xchunk", type=int, default=0)
    ap.add_argument("--group", type=int, default=0)
    ap.add_argument("--stages", type=int, default=0)
    ap.add_argument("--tile-y", type=int, default=0)
    ap.add_argument("--warps", type=int, default=0)
    ap.add_argument("--split", type=int, default=0)
    ap.add_argument("--variant", default="", choices=["", "auto", "generic", "march", "tma"])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-pdl", action="store_true", help="plain stream order between kernels")
    ap.add_argument("--form", default="flux", choices=["flux", "pw_skew"],
                    help="flux form (default, BASELINE.json) or the Piacsek-Williams skew form (DESIGN.md R4)")
    ap.add_argument("--ref-planes", type=int, default=64)
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--halo-exchange", action="store_true",
                    help="N ranks advect x-slabs of ONE periodic domain of N*nx planes and swap halos over NCCL every step"
                         " (default: independent replicas, no data-path collective)")
    ap.add_argument("--chunks", type=int, default=0,
                    help="x-slab chunks per hybrid step; 0 = the library chooses (config 4 runs BASELINE.json's 8 "
                         "and reports the automatic count beside it)")
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
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
