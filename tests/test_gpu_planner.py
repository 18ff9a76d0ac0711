"""The launch planners (csrc/monc_adv.cu: plan_tma, plan_tma_scalars) encode measurements of
one machine.  This test keeps them honest: at BASELINE.json's configs 1-3 the
geometry the library picks on its own must be within 5 % of the best of a small sweep of the
internal tuning knobs (include/monc_adv_tuning.h), timed here with CUDA events.  Timing only:
the fields are random, results are not compared (the parity tests do that)."""
import numpy as np
import pytest
import torch

from paper_2009_12850_b200 import binding, synth

pytestmark = pytest.mark.gpu

TOL = 1.05


@pytest.fixture(autouse=True)
def _need_gpu(gpu_required):
    yield
    torch.cuda.synchronize()


def _bench(cfg, knobs_list, call, steps, reps=4):
    g = synth.grid(cfg.nz)
    tdt = torch.float64 if cfg.dtype == "f64" else torch.float32
    nf = 3 + cfg.nq
    nsets = 2 if cfg.nq else 4   # more than L2 in flight between two uses of a buffer
    sets = [([torch.rand(cfg.shape, device="cuda", dtype=tdt) - 0.5 for _ in range(nf)],
             [torch.empty(cfg.shape, device="cuda", dtype=tdt) for _ in range(nf)]) for _ in range(nsets)]
    Ls = []
    for kn in knobs_list:
        L = binding.MoncAdv(cfg.nx, cfg.ny, cfg.nz, cfg.halo, synth.DX, synth.DY, g["dz"], g["dzn"], g["rho"],
                            g["rhon"], dtype=cfg.dtype)
        L.set_tuning(**kn)
        Ls.append(L)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    best = [1e30] * len(Ls)
    plans = [""] * len(Ls)
    for r in range(reps):
        for n, L in enumerate(Ls):   # interleaved: every candidate sees the same board state
            for i in range(2):
                call(L, *sets[i % nsets])
            e0.record()
            for i in range(steps):
                call(L, *sets[i % nsets])
            e1.record()
            torch.cuda.synchronize()
            best[n] = min(best[n], e0.elapsed_time(e1) / steps)
            plans[n] = L.describe_plan()
    for L in Ls:
        L.close()
    return best, plans


def _fused(L, f, o):
    L.tendencies(f[0], f[1], f[2], o[0], o[1], o[2], f[3:], o[3:])


def _momentum(L, f, o):
    L.momentum(f[0], f[1], f[2], o[0], o[1], o[2])


def _two_calls(L, f, o):
    L.momentum(f[0], f[1], f[2], o[0], o[1], o[2])
    L.scalars(f[3:], o[3:])


def _check(name, best, plans, knobs):
    auto, rest = best[0], best[1:]
    table = ", ".join(f"{k or 'auto'}: {t * 1e3:.1f} us" for k, t in zip(knobs, best))
    print(f"{name}: {table} | auto plan: {plans[0]}")
    assert auto <= TOL * min(rest), f"{name}: auto plan {auto * 1e3:.1f} us, best of the sweep " \
                                    f"{min(rest) * 1e3:.1f} us ({plans[int(np.argmin(rest)) + 1]})"


def test_config1_momentum_plan():
    knobs = [dict(), dict(tile_y=8, xchunk=64), dict(tile_y=8, xchunk=32), dict(tile_y=8, xchunk=128),
             dict(tile_y=7, xchunk=64), dict(tile_y=4, xchunk=64), dict(tile_y=8, xchunk=64, stages=5)]
    best, plans = _bench(synth.CONFIGS[1], knobs, _momentum, steps=40)
    _check("config1 momentum", best, plans, knobs)


@pytest.mark.parametrize("cid", [2, 3])
def test_config2_and_3_fused_plan(cid):
    knobs = [dict(), dict(xchunk=32), dict(xchunk=43), dict(xchunk=64), dict(xchunk=103), dict(xchunk=171),
             dict(xchunk=64, tile_y=4), dict(xchunk=64, stages=3)]
    best, plans = _bench(synth.CONFIGS[cid], knobs, _fused, steps=8)
    assert "tma_fused" in plans[0]
    _check(f"config{cid} fused", best, plans, knobs)


def test_config2_two_call_plans():
    knobs = [dict(), dict(xchunk=32), dict(xchunk=64), dict(xchunk=128), dict(xchunk=64, split=3),
             dict(xchunk=64, group=5), dict(xchunk=64, tile_y=7), dict(xchunk=64, tile_y=5)]
    best, plans = _bench(synth.CONFIGS[2], knobs, _two_calls, steps=6)
    _check("config2 momentum + scalars", best, plans, knobs)
