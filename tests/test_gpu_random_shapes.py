"""Seeded random shapes through the public calls against the oracle: every combination the launch paths branch on
(aligned / ragged nz with and without a column-group view, tall columns, 0..13 scalars, halo 1..3, both dtypes and
forms, overwrite / accumulate, fused / two calls, the hybrid step) in sizes the oracle finishes at once."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2009_12850_b200 import binding, synth
import gpu_common as gc

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def _need_gpu(gpu_required):
    yield
    torch.cuda.synchronize()


def draw(rng):
    nz = int(rng.choice([3, 4, 5, 6, 7, 8, 16, 31, 32, 33, 63, 64, 65, 66, 70, 96, 127, 128, 129, 130, 160, 255, 257, 1030]))
    big = nz > 200
    nx = int(rng.integers(1, 6 if big else 24))
    ny = int(rng.integers(1, 8 if big else 28))
    halo = int(rng.integers(1, 4))
    nq = int(rng.choice([0, 1, 2, 3, 4, 5, 7, 10, 11, 13]))
    if big:
        nq = min(nq, 4)
    return dict(nx=nx, ny=ny, nz=nz, halo=halo, nq=nq, dtype=str(rng.choice(["f64", "f32"])),
                form=str(rng.choice(["flux", "pw_skew"])), accumulate=bool(rng.integers(0, 2)),
                call=str(rng.choice(["tendencies", "two_calls", "step_async"])),
                xchunk=int(rng.choice([0, 0, 2, 5])), chunks=int(rng.choice([0, 1, 3])))


CASES = [draw(np.random.default_rng(1000 + n)) for n in range(200)]


@pytest.mark.parametrize("case", CASES, ids=lambda c: "{nx}x{ny}x{nz}h{halo}q{nq}{dtype}-{form}-{call}{a}".format(
    a="-acc" if c["accumulate"] else "", **c))
def test_random_shape(case):
    c = case
    cfg = gc.custom_cfg(c["nx"], c["ny"], c["nz"], halo=c["halo"], nq=c["nq"], dtype=c["dtype"], cid=800)
    P, L = gc.make_pair(cfg)
    L.set_form(c["form"])
    L.set_tuning(xchunk=min(c["xchunk"], c["nx"]))
    skew = c["form"] == "pw_skew"
    names = ["u", "v", "w"] + synth.field_names(cfg)
    H = [synth.field(cfg, n) for n in names]
    want = list(P.momentum(H[0], H[1], H[2], skew=skew)) + [P.scalar(H[0], H[1], H[2], q, skew=skew) for q in H[3:]]
    h, nf = cfg.halo, len(names)
    reps = 2 if c["accumulate"] else 1
    L.set_accumulate(c["accumulate"])
    if c["call"] == "step_async":
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(L.torch_dtype).pin_memory()
        hin = [pin(a) for a in H]
        hout = [torch.full(L.shape, gc.SENTINEL, dtype=L.torch_dtype).pin_memory() for _ in names]
        if c["accumulate"]:
            for o in hout:
                o[h:h + cfg.nx, h:h + cfg.ny] = 0.0
        L.set_chunks(min(c["chunks"], cfg.nx))
        for _ in range(reps):
            L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
            L.step_wait()
        outs = hout
    else:
        D = [gc.to_dev(a, L) for a in H]
        outs = gc.fresh_out(L, nf)
        if c["accumulate"]:
            for o in outs:
                o[h:h + cfg.nx, h:h + cfg.ny] = 0.0
        for _ in range(reps):
            if c["call"] == "tendencies":
                L.tendencies(D[0], D[1], D[2], outs[0], outs[1], outs[2], D[3:], outs[3:])
            else:
                L.momentum(D[0], D[1], D[2], outs[0], outs[1], outs[2])
                L.scalars(D[3:], outs[3:])
        torch.cuda.synchronize()
    plan = L.describe_plan()
    for o, w_, n in zip(outs, want, ["su", "sv", "sw"] + names[3:]):
        gc.check(cfg, o, reps * w_, f"{n} [{plan}]")
        gc.check_halo_untouched(cfg, o, n)
    L.close()
