"""The checked build of the library (libmonc_adv_checked.so, -DMONC_ADV_CHECKED=1) through
the same parity tests.  compute-sanitizer is closed on the pool this repo is built on
(profiles/r02_sanitizer.md), so the TMA ring protocol is checked from the inside:
every ring slot is filled with NaN before each refill and at kernel start, and every
warp sleeps a pseudo-random time before it reads a slot, before it releases one and
before a refill.  A read of a location the copy did not write (initcheck), or of a
slot released too early and already poisoned / overwritten for a later plane
(racecheck), reaches an output as NaN or as a wrong value and fails the comparison
with the oracle; the jitter exercises orderings the undisturbed schedule never shows.
Each case runs several times: the delays differ from launch to launch."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2009_12850_b200 import binding, synth
import gpu_common as gc
import test_gpu_parity as tp

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def _checked_build(gpu_required):
    from paper_2009_12850_b200 import build as libbuild
    libbuild.build(checked=True)
    binding.select_build(True)
    assert "checked build" in binding.version()
    yield
    torch.cuda.synchronize()
    binding.select_build(False)
    assert "checked build" not in binding.version()


REPS = 3


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_checked_momentum_ring(dtype):
    # several y tiles, z chunks and x chunks; deep and shallow rings; ragged tails
    for shape, kw in (((13, 7, 40, 2), dict()), ((10, 6, 72, 2), dict(xchunk=4)),
                      ((6, 10, 160, 2), dict(xchunk=3, stages=3, tile_y=2)), ((33, 17, 136, 2), dict(xchunk=9)),
                      ((5, 9, 256, 1), dict(stages=4))):
        nx, ny, nz, h = shape
        cfg = gc.custom_cfg(nx, ny, nz, halo=h, dtype=dtype, cid=600 + nz)
        for _ in range(REPS):
            tp.run_momentum(cfg, "tma", **kw)
            tp.run_momentum(cfg, "tma", form="pw_skew", **kw)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_checked_scalar_ring(dtype):
    cfg = gc.custom_cfg(12, 10, 72, dtype=dtype, cid=610)
    for _ in range(REPS):
        tp.run_scalars(cfg, 3, "tma", xchunk=0, group=3)
        tp.run_scalars(cfg, 3, "tma", xchunk=3, group=2, stages=2, tile_y=2, split=1)   # two-stage ring
        tp.run_scalars(cfg, 7, "tma", xchunk=2, group=7, stages=3, tile_y=2, split=3)   # ragged splits
        tp.run_scalars(cfg, 10, "tma", xchunk=5, group=10, split=2, form="pw_skew")
        tp.run_scalars(cfg, 11, "tma", xchunk=4, group=5, split=1)                       # three groups


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("form", ["flux", "pw_skew"])
def test_checked_fused_ring(dtype, form):
    # the fused launch: the momentum role releases a slot one step after the scalar warps
    cfg = gc.custom_cfg(21, 19, 200, dtype=dtype, cid=620)
    for _ in range(REPS):
        for nq, tuning in ((1, None), (4, dict(xchunk=5, tile_y=2, stages=3)), (10, dict(xchunk=6)),
                           (7, dict(xchunk=8))):
            assert "tma_fused" in tp.run_tendencies(cfg, nq, form=form, tuning=tuning)
    tp.run_tendencies(gc.custom_cfg(9, 5, 64, dtype=dtype, cid=621), 5, form=form, accumulate=True)


def test_checked_ragged_nz():
    # per-row copies of the column-group view (ragged nz): same ring, same protocol
    for shape in (tp.RAGGED_NZ[1], tp.RAGGED_NZ[5]):
        for _ in range(2):
            tp.test_ragged_nz_on_the_tma_kernels(shape)


def test_checked_random_shapes():
    # the first 60 of the seeded random cases (every launch path) on poisoned, jittered rings
    import test_gpu_random_shapes as tr
    for case in tr.CASES[:60]:
        tr.test_random_shape(case)


def test_checked_hybrid_step():
    import test_gpu_async as ta
    for _ in range(REPS):
        ta.test_step_async_small(8, True, "f64")
        ta.test_step_async_small(3, True, "f32")
        ta.test_step_async_accumulate_is_bitwise_wait_then_add("f64")


def test_checked_build_is_bitwise_the_normal_build():
    cfg = gc.custom_cfg(17, 13, 136, nq=4, cid=630)
    names = ["u", "v", "w"] + synth.field_names(cfg)
    H = [synth.field(cfg, n) for n in names]
    res = []
    for checked in (True, False):
        binding.select_build(checked)
        P, L = gc.make_pair(cfg)
        d = [gc.to_dev(a, L) for a in H]
        o = gc.fresh_out(L, len(names))
        L.tendencies(d[0], d[1], d[2], o[0], o[1], o[2], d[3:], o[3:])
        torch.cuda.synchronize()
        res.append([t.clone() for t in o])
        L.close()
    binding.select_build(True)
    for a, b in zip(*res):
        assert torch.equal(a, b)
