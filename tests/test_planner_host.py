"""The launch planners of libmonc_adv.so as host arithmetic (monc_adv_plan_describe: no handle, no GPU).

The planners' cost models hold constants measured on B200.  tests/test_gpu_planner.py checks on
the GPU that the plan picked is within 5 % of the best of a sweep; this file pins, on the CPU, the geometries
those measurements selected for BASELINE.json's configs, so that a change to the model that moves them is seen
without a GPU, and checks the invariants every plan must satisfy."""
import re

import pytest

from paper_2009_12850_b200 import binding

B200 = dict(sm_count=148, smem_optin=232448)


def parse(part):
    d = dict(re.findall(r"(\w+)=([0-9x]+)", part))
    gx, gy = d.pop("grid").split("x")
    out = {k: int(v) for k, v in d.items()}
    out["gx"], out["gy"] = int(gx), int(gy)
    return out


@pytest.fixture(scope="module")
def lib():
    return binding.load()


def test_plans_of_the_baseline_configs(lib):
    # config 1: one wave of 128 blocks (a GPC sustains 16 SMs' worth of this kernel), clusters of 4
    p = parse(binding.plan_describe(256, 256, 128, 2, "f64", 0, fused=False, **B200))
    assert (p["ty"], p["stages"], p["xc"], p["gx"], p["gy"], p["cluster"]) == (8, 7, 64, 32, 4, 4)
    # config 2, the fused step: one group of 10 scalars, 5 per warp, 2 splits + the momentum role = 15 warps
    text = binding.plan_describe(512, 512, 256, 2, "f64", 10, fused=True, **B200)
    assert text.startswith("tma_fused(momentum+scalars)")
    p = parse(text)
    assert (p["group"], p["per_warp"], p["split"], p["ty"], p["stages"], p["xc"]) == (10, 5, 2, 5, 4, 64)
    assert (p["gx"], p["gy"], p["colgroup"]) == (412, 8, 1)
    # config 2, the two north_star calls
    mom, sca = binding.plan_describe(512, 512, 256, 2, "f64", 10, fused=False, **B200).split("; ")
    pm, ps = parse(mom), parse(sca)
    assert (pm["ty"], pm["stages"], pm["gx"] * pm["gy"]) == (4, 6, 128 * 9)
    assert (ps["group"], ps["split"], ps["ty"], ps["stages"]) == (10, 2, 7, 3)
    # config 3 (fp32): twice the levels per z tile
    p = parse(binding.plan_describe(512, 512, 256, 2, "f32", 10, fused=True, **B200))
    assert (p["ty"], p["stages"], p["gx"]) == (5, 4, 206) and 50 <= p["xc"] <= 64
    # config 4: one x-slab chunk of 128 planes, 4 scalars
    p = parse(binding.plan_describe(128, 1024, 160, 2, "f64", 4, fused=True, **B200))
    assert (p["group"], p["split"], p["ty"]) == (4, 1, 7) and p["stages"] >= 5


def test_ragged_nz_plans(lib):
    # a column group of 2 (fp64, odd nz) needs ny + 2 halo even; the class blocks cost shared memory
    t = binding.plan_describe(512, 512, 255, 2, "f64", 10, fused=True, **B200)
    p = parse(t)
    assert p["colgroup"] == 2 and p["ty"] == 5 and p["stages"] == 4 and p["smem"] > 199744
    assert "momentum role only" in binding.plan_describe(256, 256, 127, 2, "f64", 0, fused=False, **B200)
    assert "colgroup=4" in binding.plan_describe(64, 64, 33, 2, "f32", 3, fused=True, **B200)
    assert "colgroup=2" in binding.plan_describe(64, 64, 34, 2, "f32", 3, fused=True, **B200)
    assert "no TMA plan" in binding.plan_describe(512, 511, 255, 2, "f64", 10, fused=True, **B200)
    # columns taller than tma_momentum's 16 warps: the z-tiled kernel's momentum role
    assert "momentum role only" in binding.plan_describe(64, 64, 1100, 2, "f64", 0, fused=False, **B200)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", [(16, 16, 32), (64, 64, 64), (256, 256, 128), (100, 37, 72), (512, 512, 256),
                                   (1024, 1024, 160), (2048, 2048, 64), (33, 1, 8), (7, 300, 1024)])
@pytest.mark.parametrize("nq", [0, 1, 4, 10])
def test_every_plan_fits_the_device(shape, dtype, nq, lib):
    nx, ny, nz = shape
    for fused in (True, False):
        text = binding.plan_describe(nx, ny, nz, 2, dtype, nq, fused=fused, **B200)
        assert "no TMA plan" not in text, text
        for part in text.split("; "):
            p = parse(part)
            assert 0 < p["smem"] <= 227 * 1024, part
            assert p["stages"] >= 2 and 1 <= p["xc"] <= nx and p["ty"] >= 1
            assert p["gy"] == -(-nx // p["xc"])                     # the x chunks cover the planes
            if "tma_momentum" in part:
                assert p["gx"] >= -(-ny // p["ty"])                  # y tiles (padded to whole clusters)
            if "group" in p:
                # the fused launch holds every scalar in one group; the scalars launch may use two groups of 5
                assert p["group"] in ((min(nq, 10),) if "tma_fused" in part else (min(nq, 5), min(nq, 10)))
                assert p["per_warp"] * p["split"] >= p["group"]
                roles = p["split"] + (1 if "tma_fused" in part else 0)
                assert p["ty"] * roles <= 15                         # consumer warps beside the producer warp


def test_plans_respect_the_shared_memory_of_the_device(lib):
    # less opt-in shared memory: a shallower ring or a smaller tile, never over the limit
    for smem in (232448, 166912, 101376):
        for args in ((512, 512, 256, 2, "f64", 10, True), (256, 256, 128, 2, "f64", 0, False), (512, 512, 255, 2, "f64", 10, True)):
            for part in binding.plan_describe(*args, sm_count=148, smem_optin=smem).split("; "):
                assert parse(part)["smem"] <= smem - 1024, (smem, part)
