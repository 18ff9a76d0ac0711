"""SURVEY.md 8(f) NEXT-3 on the hardware there is: the x-slab decomposition with its
halo swap AND the CUDA kernels together, on one device.  A periodic global domain
is cut into 2 and 3 x-slabs held as separate arrays (the paper's 8-ranks-per-GPU
picture), the rim planes move by device-to-device copies
(dist.exchange_halo_x_same_device: the data motion of the NCCL swap minus the wire),
every slab is advected by its own handle through monc_adv_tendencies, and the result
must equal the single-domain launch BITWISE (columns are independent, PAPER.md:73;
SURVEY 8(f) NEXT-3 pin).  The multi-process swap itself is covered on CPU by
tests/test_dist_gloo.py (gloo, world size 2 and 3)."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2009_12850_b200 import binding, dist as pd, synth
import gpu_common as gc
import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def _need_gpu(gpu_required):
    yield
    torch.cuda.synchronize()


def _handle(cfg, nx):
    g = synth.grid(cfg.nz)
    return binding.MoncAdv(nx, cfg.ny, cfg.nz, cfg.halo, synth.DX, synth.DY, g["dz"], g["dzn"], g["rho"],
                           g["rhon"], dtype=cfg.dtype)


@pytest.mark.parametrize("world,nx,dtype,depth", [(2, 40, "f64", 2), (3, 41, "f64", 1), (3, 37, "f32", 2)])
def test_slabs_on_one_device_match_single_domain_bitwise(world, nx, dtype, depth):
    cfg = gc.custom_cfg(nx, 19, 192, nq=3, dtype=dtype, cid=500 + world)
    h = cfg.halo
    names = ["u", "v", "w"] + synth.field_names(cfg)
    G = {n: synth.interior_field(cfg, n) for n in names}
    # ---- single-domain reference through the library, checked against the oracle
    P, L = gc.make_pair(cfg)
    full = [gc.to_dev(synth.embed(G[n], h), L) for n in names]
    ref = gc.fresh_out(L, len(names))
    L.tendencies(full[0], full[1], full[2], ref[0], ref[1], ref[2], full[3:], ref[3:])
    torch.cuda.synchronize()
    Hf = [synth.embed(G[n], h) for n in names]
    want = list(P.momentum(Hf[0], Hf[1], Hf[2])) + [P.scalar(Hf[0], Hf[1], Hf[2], q) for q in Hf[3:]]
    for o, w_, n in zip(ref, want, names):
        gc.check(cfg, o, w_, n)
    # ---- the decomposed run: separate arrays per slab, rims filled by the swap only
    slabs, ranges = [], []
    for r in range(world):
        x0, x1 = pd.slab_range(cfg.nx, world, r)
        ranges.append((x0, x1))
        fs = []
        for n in names:
            f = pd.local_from_global(G[n], h, world, r).to(device="cuda", dtype=L.torch_dtype).contiguous()
            pd.fill_halo_y_periodic(f, h)
            fs.append(f)
        slabs.append(fs)
    pd.exchange_halo_x_same_device(slabs, h, depth=depth)
    for r, (x0, x1) in enumerate(ranges):
        for f, ff in zip(slabs[r], full):
            assert torch.equal(f[h - depth:h + (x1 - x0) + depth], ff[x0 + h - depth:x1 + h + depth]), "rim differs"
        Lr = _handle(cfg, x1 - x0)
        outs = gc.fresh_out(Lr, len(names))
        fs = slabs[r]
        Lr.tendencies(fs[0], fs[1], fs[2], outs[0], outs[1], outs[2], fs[3:], outs[3:])
        torch.cuda.synchronize()
        for o, o_ref, n in zip(outs, ref, names):
            assert torch.equal(o[h:h + (x1 - x0), h:h + cfg.ny], o_ref[h + x0:h + x1, h:h + cfg.ny]), \
                f"slab {r} of {world}: tendency of {n} differs from the single-domain launch"
        Lr.close()
    L.close()


def test_exchange_halo_x_world_one_on_cuda_tensors():
    # the torch.distributed entry point with one rank: the periodic wrap is a local copy on the device
    cfg = gc.custom_cfg(9, 6, 32, nq=1, cid=510)
    h = cfg.halo
    Gi = synth.interior_field(cfg, "theta")
    f = pd.local_from_global(Gi, h, 1, 0).cuda()
    pd.fill_halo_y_periodic(f, h)
    pd.exchange_halo_x([f], h)
    assert np.array_equal(f.cpu().numpy(), synth.embed(Gi, h))
