"""N > 1 host logic on CPU: world_size 2 and 3 `gloo` process groups.

Covers paper_2009_12850_b200/dist.py: the x-slab decomposition,
the periodic halo swap that precedes advection and the
max-over-ranks timing rule bench.py uses.  The advection itself runs in the
CPU oracle here (tests may use it): a decomposed run must reproduce the
single-domain result BITWISE, because columns are independent.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, nx, depth):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from paper_2009_12850_b200 import dist as pd, synth

        cfg = synth.Config(77, nx, 6, 8, halo=2, nq=2)
        h = cfg.halo
        names = ["u", "v", "w"] + synth.field_names(cfg)
        G = {n: synth.interior_field(cfg, n) for n in names}
        full = {n: synth.embed(G[n], h) for n in names}           # single-domain reference
        x0, x1 = pd.slab_range(cfg.nx, world, rank)
        loc = [pd.local_from_global(G[n], h, world, rank) for n in names]
        for f in loc:
            pd.fill_halo_y_periodic(f, h)
        pd.exchange_halo_x(loc, h, depth=depth)
        for n, f in zip(names, loc):
            want = full[n][x0 + h - depth:x1 + h + depth]
            got = f.numpy()[h - depth:h + (x1 - x0) + depth]
            assert np.array_equal(got, want), f"rank {rank}: halo of {n} differs"

        # advection on the slab == the same planes of the single-domain result, bitwise
        g = synth.grid(cfg.nz)
        Pg = oracle.Problem(cfg.nx, cfg.ny, cfg.nz, h, synth.DX, synth.DY, g["dz"], g["dzn"], g["rho"], g["rhon"])
        Pl = oracle.Problem(x1 - x0, cfg.ny, cfg.nz, h, synth.DX, synth.DY, g["dz"], g["dzn"], g["rho"], g["rhon"])
        A = [f.numpy() for f in loc]
        wg = list(Pg.momentum(full["u"], full["v"], full["w"])) + \
            [Pg.scalar(full["u"], full["v"], full["w"], full[n]) for n in names[3:]]
        wl = list(Pl.momentum(A[0], A[1], A[2])) + [Pl.scalar(A[0], A[1], A[2], q) for q in A[3:]]
        for a, b, n in zip(wl, wg, names):
            assert np.array_equal(a[h:h + x1 - x0, h:h + cfg.ny], b[h + x0:h + x1, h:h + cfg.ny]), \
                f"rank {rank}: tendency of {n} differs from the single-domain run"

        # timing rule: max over ranks; whole-job value counts every rank's points
        assert pd.max_over_ranks(10.0 + rank) == 10.0 + world - 1
        assert pd.whole_job_value(1000, 5, 2.0, world) == pytest.approx(world * 1000 * 5 / 2e-3 / 1e9)
        # every interior plane belongs to exactly one rank
        cover = torch.zeros(cfg.nx, dtype=torch.int64)
        cover[x0:x1] += 1
        dist.all_reduce(cover)
        assert bool((cover == 1).all())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,nx,depth", [(2, 12, 2), (2, 7, 1), (3, 11, 2)])
def test_decomposed_run_matches_single_domain(world, nx, depth):
    mp.spawn(_worker, args=(world, _free_port(), nx, depth), nprocs=world, join=True)


def test_single_rank_wrap_and_ranges():
    sys.path.insert(0, ROOT)
    from paper_2009_12850_b200 import dist as pd, synth
    cfg = synth.Config(78, 5, 4, 6, halo=2)
    Gi = synth.interior_field(cfg, "u")
    f = pd.local_from_global(Gi, 2, 1, 0)
    pd.fill_halo_y_periodic(f, 2)
    pd.exchange_halo_x([f], 2)
    assert np.array_equal(f.numpy(), synth.embed(Gi, 2))
    assert [pd.slab_range(10, 4, r) for r in range(4)] == [(0, 3), (3, 6), (6, 8), (8, 10)]
    with pytest.raises(ValueError):
        pd.slab_range(2, 3, 0)
    with pytest.raises(ValueError):
        pd.exchange_halo_x([f], 2, depth=3)


@pytest.mark.parametrize("world,nx,depth", [(2, 9, 2), (3, 11, 1), (4, 8, 2)])
def test_same_device_slab_swap_matches_single_domain(world, nx, depth):
    """Several sub-domains in one process (8 ranks share a GPU): the rims
    filled by exchange_halo_x_same_device equal the single-domain periodic halos."""
    sys.path.insert(0, ROOT)
    from paper_2009_12850_b200 import dist as pd, synth
    cfg = synth.Config(79, nx, 5, 6, halo=2, nq=1)
    h = cfg.halo
    names = ["u", "theta"]
    G = {n: synth.interior_field(cfg, n) for n in names}
    slabs = []
    for r in range(world):
        fs = [pd.local_from_global(G[n], h, world, r) for n in names]
        for f in fs:
            pd.fill_halo_y_periodic(f, h)
        slabs.append(fs)
    pd.exchange_halo_x_same_device(slabs, h, depth=depth)
    for r in range(world):
        x0, x1 = pd.slab_range(nx, world, r)
        for n, f in zip(names, slabs[r]):
            want = synth.embed(G[n], h)[x0 + h - depth:x1 + h + depth]
            assert np.array_equal(f.numpy()[h - depth:h + (x1 - x0) + depth], want)
