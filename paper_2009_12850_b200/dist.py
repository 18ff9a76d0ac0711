"""Multi-GPU plumbing: x-slab domain decomposition and the periodic halo swap.

SURVEY.md 8(e): advection columns are independent and the stencil
reaches +-1 in x and y, so the horizontal domain is partitioned, one sub-domain
plus a `halo`-deep rim per GPU -- the paper's MPI picture ("all
prognostics [are] halo swapped between neighbouring processes" at the start of
a timestep).  The advection kernels themselves contain no collective: the only
exchange step is the halo swap that precedes them, and it is done here with
`torch.distributed` point-to-point operations (NCCL over NVLink/NVSwitch on
GPUs; gloo on CPU tensors in the tests).

Decomposition axis: x, the slowest axis of the z-fastest layout
F[NXH][NYH][nz].  An x plane is one contiguous run of NYH*nz elements, so the
planes a neighbour needs are sent straight out of the field array and received
straight into the neighbour's rim: no pack/unpack kernels, no staging buffers.
y is not decomposed; its periodic wrap is a local copy.

This module holds no advection arithmetic.  It never imports the oracle.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def slab_range(nx_global: int, world: int, rank: int) -> tuple[int, int]:
    """Interior x range [x0, x1) of `rank`'s slab: as even as possible, the
    remainder spread over the first ranks."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    if nx_global < world:
        raise ValueError("need at least one x plane per rank")
    base, rem = divmod(nx_global, world)
    x0 = rank * base + min(rank, rem)
    return x0, x0 + base + (1 if rank < rem else 0)


def local_from_global(interior_global, halo: int, world: int, rank: int) -> torch.Tensor:
    """This rank's slab of a global interior array [nx, ny, nz] as a tensor
    [nxl + 2h, ny + 2h, nz] whose rims are NOT yet valid (zeros)."""
    g = torch.as_tensor(interior_global)
    x0, x1 = slab_range(g.shape[0], world, rank)
    f = torch.zeros((x1 - x0 + 2 * halo, g.shape[1] + 2 * halo, g.shape[2]), dtype=g.dtype)
    f[halo:halo + (x1 - x0), halo:halo + g.shape[1]] = g[x0:x1]
    return f


def fill_halo_y_periodic(f: torch.Tensor, halo: int) -> torch.Tensor:
    """Periodic wrap in y (not decomposed): a local copy, all x planes. In place."""
    ny = f.shape[1] - 2 * halo
    f[:, :halo] = f[:, ny:ny + halo]
    f[:, ny + halo:] = f[:, halo:2 * halo]
    return f


def exchange_halo_x(fields, halo: int, depth: int | None = None, group=None):
    """Periodic halo swap in x of every tensor in `fields` (each
    [nxl + 2h, NYH, nz], contiguous, same device).  After the call the `depth`
    rim planes next to the interior on both sides hold the neighbours' edge
    planes (ring topology: rank r-1 to the west, r+1 to the east, wrapping).
    `depth` defaults to `halo`; the advection stencil itself needs only 1.

    All sends and receives of all fields go out as ONE batch
    (`batch_isend_irecv`: a single NCCL group call on GPUs), planes sent in
    place.  With one rank the wrap is a local copy.  The y rims of the received
    planes are whatever the sender held: call `fill_halo_y_periodic` BEFORE the
    swap so that corners arrive filled.
    """
    fields = list(fields)
    depth = halo if depth is None else depth
    if not 1 <= depth <= halo:
        raise ValueError("need 1 <= depth <= halo")
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    for f in fields:
        if not f.is_contiguous():
            raise ValueError("exchange_halo_x needs contiguous fields")
        if f.shape[0] - 2 * halo < depth:
            raise ValueError("slab thinner than the halo depth")
    if world == 1:
        for f in fields:
            nxl = f.shape[0] - 2 * halo
            f[halo - depth:halo] = f[nxl + halo - depth:nxl + halo]
            f[nxl + halo:nxl + halo + depth] = f[halo:halo + depth]
        return None
    west = (rank - 1) % world
    east = (rank + 1) % world
    if group is not None:
        west, east = dist.get_global_rank(group, west), dist.get_global_rank(group, east)
    ops = []
    for f in fields:
        nxl = f.shape[0] - 2 * halo
        send_w = f[halo:halo + depth]                   # my first interior planes -> west's east rim
        send_e = f[nxl + halo - depth:nxl + halo]       # my last interior planes -> east's west rim
        recv_w = f[halo - depth:halo]
        recv_e = f[nxl + halo:nxl + halo + depth]
        ops += [dist.P2POp(dist.isend, send_e, east, group), dist.P2POp(dist.irecv, recv_w, west, group),
                dist.P2POp(dist.isend, send_w, west, group), dist.P2POp(dist.irecv, recv_e, east, group)]
    reqs = dist.batch_isend_irecv(ops)
    for r in reqs:
        r.wait()
    return None


def exchange_halo_x_same_device(slabs, halo: int, depth: int | None = None):
    """The same periodic swap for several sub-domains that live in ONE process on ONE
    device (the paper runs 8 ranks per GPU; with a single GPU it
    is also how the decomposed path is exercised on hardware): `slabs[r]` is the
    list of field tensors of sub-domain r, ring order.  Planes move by
    device-to-device copies on the current stream, straight from the neighbour's
    edge planes into the rim: the data motion `exchange_halo_x` performs with
    isend/irecv, minus the wire."""
    depth = halo if depth is None else depth
    if not 1 <= depth <= halo:
        raise ValueError("need 1 <= depth <= halo")
    world = len(slabs)
    for r in range(world):
        east = slabs[(r + 1) % world]
        for f, fe in zip(slabs[r], east):
            if not (f.is_contiguous() and fe.is_contiguous()):
                raise ValueError("exchange_halo_x_same_device needs contiguous fields")
            nxl, nxe = f.shape[0] - 2 * halo, fe.shape[0] - 2 * halo
            if min(nxl, nxe) < depth:
                raise ValueError("slab thinner than the halo depth")
            fe[halo - depth:halo].copy_(f[nxl + halo - depth:nxl + halo], non_blocking=True)  # my last planes -> east's west rim
            f[nxl + halo:nxl + halo + depth].copy_(fe[halo:halo + depth], non_blocking=True)   # east's first planes -> my east rim
    return None


def max_over_ranks(value: float, device="cpu", group=None) -> float:
    """Timing rule: a multi-rank number is the MAX over ranks."""
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def whole_job_value(points_per_rank: int, steps: int, ms: float, world: int) -> float:
    """Aggregate Gpts/s of a weak-scaling job: every rank advects
    `points_per_rank` per step; `ms` is the max-over-ranks time of `steps` steps."""
    return world * points_per_rank * steps / (ms * 1e-3) / 1e9
