"""Hybrid asynchronous step and the
large configs of BASELINE.json, through the C ABI."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2009_12850_b200 import binding, synth
import gpu_common as gc
import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def _need_gpu(gpu_required):
    yield
    torch.cuda.synchronize()


def pinned(a, L):
    t = torch.empty(L.shape, dtype=L.torch_dtype).pin_memory()
    t.copy_(torch.from_numpy(a))
    return t


def pinned_out(L, n):
    return [torch.full(L.shape, gc.SENTINEL, dtype=L.torch_dtype).pin_memory() for _ in range(n)]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("nchunks,overlap", [(8, True), (3, True), (1, True), (8, False), (20, True)])
def test_step_async_small(nchunks, overlap, dtype):
    cfg = gc.custom_cfg(20, 12, 64, nq=3, dtype=dtype, cid=400)
    P, L = gc.make_pair(cfg)
    L.set_chunks(nchunks)
    L.set_overlap(overlap)
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    names = synth.field_names(cfg)
    Q = [synth.field(cfg, n) for n in names]
    hin = [pinned(a, L) for a in (U, V, W)]
    hq = [pinned(a, L) for a in Q]
    hout = pinned_out(L, 3)
    hsq = pinned_out(L, 3)
    L.step_async(*hin, hq, *hout, hsq)
    with pytest.raises(binding.MoncAdvError) as e:  # EBUSY until waited
        L.step_async(*hin, hq, *hout, hsq)
    assert e.value.code == binding.EBUSY
    L.step_inputs_consumed()
    # per-chunk completion: chunk 0's planes are final once its event fired
    L.step_wait_chunk(0)
    a, b = L.step_chunk_range(0)
    want = P.momentum(U, V, W)
    h = cfg.halo
    got0 = hout[0].numpy()[h + a:h + b, h:h + cfg.ny].astype(np.float64)
    scale = np.abs(gc.interior(cfg, want[0])).max()
    assert np.max(np.abs(got0 - want[0][h + a:h + b, h:h + cfg.ny])) <= gc.TOL[dtype] * scale
    L.step_wait()
    t = L.step_times_ms()
    assert t["total"] > 0 and t["kernels"] > 0
    for o, w_, n in zip(hout, want, ("su", "sv", "sw")):
        gc.check(cfg, o, w_, n)
        gc.check_halo_untouched(cfg, o, n)
    for o, q, n in zip(hsq, Q, names):
        gc.check(cfg, o, P.scalar(U, V, W, q), n)
        gc.check_halo_untouched(cfg, o, n)
    # chunking is invisible: bitwise equal to one whole-domain call (PAPER.md:73,
    # no dependency between columns)
    d = [gc.to_dev(x, L) for x in (U, V, W)]
    outs = gc.fresh_out(L, 3)
    L.momentum(*d, *outs)
    torch.cuda.synchronize()
    for o, ho in zip(outs, hout):
        assert np.array_equal(gc.interior(cfg, o.cpu().numpy()), gc.interior(cfg, ho.numpy()))
    # second step reuses the staging buffers; scalars-only call
    hsq2 = pinned_out(L, 3)
    L.step_async(*hin, hq, None, None, None, hsq2)
    L.step_wait()
    for a_, b_ in zip(hsq, hsq2):
        assert torch.equal(a_, b_)
    L.close()


def test_step_async_pw_skew():
    # the hybrid step in the PW-skew form (NEXT-1): x-slab launches of the TMA kernels
    cfg = gc.custom_cfg(24, 17, 128, nq=4, cid=403)
    P, L = gc.make_pair(cfg)
    L.set_form("pw_skew")
    L.set_chunks(5)
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    names = synth.field_names(cfg)
    Q = [synth.field(cfg, n) for n in names]
    hin = [pinned(a, L) for a in (U, V, W)]
    hq = [pinned(a, L) for a in Q]
    hout, hsq = pinned_out(L, 3), pinned_out(L, 4)
    L.step_async(*hin, hq, *hout, hsq)
    L.step_wait()
    assert "tma_fused" in L.describe_plan()  # one fused TMA launch per chunk
    for o, w_, n in zip(hout, P.momentum(U, V, W, skew=True), ("su", "sv", "sw")):
        gc.check(cfg, o, w_, n)
        gc.check_halo_untouched(cfg, o, n)
    for o, q, n in zip(hsq, Q, names):
        gc.check(cfg, o, P.scalar(U, V, W, q, skew=True), n)
    L.close()


def test_step_async_after_user_stream_work():
    cfg = gc.custom_cfg(16, 8, 32, cid=401)
    P, L = gc.make_pair(cfg)
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    hin = [pinned(a, L) for a in (U, V, W)]
    hout = pinned_out(L, 3)
    st = torch.cuda.Stream()
    L.step_async(*hin, [], *hout, [], stream=st)
    st.synchronize()          # the user stream waits for the step's last copy
    L.step_wait()
    for o, w_, n in zip(hout, P.momentum(U, V, W), ("su", "sv", "sw")):
        gc.check(cfg, o, w_, n)
    L.close()


# ---------------------------------------------------------------------------
# BASELINE.json configs 2, 3 (512x512x256, 3 momentum + 10 scalars) at full
# size: every output field checked on sampled points the oracle computes one
# by one, plus one x-slab compared element by element.
# ---------------------------------------------------------------------------
def _big_fields(cfg):
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    names = synth.field_names(cfg)
    return U, V, W, names


@pytest.mark.parametrize("cid", [2, 3])
def test_config2_and_3_full_size_sampled(cid):
    cfg = synth.CONFIGS[cid]
    P, L = gc.make_pair(cfg)
    U, V, W, names = _big_fields(cfg)
    d = [gc.to_dev(a, L) for a in (U, V, W)]
    outs = gc.fresh_out(L, 3)
    L.momentum(*d, *outs)
    torch.cuda.synchronize()
    rng = np.random.default_rng(cid)
    ii, jj, kk = gc.sample_points(cfg, 40000, rng)
    # scale: max |tendency| of the field, from the oracle on one x-slab (>= 8 planes)
    slab = dataclasses.replace(cfg, nx=8)
    Ps = oracle.Problem(slab.nx, slab.ny, slab.nz, slab.halo, synth.DX, synth.DY,
                        *[synth.grid(cfg.nz)[k] for k in ("dz", "dzn", "rho", "rhon")])
    sl = slice(100, 100 + 8 + 2 * cfg.halo)
    Us, Vs, Ws = (np.ascontiguousarray(a[sl]) for a in (U, V, W))
    want_slab = Ps.momentum(Us, Vs, Ws, nthreads=oracle.max_threads())
    for o, w_, n in zip(outs, want_slab, ("su", "sv", "sw")):
        scale = np.abs(gc.interior(slab, w_)).max()
        gc.check_sampled(cfg, P, n, o, U, V, W, None, ii, jj, kk, scale)
        # the slab, element by element (columns are independent: PAPER.md:73)
        got = o[sl].cpu().numpy()
        gc.check(slab, got, w_, n + "[slab]")
    outs_m, scales = outs, [np.abs(gc.interior(slab, w_)).max() for w_ in want_slab]
    # scalars, all nq in one batched call
    outs = gc.fresh_out(L, cfg.nq)
    dq = []
    for n in names:
        dq.append(gc.to_dev(synth.field(cfg, n), L))
    L.scalars(dq, outs)
    torch.cuda.synchronize()
    for n, o, q in zip(names, outs, dq):
        Q = synth.field(cfg, n)
        qs = np.ascontiguousarray(Q[sl])
        w_ = Ps.scalar(Us, Vs, Ws, qs, nthreads=oracle.max_threads())
        scale = np.abs(gc.interior(slab, w_)).max()
        gc.check_sampled(cfg, P, n, o, U, V, W, Q, ii, jj, kk, scale)
        gc.check(slab, o[sl].cpu().numpy(), w_, n + "[slab]")
        scales.append(scale)
    # the whole step through monc_adv_tendencies (the launch bench.py times as the
    # headline of this config): ONE fused launch, every element within tolerance of the
    # two-call results just checked against the oracle
    fo = gc.fresh_out(L, 3 + cfg.nq)
    L.tendencies(*d, fo[0], fo[1], fo[2], dq, fo[3:])
    torch.cuda.synchronize()
    assert "tma_fused" in L.describe_plan(), L.describe_plan()
    h = cfg.halo
    for a, b, sc, n in zip(fo, list(outs_m) + list(outs), scales, ["su", "sv", "sw"] + list(names)):
        ai, bi = (t[h:h + cfg.nx, h:h + cfg.ny] for t in (a, b))
        err = float((ai - bi).abs().max()) / sc
        assert err <= gc.TOL[cfg.dtype], f"{n}: fused vs two calls {err:.3e}"
        gc.check_sampled(cfg, P, n if n in ("su", "sv", "sw") else n, a, U, V, W,
                         None if n in ("su", "sv", "sw") else synth.field(cfg, n), ii, jj, kk, sc)
    L.close()


def test_config4_hybrid_async_full_size():
    """1024x1024x160, 3 momentum + 4 scalars in pinned host memory, 8 chunks.
    The seeded fields are perturbed every step; steps checked
    against the oracle on sampled points and one x-slab."""
    cfg = synth.CONFIGS[4]
    steps_checked = (1, 2, 3)
    P, L = gc.make_pair(cfg)
    L.set_chunks(8)
    names = ["u", "v", "w"] + synth.field_names(cfg)
    H = [synth.field(cfg, n) for n in names]
    hin = [pinned(a, L) for a in H]
    hout = pinned_out(L, len(names))
    rng = np.random.default_rng(4)
    slab = dataclasses.replace(cfg, nx=4)
    g = synth.grid(cfg.nz)
    Ps = oracle.Problem(slab.nx, slab.ny, slab.nz, slab.halo, synth.DX, synth.DY, g["dz"], g["dzn"], g["rho"], g["rhon"])
    for step in range(1, max(steps_checked) + 1):
        for n, t in zip(names, hin):
            synth.perturb(cfg, n, t.numpy(), step)   # in place on the pinned inputs
        L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
        L.step_inputs_consumed()
        L.step_wait()
        if step not in steps_checked:
            continue
        U, V, W = (t.numpy() for t in hin[:3])
        ii, jj, kk = gc.sample_points(cfg, 20000, rng)
        # chunk seams along x: sample planes next to every chunk boundary
        seams = [L.step_chunk_range(c)[0] + cfg.halo for c in range(1, 8)]
        ii[:2000] = np.array(seams + [s - 1 for s in seams])[rng.integers(0, 14, 2000)]
        sl = slice(381, 381 + 4 + 2 * cfg.halo)   # straddles the chunk seam at x = 384
        Us, Vs, Ws = (np.ascontiguousarray(a[sl]) for a in (U, V, W))
        wm = Ps.momentum(Us, Vs, Ws, nthreads=oracle.max_threads())
        for idx, n in enumerate(names):
            if idx < 3:
                w_ = wm[idx]
                q = None
                nm = ("su", "sv", "sw")[idx]
            else:
                q = hin[idx].numpy()
                w_ = Ps.scalar(Us, Vs, Ws, np.ascontiguousarray(q[sl]), nthreads=oracle.max_threads())
                nm = n
            scale = np.abs(gc.interior(slab, w_)).max()
            gc.check_sampled(cfg, P, nm, hout[idx].numpy(), U, V, W, q, ii, jj, kk, scale)
            gc.check(slab, hout[idx].numpy()[sl], w_, nm + "[slab]")
    t = L.step_times_ms()
    print("config4 step times (ms):", t)
    L.close()
