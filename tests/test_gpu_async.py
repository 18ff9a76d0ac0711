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


def test_step_async_automatic_chunk_count():
    # monc_adv_set_chunks(h, 0), the default: the library picks the count per step from the bytes
    # on the host link (T (1 + 1/C) + C c); the count is known once a step is enqueued
    cfg = gc.custom_cfg(40, 24, 64, nq=2, cid=405)
    P, L = gc.make_pair(cfg)
    assert L.step_chunk_count() == 0  # automatic, nothing enqueued yet
    with pytest.raises(binding.MoncAdvError) as e:
        L.step_chunk_range(0)
    assert e.value.code == binding.EINVAL
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    names = synth.field_names(cfg)
    Q = [synth.field(cfg, n) for n in names]
    hin = [pinned(a, L) for a in (U, V, W)]
    hq = [pinned(a, L) for a in Q]
    hout, hsq = pinned_out(L, 3), pinned_out(L, 2)
    L.step_async(*hin, hq, *hout, hsq)
    C = L.step_chunk_count()
    assert 1 <= C <= cfg.nx
    covered = []
    for c in range(C):
        L.step_wait_chunk(c)
        covered.append(L.step_chunk_range(c))
    assert covered[0][0] == 0 and covered[-1][1] == cfg.nx
    assert all(a[1] == b[0] for a, b in zip(covered[:-1], covered[1:]))
    L.step_wait()
    for o, w_, n in zip(hout, P.momentum(U, V, W), ("su", "sv", "sw")):
        gc.check(cfg, o, w_, n)
        gc.check_halo_untouched(cfg, o, n)
    for o, q, n in zip(hsq, Q, names):
        gc.check(cfg, o, P.scalar(U, V, W, q), n)
    # a fixed count again: known without a step, and the result does not depend on it
    L.set_chunks(3)
    assert L.step_chunk_count() == 3
    hout2, hsq2 = pinned_out(L, 3), pinned_out(L, 2)
    L.step_async(*hin, hq, *hout2, hsq2)
    L.step_wait()
    for a_, b_ in zip(hout + hsq, hout2 + hsq2):
        assert torch.equal(a_, b_)
    L.close()


@pytest.mark.parametrize("nz,dtype", [(65, "f64"), (66, "f32"), (35, "f32")])
def test_step_async_ragged_nz(nz, dtype):
    # nz that is not a whole number of 16-byte vectors: the fused TMA launch per chunk all the same
    cfg = gc.custom_cfg(18, 12, nz, nq=3, dtype=dtype, cid=406)
    P, L = gc.make_pair(cfg)
    L.set_variant("tma")
    L.set_chunks(4)
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    names = synth.field_names(cfg)
    Q = [synth.field(cfg, n) for n in names]
    hin = [pinned(a, L) for a in (U, V, W)]
    hq = [pinned(a, L) for a in Q]
    hout, hsq = pinned_out(L, 3), pinned_out(L, 3)
    L.step_async(*hin, hq, *hout, hsq)
    L.step_wait()
    assert "tma_fused" in L.describe_plan()
    for o, w_, n in zip(hout, P.momentum(U, V, W), ("su", "sv", "sw")):
        gc.check(cfg, o, w_, n)
        gc.check_halo_untouched(cfg, o, n)
    for o, q, n in zip(hsq, Q, names):
        gc.check(cfg, o, P.scalar(U, V, W, q), n)
        gc.check_halo_untouched(cfg, o, n)
    L.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("accumulate", [False, True])
def test_step_async_graph_replay(dtype, accumulate):
    # a step whose arguments equal those of the step before is captured into a CUDA graph and replayed:
    # step 1 call by call, step 2 captured + launched, steps 3.. replayed.  The host changes its fields
    # between steps (same arrays); every step must equal the call-by-call enqueue bitwise, the per-chunk
    # completion calls and the timing record must keep working, a setter must drop the graph
    cfg = gc.custom_cfg(24, 12, 64, nq=3, dtype=dtype, cid=407)
    P, L = gc.make_pair(cfg)
    _, Lref = gc.make_pair(cfg)
    Lref.set_graph(False)
    for lib in (L, Lref):
        lib.set_chunks(4)
        lib.set_accumulate(accumulate)
    names = ["u", "v", "w"] + synth.field_names(cfg)
    H = [synth.field(cfg, n) for n in names]
    hin = [pinned(a, L) for a in H]
    hout, href = pinned_out(L, 6), pinned_out(L, 6)
    h = cfg.halo
    rng = np.random.default_rng(5)
    for step in range(1, 7):
        if step == 5:
            L.set_form("flux")   # any setter drops the graph: this step is enqueued call by call again
        for t in hin:                # the model moves on: new values in the same pinned arrays
            t.numpy()[...] += rng.normal(0.0, 0.01, size=t.shape).astype(t.numpy().dtype)
        if accumulate:               # in/out source terms: both start from the same host values
            for a_, b_ in zip(hout, href):
                a_.numpy()[h:h + cfg.nx, h:h + cfg.ny] = step
                b_.numpy()[h:h + cfg.nx, h:h + cfg.ny] = step
        L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
        assert L.step_chunk_count() == 4
        # steps 1 and 5 (new settings) go call by call, 2 and 6 are captured, 3 and 4 replayed
        assert L.graph_state() == (1 if step in (1, 5) else 2), (step, L.graph_state())
        assert Lref.graph_state() == 0
        L.step_inputs_consumed()
        covered = 0
        for c in range(4):           # streaming combine on a replayed step
            L.step_wait_chunk(c)
            a, b = L.step_chunk_range(c)
            covered += b - a
        assert covered == cfg.nx
        L.step_wait()
        t = L.step_times_ms()
        assert t["total"] > 0 and t["kernels"] > 0 and t["h2d"] > 0 and t["d2h"] > 0
        Lref.step_async(hin[0], hin[1], hin[2], hin[3:], href[0], href[1], href[2], href[3:])
        Lref.step_wait()
        for a_, b_, n in zip(hout, href, ["su", "sv", "sw"] + names[3:]):
            assert torch.equal(a_, b_), (step, n)
        if not accumulate:
            U, V, W = (t_.numpy().astype(np.float64) for t_ in hin[:3])
            for o, w_, n in zip(hout[:3], P.momentum(U, V, W), ("su", "sv", "sw")):
                gc.check(cfg, o, w_, f"{n}[step {step}]")
    # 6 steps x 4 chunks, one fused launch each, replayed launches counted too
    assert L.launch_count() == 24 and Lref.launch_count() == 24
    # a user stream: the step starts after the stream's work and the stream waits for the step
    st = torch.cuda.Stream()
    for _ in range(3):
        L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:], stream=st)
        st.synchronize()
        L.step_wait()
    L.close()
    Lref.close()


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
# size, in the launch configuration bench.py times: EVERY interior element of
# all 13 outputs, of the two north_star calls and of the fused launch, against
# the oracle (threaded over the host cores: a full pass costs seconds).
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("cid", [2, 3])
def test_config2_and_3_full_size_every_element(cid):
    cfg = synth.CONFIGS[cid]
    P, L = gc.make_pair(cfg)
    nthr = oracle.max_threads()
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    names = synth.field_names(cfg)
    d = [gc.to_dev(a, L) for a in (U, V, W)]
    dq = [gc.to_dev(synth.field(cfg, n), L) for n in names]
    two = gc.fresh_out(L, 3 + cfg.nq)
    L.momentum(*d, *two[:3])
    L.scalars(dq, two[3:])
    assert "tma_momentum" in L.describe_plan() and "tma_scalars" in L.describe_plan(), L.describe_plan()
    # the whole step through monc_adv_tendencies (bench.py's headline): ONE fused launch
    fo = gc.fresh_out(L, 3 + cfg.nq)
    L.tendencies(*d, fo[0], fo[1], fo[2], dq, fo[3:])
    torch.cuda.synchronize()
    assert "tma_fused" in L.describe_plan(), L.describe_plan()
    errs = {}
    want = P.momentum(U, V, W, nthreads=nthr)
    for idx, nm in enumerate(("su", "sv", "sw")):
        errs[nm] = (gc.check(cfg, two[idx], want[idx], nm + "[two calls]"),
                    gc.check(cfg, fo[idx], want[idx], nm + "[fused]"))
        gc.check_halo_untouched(cfg, two[idx], nm)
        gc.check_halo_untouched(cfg, fo[idx], nm)
    del want
    sq = np.zeros(P.shape)
    for idx, nm in enumerate(names):
        P.scalar(U, V, W, synth.field(cfg, nm), nthreads=nthr, out=sq)
        errs[nm] = (gc.check(cfg, two[3 + idx], sq, nm + "[two calls]"),
                    gc.check(cfg, fo[3 + idx], sq, nm + "[fused]"))
        gc.check_halo_untouched(cfg, fo[3 + idx], nm)
    print(f"config{cid} full-array max rel errs (two calls, fused):",
          {k: (f"{a:.1e}", f"{b:.1e}") for k, (a, b) in errs.items()})
    L.close()


def test_ragged_nz_full_size_every_element():
    # bench.py's `ragged_nz` record: config 2 with one level less (512x512x255 fp64, 3 + 10 fields,
    # the fused launch on the grouped-column view), every interior element of all 13 outputs
    cfg = dataclasses.replace(synth.CONFIGS[2], nz=255)
    P, L = gc.make_pair(cfg)
    nthr = oracle.max_threads()
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    names = synth.field_names(cfg)
    d = [gc.to_dev(a, L) for a in (U, V, W)]
    dq = [gc.to_dev(synth.field(cfg, n), L) for n in names]
    fo = gc.fresh_out(L, 3 + cfg.nq)
    L.tendencies(*d, fo[0], fo[1], fo[2], dq, fo[3:])
    torch.cuda.synchronize()
    assert "tma_fused" in L.describe_plan() and "colgroup=2" in L.describe_plan(), L.describe_plan()
    errs = {}
    want = P.momentum(U, V, W, nthreads=nthr)
    for idx, nm in enumerate(("su", "sv", "sw")):
        errs[nm] = gc.check(cfg, fo[idx], want[idx], nm)
        gc.check_halo_untouched(cfg, fo[idx], nm)
    del want
    sq = np.zeros(P.shape)
    for idx, nm in enumerate(names):
        P.scalar(U, V, W, synth.field(cfg, nm), nthreads=nthr, out=sq)
        errs[nm] = gc.check(cfg, fo[3 + idx], sq, nm)
        gc.check_halo_untouched(cfg, fo[3 + idx], nm)
    print("ragged nz = 255 full-array max rel errs:", {k: f"{a:.1e}" for k, a in errs.items()})
    L.close()


def test_config4_hybrid_async_full_size():
    """1024x1024x160, 3 momentum + 4 scalars in pinned host memory, 8 chunks, the
    20-step loop of BASELINE.json configs[4]: the seeded fields are perturbed every
    step; steps 1, 10 and 20 are compared with the oracle on EVERY
    interior element of all 7 outputs (chunk seams included)."""
    cfg = synth.CONFIGS[4]
    steps_checked = (1, 10, 20)
    P, L = gc.make_pair(cfg)
    L.set_chunks(8)
    nthr = oracle.max_threads()
    names = ["u", "v", "w"] + synth.field_names(cfg)
    hin = [pinned(synth.field(cfg, n), L) for n in names]
    hout = pinned_out(L, len(names))
    sq = np.zeros(P.shape)
    for step in range(1, cfg.steps + 1):
        if step > 1:
            L.step_inputs_consumed()   # the host may overwrite its fields once the H2D copies are done
            L.step_wait()
        for n, t in zip(names, hin):
            synth.perturb(cfg, n, t.numpy(), step)   # in place on the pinned inputs
        L.step_async(hin[0], hin[1], hin[2], hin[3:], hout[0], hout[1], hout[2], hout[3:])
        if step not in steps_checked:
            continue
        L.step_wait()
        assert "tma_fused" in L.describe_plan(), L.describe_plan()
        U, V, W = (t.numpy() for t in hin[:3])
        errs = {}
        wm = P.momentum(U, V, W, nthreads=nthr)
        for idx, nm in enumerate(("su", "sv", "sw")):
            errs[nm] = gc.check(cfg, hout[idx].numpy(), wm[idx], f"{nm}[step {step}]")
        del wm
        for idx in range(3, len(names)):
            P.scalar(U, V, W, hin[idx].numpy(), nthreads=nthr, out=sq)
            errs[names[idx]] = gc.check(cfg, hout[idx].numpy(), sq, f"{names[idx]}[step {step}]")
        print(f"config4 step {step} full-array max rel errs:", {k: f"{v:.1e}" for k, v in errs.items()})
    for o, n in zip(hout, names):
        gc.check_halo_untouched(cfg, o, n)
    print("config4 step times (ms):", L.step_times_ms())
    L.close()


# ---------------------------------------------------------------------------
# accumulate inside the hybrid step:
# the host's own source terms go up with the fields, the advection tendencies are
# added on the device, the combined terms come back into the same arrays
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_step_async_accumulate_is_bitwise_wait_then_add(dtype):
    cfg = gc.custom_cfg(22, 13, 96, nq=3, dtype=dtype, cid=404)
    P, L = gc.make_pair(cfg)
    L.set_chunks(4)
    names = ["u", "v", "w"] + synth.field_names(cfg)
    hin = [pinned(synth.field(cfg, n), L) for n in names]
    # wait-all-then-add: the plain step into a separate result buffer, host adds
    plain = pinned_out(L, len(names))
    L.step_async(hin[0], hin[1], hin[2], hin[3:], plain[0], plain[1], plain[2], plain[3:])
    L.step_wait()
    rng = np.random.default_rng(5)
    host_terms = [torch.from_numpy(rng.standard_normal(L.shape)).to(L.torch_dtype) for _ in names]
    acc = [pinned(t.numpy(), L) for t in host_terms]
    L.set_accumulate(True)
    h = cfg.halo
    sl = (slice(h, h + cfg.nx), slice(h, h + cfg.ny))
    for rep in (1, 2):   # twice: the staging buffers must not carry step 1 into step 2
        base = [a_.clone() for a_ in acc]
        L.step_async(hin[0], hin[1], hin[2], hin[3:], acc[0], acc[1], acc[2], acc[3:])
        for c in range(4):   # streaming combine: a chunk's slab is final when its event fires
            L.step_wait_chunk(c)
            a, b = L.step_chunk_range(c)
            xs = slice(h + a, h + b)
            assert torch.equal(acc[0][xs, sl[1]], base[0][xs, sl[1]] + plain[0][xs, sl[1]])
        L.step_wait()
        for b_, a_, p_ in zip(base, acc, plain):
            assert torch.equal(a_[sl], b_[sl] + p_[sl])   # bitwise: the same add, done on the device
            m = torch.ones(L.shape, dtype=torch.bool)
            m[sl] = False
            assert torch.equal(a_[m], b_[m])              # halos untouched
    # scalars only, accumulate still on
    acc2 = [pinned(t.numpy(), L) for t in host_terms[3:]]
    L.step_async(hin[0], hin[1], hin[2], hin[3:], None, None, None, acc2)
    L.step_wait()
    for t0, a_, p_ in zip(host_terms[3:], acc2, plain[3:]):
        assert torch.equal(a_[sl], t0[sl] + p_[sl])
    L.close()


# ---------------------------------------------------------------------------
# the boundary refuses what would silently change the behaviour (C ABI called
# directly, without the binding's own checks)
# ---------------------------------------------------------------------------
def test_step_async_refuses_pageable_and_overlapping_arrays():
    import ctypes as C
    cfg = gc.custom_cfg(8, 6, 32, nq=1, cid=405)
    P, L = gc.make_pair(cfg)
    lib, hd = L._lib, L._h
    vp = C.c_void_p
    pin = [torch.zeros(L.shape, dtype=L.torch_dtype).pin_memory() for _ in range(8)]
    pageable = torch.zeros(L.shape, dtype=L.torch_dtype)

    def call(hu, hv, hw, hq, hsu, hsv, hsw, hsq):
        qt = (vp * 1)(hq.data_ptr())
        st = (vp * 1)(hsq.data_ptr())
        return lib.monc_adv_step_async(hd, vp(hu.data_ptr()), vp(hv.data_ptr()), vp(hw.data_ptr()), qt, 1,
                                       vp(hsu.data_ptr()), vp(hsv.data_ptr()), vp(hsw.data_ptr()), st, None)

    # "silently reverting from an asynchronous to a synchronous deep copy"
    assert call(pageable, pin[1], pin[2], pin[3], pin[4], pin[5], pin[6], pin[7]) == binding.EINVAL
    assert b"page-locked" in lib.monc_adv_last_error(hd)
    assert call(pin[0], pin[1], pin[2], pin[3], pin[4], pin[5], pin[6], pageable) == binding.EINVAL
    # a device pointer is not a host array either
    dev = torch.zeros(L.shape, dtype=L.torch_dtype, device="cuda")
    assert call(dev, pin[1], pin[2], pin[3], pin[4], pin[5], pin[6], pin[7]) == binding.EINVAL
    # overlapping (not merely identical) arrays: an output that starts inside an input
    big = torch.zeros(2 * int(np.prod(L.shape)), dtype=L.torch_dtype).pin_memory()
    n = int(np.prod(L.shape))
    a_in, b_out = big[:n].view(L.shape), big[n // 2 + 2:n // 2 + 2 + n].view(L.shape)
    assert call(a_in, pin[1], pin[2], pin[3], b_out, pin[5], pin[6], pin[7]) == binding.EINVAL
    assert b"overlap" in lib.monc_adv_last_error(hd)
    # nothing is in flight after the refusals: a good call goes through
    assert call(pin[0], pin[1], pin[2], pin[3], pin[4], pin[5], pin[6], pin[7]) == binding.OK
    assert lib.monc_adv_step_wait(hd) == binding.OK
    L.close()
