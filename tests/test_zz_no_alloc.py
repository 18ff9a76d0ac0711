"""monc_adv_step_noalloc: the momentum step from pinned host memory with its device staging in the library's
file-scope scratch array (no cudaMalloc, no stream or event creation), against the existing paths.

Collected last on purpose (the file name sorts after every other test file)."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2009_12850_b200 import binding, synth
import gpu_common as gc

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def _need_gpu(gpu_required):
    binding.select_build(False)
    yield
    torch.cuda.synchronize()


def pinned(a, L):
    t = torch.empty(L.shape, dtype=L.torch_dtype).pin_memory()
    t.copy_(torch.from_numpy(a))
    return t


def free_device_bytes():
    return torch.cuda.mem_get_info()[0]


# config 0's shape, the paper's per-process sub-domain (262144 points, the largest fp64 shape the
# scratch holds), a ragged nz
@pytest.mark.parametrize("shape,dtype", [((16, 16, 32), "f64"), ((64, 64, 64), "f64"), ((64, 64, 64), "f32"),
                                         ((20, 14, 37), "f64")])
def test_step_noalloc_matches_the_existing_paths_twice_in_a_row(shape, dtype):
    nx, ny, nz = shape
    cfg = gc.custom_cfg(nx, ny, nz, dtype=dtype, cid=900)
    cfg2 = gc.custom_cfg(nx, ny, nz, dtype=dtype, cid=901)      # other seeds: other fields for the second call
    P, L = gc.make_pair(cfg)
    fields = [[synth.field(c, n) for n in "uvw"] for c in (cfg, cfg2)]
    hin = [[pinned(a, L) for a in f] for f in fields]
    hout = [[torch.full(L.shape, gc.SENTINEL, dtype=L.torch_dtype).pin_memory() for _ in range(3)] for _ in range(3)]
    # the existing paths on the same inputs: monc_adv_momentum on device arrays, monc_adv_step_async
    dev_ref, async_ref = [], []
    for f, hi in zip(fields, hin):
        d = [gc.to_dev(a, L) for a in f]
        o = gc.fresh_out(L, 3)
        L.momentum(*d, *o)
        torch.cuda.synchronize()
        dev_ref.append([t.cpu() for t in o])
        ho = [torch.full(L.shape, gc.SENTINEL, dtype=L.torch_dtype).pin_memory() for _ in range(3)]
        L.step_async(*hi, [], *ho, [])
        L.step_wait()
        async_ref.append(ho)
    st = torch.cuda.Stream()
    # two calls in a row on one stream, no synchronisation in between: the second finds the first's
    # contents in the scratch; then the first inputs again
    L.step_noalloc(*hin[0], *hout[0], stream=st)
    L.step_noalloc(*hin[1], *hout[1], stream=st)
    st.synchronize()
    free_before = free_device_bytes()
    launches_before = L.launch_count()
    L.step_noalloc(*hin[0], *hout[2], stream=st)
    st.synchronize()
    assert free_device_bytes() == free_before, "a warm call changed the free device memory"
    assert L.launch_count() == launches_before + 1
    h = cfg.halo
    for call, which in ((0, 0), (1, 1), (2, 0)):
        want = P.momentum(*fields[which])
        for o, w_, dref, aref, n in zip(hout[call], want, dev_ref[which], async_ref[which], ("su", "sv", "sw")):
            gc.check(cfg, o, w_, f"{n}[call {call}] against the oracle")
            gc.check_halo_untouched(cfg, o, n)
            # against the existing paths, within the tolerance of the parity tests (the kernel is the
            # same, so the bits are too)
            scale = float(np.abs(gc.interior(cfg, w_)).max())
            gi = gc.interior(cfg, o.numpy()).astype(np.float64)
            for ref, nm in ((dref, "monc_adv_momentum"), (aref, "monc_adv_step_async")):
                ri = gc.interior(cfg, ref.numpy()).astype(np.float64)
                assert np.abs(gi - ri).max() <= gc.TOL[dtype] * scale, (n, call, nm)
                assert np.array_equal(gi, ri), (n, call, nm)
    L.close()


def test_step_noalloc_rejects_what_does_not_fit_and_bad_arguments():
    # BASELINE config 1 (256 x 256 x 128 fp64): 6 x 69 MB against the 16 MiB scratch
    cfg = synth.CONFIGS[1]
    g = synth.grid(cfg.nz)
    L = binding.MoncAdv(cfg.nx, cfg.ny, cfg.nz, cfg.halo, synth.DX, synth.DY, g["dz"], g["dzn"], g["rho"], g["rhon"])
    t = [torch.zeros(L.shape, dtype=torch.float64).pin_memory() for _ in range(6)]
    n0 = L.launch_count()
    with pytest.raises(binding.MoncAdvError) as e:
        L.step_noalloc(*t)
    assert e.value.code == binding.EINVAL and "MONC_ADV_NOALLOC_MAX_BYTES" in str(e.value)
    assert L.launch_count() == n0
    L.close()
    # the largest cube that fits / the first that does not (6 fields, 256-byte slots)
    assert 6 * (-(-(68 * 68 * 64 * 8) // 256) * 256) <= binding.NOALLOC_MAX_BYTES < 6 * 72 * 72 * 68 * 8
    cfg = gc.custom_cfg(12, 10, 16, cid=902)
    P, L = gc.make_pair(cfg)
    lib = binding.load()
    good = [torch.zeros(L.shape, dtype=torch.float64).pin_memory() for _ in range(6)]
    ptr = [C.c_void_p(x.data_ptr()) for x in good]
    pageable = torch.zeros(L.shape, dtype=torch.float64)
    raw = lambda *a: lib.monc_adv_step_noalloc(L._h, *a, None)
    assert raw(*ptr) == binding.OK
    torch.cuda.synchronize()
    assert raw(None, *ptr[1:]) == binding.EINVAL                                    # NULL
    assert raw(C.c_void_p(pageable.data_ptr()), *ptr[1:]) == binding.EINVAL         # pageable host memory
    assert raw(ptr[0], ptr[1], ptr[2], ptr[0], ptr[4], ptr[5]) == binding.EINVAL    # output overlaps an input
    assert raw(ptr[0], ptr[1], ptr[2], ptr[3], ptr[3], ptr[5]) == binding.EINVAL    # outputs overlap
    L.set_accumulate(True)
    assert raw(*ptr) == binding.EINVAL                                              # overwrite mode only
    L.set_accumulate(False)
    assert raw(*ptr) == binding.OK
    torch.cuda.synchronize()
    L.close()


def test_step_noalloc_shares_one_scratch_between_handles():
    # two handles of different shapes, calls alternating on one stream: every call overwrites what it reads
    a = gc.custom_cfg(24, 20, 64, cid=903)
    b = gc.custom_cfg(9, 30, 32, dtype="f32", cid=904)
    st = torch.cuda.Stream()
    pairs = [gc.make_pair(c) for c in (a, b)]
    data = []
    for cfg, (P, L) in zip((a, b), pairs):
        f = [synth.field(cfg, n) for n in "uvw"]
        data.append((f, [pinned(x, L) for x in f],
                     [torch.full(L.shape, gc.SENTINEL, dtype=L.torch_dtype).pin_memory() for _ in range(3)]))
    for _ in range(3):
        for (P, L), (f, hi, ho) in zip(pairs, data):
            L.step_noalloc(*hi, *ho, stream=st)
    st.synchronize()
    for cfg, (P, L), (f, hi, ho) in zip((a, b), pairs, data):
        for o, w_, n in zip(ho, P.momentum(*f), ("su", "sv", "sw")):
            gc.check(cfg, o, w_, n)
            gc.check_halo_untouched(cfg, o, n)
        L.close()
