"""GPU parity: the CUDA library (through the C ABI) against the CPU oracle on
the same seeded inputs, element by element.  Run on the B200 box: -m gpu."""
import dataclasses
from fractions import Fraction

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


def run_momentum(cfg, variant="auto", xchunk=0, fields=None, form="flux", stages=0, tile_y=0):
    P, L = gc.make_pair(cfg)
    L.set_variant(variant)
    L.set_tuning(xchunk=xchunk, stages=stages, tile_y=tile_y)
    L.set_form(form)
    U, V, W = fields if fields is not None else [synth.field(cfg, n) for n in "uvw"]
    want = P.momentum(U, V, W, skew=(form == "pw_skew"), nthreads=oracle.max_threads())
    du, dv, dw = (gc.to_dev(a, L) for a in (U, V, W))
    outs = gc.fresh_out(L, 3)
    L.momentum(du, dv, dw, *outs)
    torch.cuda.synchronize()
    errs = [gc.check(cfg, o, w_, n) for o, w_, n in zip(outs, want, ("su", "sv", "sw"))]
    for o, n in zip(outs, ("su", "sv", "sw")):
        gc.check_halo_untouched(cfg, o, n)
    L.close()
    return errs


def run_scalars(cfg, nq, variant="auto", xchunk=0, group=0, form="flux", stages=0, tile_y=0, warps=0,
                split=0):
    cfgq = dataclasses.replace(cfg, nq=nq)
    P, L = gc.make_pair(cfgq)
    L.set_variant(variant)
    L.set_tuning(xchunk=xchunk, group=group, stages=stages, tile_y=tile_y, warps=warps, split=split)
    L.set_form(form)
    U, V, W = [synth.field(cfgq, n) for n in "uvw"]
    names = synth.field_names(cfgq)
    Q = [synth.field(cfgq, n) for n in names]
    du, dv, dw = (gc.to_dev(a, L) for a in (U, V, W))
    dq = [gc.to_dev(a, L) for a in Q]
    outs = gc.fresh_out(L, nq)
    L.bind_wind(du, dv, dw)
    L.scalars(dq, outs)
    torch.cuda.synchronize()
    for n, (o, q) in enumerate(zip(outs, Q)):
        want = P.scalar(U, V, W, q, skew=(form == "pw_skew"), nthreads=oracle.max_threads())
        gc.check(cfgq, o, want, f"sq[{names[n]}]")
        gc.check_halo_untouched(cfgq, o, names[n])
    L.close()


# ---------------------------------------------------------------------------
# BASELINE.json configs 0 and 1: full element-by-element comparison
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("variant", ["tma", "march", "generic"])
def test_config0_momentum_fp64(variant):
    run_momentum(synth.CONFIGS[0], variant)


@pytest.mark.parametrize("variant", ["tma", "march", "generic"])
def test_config0_scalars_fp64(variant):
    run_scalars(synth.CONFIGS[0], 4, variant)


@pytest.mark.parametrize("variant", ["auto", "tma", "march"])
def test_config1_momentum_fp64_full_size(variant):
    # "auto" is the launch configuration bench.py times (default tuning)
    errs = run_momentum(synth.CONFIGS[1], variant)
    print("config1 max rel errs", errs)


def test_config1_shape_fp32_and_scalars():
    cfg = dataclasses.replace(synth.CONFIGS[1], dtype="f32")
    run_momentum(cfg)
    run_scalars(dataclasses.replace(synth.CONFIGS[1], nx=64), 3)


# ---------------------------------------------------------------------------
# ragged / edge shapes: several tiles, partial warps, z-chunk edges, odd sizes
# ---------------------------------------------------------------------------
SHAPES = [
    (13, 7, 38, 2),    # fp64 vectors ok; fp32 ragged (38 % 4 != 0) and ny + 2h odd: generic kernels
    (9, 11, 37, 2),    # odd nz and ny + 2h odd: generic kernels (the ragged-nz TMA path: RAGGED_NZ below)
    (10, 6, 70, 2),    # two z-chunks per column, ragged second chunk
    (6, 10, 160, 2),   # config 4's nz: 2.5 warps per column (fp64)
    (5, 9, 256, 1),    # halo 1, 4 z-chunks per column (fp64), 2 (fp32)
    (7, 5, 64, 3),     # halo 3, exactly one full warp per column (fp64)
    (3, 1, 4, 2),      # ny = 1
    (1, 3, 3, 2),      # nx = 1, minimum nz
    (33, 17, 132, 2),  # > 1 chunk in every direction
]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("shape", SHAPES)
def test_ragged_shapes(shape, dtype):
    nx, ny, nz, h = shape
    cfg = gc.custom_cfg(nx, ny, nz, halo=h, dtype=dtype, cid=200 + nz)
    run_momentum(cfg, "auto", xchunk=0)
    run_momentum(cfg, "auto", xchunk=4)   # several x-chunks: chunk seams
    vec_ok = nz % (2 if dtype == "f64" else 4) == 0
    if vec_ok:
        for variant in ("march", "tma"):
            run_momentum(cfg, variant, xchunk=0)
            run_momentum(cfg, variant, xchunk=3, stages=3, tile_y=2)
    run_scalars(cfg, 3, "auto", xchunk=5, group=2)   # ragged group (2 + 1)
    if vec_ok:
        run_scalars(cfg, 3, "march", xchunk=5, group=2)
        # TMA ring: z split over 1 or 2 warps per column per block (ragged last z
        # tile), short ring, ragged y tiles, several x chunks
        run_scalars(cfg, 3, "tma", xchunk=0, group=3)
        run_scalars(cfg, 3, "tma", xchunk=3, group=2, stages=2, tile_y=2, warps=1, split=1)
        run_scalars(cfg, 4, "tma", xchunk=4, group=3, stages=4, tile_y=3, warps=2, split=2)
        run_scalars(cfg, 7, "tma", xchunk=2, group=7, stages=3, tile_y=2, warps=1, split=3)


@pytest.mark.parametrize("variant", ["tma", "march"])
@pytest.mark.parametrize("group", [1, 2, 3, 4, 5])
def test_scalar_group_sizes(group, variant):
    cfg = gc.custom_cfg(12, 9, 70, nq=7, cid=300)
    run_scalars(cfg, 7, variant, xchunk=5, group=group)


@pytest.mark.parametrize("group,split", [(10, 2), (10, 3), (10, 4), (9, 2), (6, 3), (5, 1), (4, 4), (7, 2)])
def test_scalar_block_groups_and_splits(group, split):
    """tma_scalars: `group` scalars per block shared between `split` warps per
    column chunk, ragged last group and ragged last split."""
    cfg = gc.custom_cfg(9, 10, 72, nq=11, cid=302)
    run_scalars(cfg, 11, "tma", xchunk=4, group=group, split=split)


def test_max_scalars_and_zero():
    cfg = gc.custom_cfg(4, 4, 8, cid=301)
    P, L = gc.make_pair(cfg)
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    du, dv, dw = (gc.to_dev(a, L) for a in (U, V, W))
    L.bind_wind(du, dv, dw)
    L.scalars([], [])  # nq = 0: no-op
    cfgq = dataclasses.replace(cfg, nq=binding.MAX_SCALARS)
    names = synth.field_names(cfgq)
    Q = [synth.field(cfgq, n) for n in names]
    dq = [gc.to_dev(a, L) for a in Q]
    outs = gc.fresh_out(L, len(Q))
    L.scalars(dq, outs)
    torch.cuda.synchronize()
    for o, q in zip(outs, Q):
        gc.check(cfg, o, P.scalar(U, V, W, q), "sq")
    with pytest.raises(binding.MoncAdvError) as e:
        L.scalars(dq + [dq[0]], outs + gc.fresh_out(L, 1))
    assert e.value.code == binding.EINVAL


# ---------------------------------------------------------------------------
# P7 worked example through the library: exact in fp64 AND fp32
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("variant", ["tma", "march", "generic"])
def test_P7_exact_through_gpu(dtype, variant):
    from test_oracle_pins import p7_problem, read_golden
    P, (U, V, W, Q) = p7_problem()
    dz = np.array([1, 1, 2, 2, 4, 4], float)
    L = binding.MoncAdv(4, 4, 6, 2, 2.0, 4.0, dz, dz, np.array([1, 1, .5, .5, .25, .25]),
                        np.array([2, 1, 1, .5, .5, .25]), dtype=dtype)
    if variant == "march" and dtype == "f32":
        with pytest.raises(binding.MoncAdvError):
            L.set_variant(variant)  # nz = 6 is not a multiple of 4: no direct-load marching kernel
        return
    L.set_variant(variant)  # "tma" in fp32: nz = 6 is ragged, two columns per row of the tensor view
    # coefficient tables as the library stores them
    tz = dict(zip(("tzc1", "tzc2", "tzd1", "tzd2"), L.get_coefficients()))
    d = [gc.to_dev(a, L) for a in (U, V, W, Q)]
    outs = gc.fresh_out(L, 4)
    L.momentum(d[0], d[1], d[2], *outs[:3])
    L.scalars([d[3]], [outs[3]])
    torch.cuda.synchronize()
    res = {k: o.cpu().numpy().astype(np.float64)[2:6, 2:6] for k, o in zip(("su", "sv", "sw", "sq"), outs)}
    pos = np.arange(1, 97, dtype=float).reshape(4, 4, 6)
    n = 0
    for r in read_golden():
        if r[0] == "coef" and r[1] in tz:
            vals = [float(Fraction(x)) for x in r[2:]]
            if r[1] == "tzc2":
                vals[-1] = 0.0  # the library pins the unused lid entry to 0
            assert list(tz[r[1]]) == vals
        if r[0] == "column" and r[1] == "flux":
            vals = [float(Fraction(x)) for x in r[5:]]
            assert list(res[r[2]][int(r[3]), int(r[4])]) == vals, (r[2], r[3], r[4])
            n += 1
        if r[0] == "checksum":
            s, sa, mx, sidx = (float(Fraction(x)) for x in r[3:])
            a = res[r[2]]
            assert a.sum() == s and np.abs(a).sum() == sa and np.abs(a).max() == mx
            assert (a * pos).sum() == sidx
            n += 1
    assert n == 16
    # and every point equals the oracle bitwise (all values exactly representable)
    want = list(P.momentum(U, V, W)) + [P.scalar(U, V, W, Q)]
    for k, w_ in zip(("su", "sv", "sw", "sq"), want):
        assert np.array_equal(res[k], w_[2:6, 2:6]), k
    L.close()


# ---------------------------------------------------------------------------
# semantics: accumulate, wind binding, skew form, errors
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("variant", ["tma", "march", "generic"])
def test_accumulate_mode(variant):
    cfg = gc.custom_cfg(9, 8, 66, nq=2, cid=302)
    P, L = gc.make_pair(cfg)
    L.set_variant(variant)
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    Q = [synth.field(cfg, n) for n in synth.field_names(cfg)]
    d = [gc.to_dev(a, L) for a in (U, V, W)]
    dq = [gc.to_dev(a, L) for a in Q]
    base = [torch.randn(L.shape, device="cuda", dtype=torch.float64) for _ in range(5)]
    outs = [b.clone() for b in base]
    L.set_accumulate(True)
    L.momentum(*d, *outs[:3])
    L.scalars(dq, outs[3:])
    L.set_accumulate(False)
    plain = gc.fresh_out(L, 5)
    L.momentum(*d, *plain[:3])
    L.scalars(dq, plain[3:])
    torch.cuda.synchronize()
    h = cfg.halo
    for b, o, p_ in zip(base, outs, plain):
        sl = (slice(h, h + cfg.nx), slice(h, h + cfg.ny))
        # additivity: bitwise equal to a separate add
        assert torch.equal(o[sl], b[sl] + p_[sl])
        m = torch.ones(L.shape, dtype=torch.bool, device="cuda")
        m[sl] = False
        assert torch.equal(o[m], b[m])  # halos untouched
    L.close()


def test_scalars_need_wind_and_wind_binding_equivalence():
    cfg = gc.custom_cfg(8, 8, 32, nq=2, cid=303)
    P, L = gc.make_pair(cfg)
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    Q = [synth.field(cfg, n) for n in synth.field_names(cfg)]
    d = [gc.to_dev(a, L) for a in (U, V, W)]
    dq = [gc.to_dev(a, L) for a in Q]
    o1, o2 = gc.fresh_out(L, 2), gc.fresh_out(L, 2)
    with pytest.raises(binding.MoncAdvError) as e:
        L.scalars(dq, o1)
    assert e.value.code == binding.ENOWIND
    L.bind_wind(*d)
    L.scalars(dq, o1)
    L.momentum(*d, *gc.fresh_out(L, 3))   # binds the same wind
    L.scalars(dq, o2)
    torch.cuda.synchronize()
    for a, b in zip(o1, o2):
        assert torch.equal(a, b)
    # aliasing is refused
    with pytest.raises(binding.MoncAdvError):
        L.momentum(d[0], d[1], d[2], d[0], o1[0], o1[1])
    L.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("variant", ["tma", "generic"])
def test_pw_skew_form(dtype, variant):
    # NEXT-1 (R4): the Piacsek-Williams skew form on the fast kernels;
    # several y tiles, z chunks and x chunks with ragged tails
    cfg = gc.custom_cfg(10, 9, 40, dtype=dtype, cid=304)
    run_momentum(cfg, variant=variant, form="pw_skew")
    run_scalars(cfg, 2, variant=variant, form="pw_skew")
    cfg = gc.custom_cfg(21, 19, 200, dtype=dtype, cid=306)
    run_momentum(cfg, variant=variant, form="pw_skew", xchunk=8)
    run_scalars(cfg, 7, variant=variant, form="pw_skew", xchunk=8)


def test_pw_skew_accumulate_and_P7_sums():
    # skew + accumulate on the TMA kernels, and the exact skew checksums of the
    # worked example (tests/golden/p7_worked_example.txt, rows "skewsum")
    from test_oracle_pins import p7_problem, read_golden
    P, (U, V, W, Q) = p7_problem()
    dz = np.array([1, 1, 2, 2, 4, 4], float)
    L = binding.MoncAdv(4, 4, 6, 2, 2.0, 4.0, dz, dz, np.array([1, 1, .5, .5, .25, .25]),
                        np.array([2, 1, 1, .5, .5, .25]), dtype="f64")
    L.set_variant("tma")
    L.set_form("pw_skew")
    d = [gc.to_dev(a, L) for a in (U, V, W, Q)]
    outs = gc.fresh_out(L, 4)
    L.momentum(d[0], d[1], d[2], *outs[:3])
    L.scalars([d[3]], [outs[3]])
    torch.cuda.synchronize()
    assert "tma_momentum" in L.describe_plan() and "tma_scalars" in L.describe_plan()
    res = {k: o.cpu().numpy()[2:6, 2:6] for k, o in zip(("su", "sv", "sw", "sq"), outs)}
    n = 0
    for r in read_golden():
        if r[0] == "skewsum":
            assert res[r[2]].sum() == float(Fraction(r[3])), r
            assert np.abs(res[r[2]]).max() == float(Fraction(r[4])), r
            n += 1
    assert n == 4
    L.set_accumulate(True)
    L.momentum(d[0], d[1], d[2], *outs[:3])
    L.scalars([d[3]], [outs[3]])
    torch.cuda.synchronize()
    for k, o in zip(("su", "sv", "sw", "sq"), outs):
        assert np.array_equal(o.cpu().numpy()[2:6, 2:6], 2.0 * res[k]), k
    L.close()


def test_translation_invariance_bitwise_on_gpu():
    # P10 through the library: no dependence on absolute position or block seams
    cfg = gc.custom_cfg(16, 12, 64, cid=305)
    P, L = gc.make_pair(cfg)
    L.set_tuning(xchunk=5)
    fs = [synth.interior_field(cfg, n) for n in "uvw"]
    res = []
    for shift in ((0, 0), (3, 5)):
        F = [synth.embed(np.roll(a, shift, axis=(0, 1)), cfg.halo) for a in fs]
        d = [gc.to_dev(a, L) for a in F]
        outs = gc.fresh_out(L, 3)
        L.momentum(*d, *outs)
        torch.cuda.synchronize()
        res.append([gc.interior(cfg, o.cpu().numpy()) for o in outs])
    for a, b in zip(*res):
        assert np.array_equal(np.roll(a, (3, 5), axis=(0, 1)), b)
    L.close()


def test_user_supplied_tz_arrays_and_stream():
    cfg = gc.custom_cfg(8, 8, 32, cid=306)
    g = synth.grid(cfg.nz)
    P = oracle.Problem(cfg.nx, cfg.ny, cfg.nz, cfg.halo, 50.0, 50.0, g["dz"], g["dzn"], g["rho"], g["rhon"])
    L = binding.MoncAdv(cfg.nx, cfg.ny, cfg.nz, cfg.halo, 50.0, 50.0,
                        tzc1=P.tzc1, tzc2=P.tzc2, tzd1=P.tzd1, tzd2=P.tzd2)
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    d = [gc.to_dev(a, L) for a in (U, V, W)]
    outs = gc.fresh_out(L, 3)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        L.momentum(*d, *outs, stream=st)
    st.synchronize()
    for o, w_, n in zip(outs, P.momentum(U, V, W), ("su", "sv", "sw")):
        gc.check(cfg, o, w_, n)
    assert L.launch_count() == 1
    L.close()


# ---------------------------------------------------------------------------
# ragged nz (a column is not a whole number of 16-byte vectors) on the TMA kernels:
# the tensor-map view groups 2 or 4 columns per row, every row of a tile is its own
# copy, stores of unaligned / partial vectors go element by element
# ---------------------------------------------------------------------------
RAGGED_NZ = [
    (13, 8, 37, 2, "f64"),    # one z tile, partial last vector, columns alternate between aligned and not
    (9, 14, 129, 2, "f64"),   # three z tiles, the last holds one level
    (10, 6, 255, 1, "f64"),   # halo 1, four z tiles
    (7, 10, 3, 2, "f64"),     # minimum nz
    (13, 8, 38, 2, "f32"),    # nz % 4 = 2: two columns per row
    (9, 8, 37, 2, "f32"),     # odd nz: four columns per row
    (6, 12, 129, 2, "f32"),   # two z tiles, the last holds one level
    (10, 6, 254, 1, "f32"),   # halo 1
    (5, 4, 7, 2, "f32"),
]


@pytest.mark.parametrize("shape", RAGGED_NZ, ids=lambda s: "x".join(map(str, s)))
def test_ragged_nz_on_the_tma_kernels(shape):
    nx, ny, nz, h, dtype = shape
    cfg = gc.custom_cfg(nx, ny, nz, halo=h, nq=4, dtype=dtype, cid=700 + nz)
    names = ["u", "v", "w"] + synth.field_names(cfg)
    H = [synth.field(cfg, n) for n in names]
    for form in ("flux", "pw_skew"):
        skew = form == "pw_skew"
        P, L = gc.make_pair(cfg)
        L.set_variant("tma")  # no silent fall-back to the generic kernels
        L.set_form(form)
        D = [gc.to_dev(a, L) for a in H]
        want = list(P.momentum(H[0], H[1], H[2], skew=skew)) + [P.scalar(H[0], H[1], H[2], q, skew=skew) for q in H[3:]]
        for tuning in (dict(), dict(xchunk=4, tile_y=3, stages=3), dict(xchunk=3, tile_y=2, split=2)):
            L.set_tuning(**tuning)
            # momentum alone: the momentum role of the tensor-map kernel without scalar warps
            outs = gc.fresh_out(L, 7)
            L.momentum(D[0], D[1], D[2], *outs[:3])
            assert "momentum role only" in L.describe_plan() and "colgroup=1 " not in L.describe_plan()
            # scalars alone
            L.scalars(D[3:], outs[3:])
            assert "tma_scalars" in L.describe_plan()
            torch.cuda.synchronize()
            for o, w_, n in zip(outs, want, ["su", "sv", "sw"] + names[3:]):
                gc.check(cfg, o, w_, n)
                gc.check_halo_untouched(cfg, o, n)
            # the whole step in one launch, then once more accumulating
            outs2 = gc.fresh_out(L, 7)
            L.tendencies(D[0], D[1], D[2], outs2[0], outs2[1], outs2[2], D[3:], outs2[3:])
            assert "tma_fused(momentum+scalars)" in L.describe_plan()
            torch.cuda.synchronize()
            for a, b in zip(outs, outs2):
                assert torch.equal(a, b)  # same arithmetic in both launches
            L.set_accumulate(True)
            L.tendencies(D[0], D[1], D[2], outs2[0], outs2[1], outs2[2], D[3:], outs2[3:])
            L.momentum(D[0], D[1], D[2], *outs2[:3])
            L.set_accumulate(False)
            torch.cuda.synchronize()
            for o, w_, n, m in zip(outs2, want, ["su", "sv", "sw"] + names[3:], (3, 3, 3, 2, 2, 2, 2)):
                gc.check(cfg, o, m * w_, n + " accumulated")
                gc.check_halo_untouched(cfg, o, n)
        L.close()


@pytest.mark.parametrize("cluster", [2, 3, 4, 8])
def test_cluster_launches_are_a_placement_hint_only(cluster):
    # thread-block clusters of y-neighbour tiles (monc_adv_set_cluster): the grid is padded to whole
    # clusters, the extra blocks exit; results bitwise those of the plain launch
    for nz, tuning in ((200, dict(tile_y=2, xchunk=5)), (200, dict()), (129, dict(tile_y=3, xchunk=4))):
        cfg = gc.custom_cfg(11, 18, nz, nq=4, cid=740)  # ny + 2 halo even: the ragged nz = 129 takes the TMA kernels too
        P, L = gc.make_pair(cfg)
        L.set_tuning(**tuning)
        names = ["u", "v", "w"] + synth.field_names(cfg)
        D = [gc.to_dev(synth.field(cfg, n), L) for n in names]
        res = []
        for cl in (1, cluster):
            L.set_cluster(cl)
            o = gc.fresh_out(L, 7)
            L.momentum(D[0], D[1], D[2], *o[:3])
            # (the size is capped at the y-tile count; the text after ";" is the last scalars launch)
            assert ("cluster=1 " in L.describe_plan().split(";")[0]) == (cl == 1), L.describe_plan()
            L.scalars(D[3:], o[3:])
            o2 = gc.fresh_out(L, 7)
            L.tendencies(D[0], D[1], D[2], o2[0], o2[1], o2[2], D[3:], o2[3:])
            assert ("cluster=1 " in L.describe_plan()) == (cl == 1), L.describe_plan()
            torch.cuda.synchronize()
            res.append(o + o2)
        for a, b in zip(*res):
            assert torch.equal(a, b)
        want = P.momentum(*[synth.field(cfg, n) for n in "uvw"])
        for o, w_, n in zip(res[1][:3], want, ("su", "sv", "sw")):
            gc.check(cfg, o, w_, n)
            gc.check_halo_untouched(cfg, o, n)
        L.close()


@pytest.mark.parametrize("dtype,nz", [("f64", 1100), ("f32", 2200), ("f64", 1101)])
def test_tall_columns_take_the_tensor_map_kernel(dtype, nz):
    # more than 16 warps per column: tma_momentum (whole columns per block) does not fit, the z-tiled
    # tensor-map kernel does, momentum alone included
    cfg = gc.custom_cfg(5, 6, nz, nq=2, dtype=dtype, cid=730)
    P, L = gc.make_pair(cfg)
    L.set_variant("tma")
    names = ["u", "v", "w"] + synth.field_names(cfg)
    H = [synth.field(cfg, n) for n in names]
    D = [gc.to_dev(a, L) for a in H]
    want = list(P.momentum(H[0], H[1], H[2])) + [P.scalar(H[0], H[1], H[2], q) for q in H[3:]]
    outs = gc.fresh_out(L, 5)
    L.momentum(D[0], D[1], D[2], *outs[:3])
    assert "momentum role only" in L.describe_plan()
    L.scalars(D[3:], outs[3:])
    outs2 = gc.fresh_out(L, 5)
    L.tendencies(D[0], D[1], D[2], outs2[0], outs2[1], outs2[2], D[3:], outs2[3:])
    assert "tma_fused(momentum+scalars)" in L.describe_plan()
    torch.cuda.synchronize()
    for o, o2, w_, n in zip(outs, outs2, want, ["su", "sv", "sw"] + names[3:]):
        gc.check(cfg, o, w_, n)
        gc.check_halo_untouched(cfg, o, n)
        assert torch.equal(o, o2)
    L.close()


def test_ragged_nz_without_a_column_group_view_runs_the_generic_kernels():
    # odd nz in fp64 needs ny + 2 halo even; otherwise the generic kernels run and the TMA variant is refused
    cfg = gc.custom_cfg(9, 11, 37, dtype="f64", cid=720)
    P, L = gc.make_pair(cfg)
    with pytest.raises(binding.MoncAdvError) as e:
        L.set_variant("tma")
    assert e.value.code == binding.EINVAL
    U, V, W = [synth.field(cfg, n) for n in "uvw"]
    outs = gc.fresh_out(L, 3)
    L.momentum(*[gc.to_dev(a, L) for a in (U, V, W)], *outs)
    assert "generic_momentum" in L.describe_plan()
    for o, w_, n in zip(outs, P.momentum(U, V, W), ("su", "sv", "sw")):
        gc.check(cfg, o, w_, n)
    L.close()


# ---------------------------------------------------------------------------
# guard bands: nothing outside the caller's arrays is read into a result or written
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("variant", ["tma", "march", "generic", "tma-ragged-nz"])
@pytest.mark.parametrize("form", ["flux", "pw_skew"])
def test_guard_bands(dtype, variant, form):
    """Every field sits inside a larger allocation whose guard regions hold NaN
    (inputs) or a sentinel (outputs), with the tightest halo (1).  A read past
    an array that reaches a result shows up as NaN (0 * NaN included); a write
    past an output array changes its guard."""
    if variant == "march" and form == "pw_skew":
        pytest.skip("march kernels are flux-form only")
    nz = 72
    if variant == "tma-ragged-nz":  # the last column's top vector and the first column's z halo straddle the array ends
        variant, nz = "tma", 71
    cfg = gc.custom_cfg(9, 10, nz, halo=1, nq=3, dtype=dtype, cid=307)
    P, L = gc.make_pair(cfg)
    L.set_variant(variant)
    L.set_form(form)
    L.set_tuning(xchunk=4)
    names = ["u", "v", "w"] + synth.field_names(cfg)
    H = [synth.field(cfg, n) for n in names]
    n = int(np.prod(L.shape))
    G = 4096  # guard elements on each side (keeps 16-byte alignment)

    def embed(a, fill):
        buf = torch.full((n + 2 * G,), fill, device="cuda", dtype=L.torch_dtype)
        view = buf[G:G + n].view(L.shape)
        if a is not None:
            view.copy_(torch.from_numpy(a).to(L.torch_dtype))
        return buf, view

    ins = [embed(a, float("nan")) for a in H]
    outs = [embed(None, gc.SENTINEL) for _ in range(3 + cfg.nq)]
    L.momentum(ins[0][1], ins[1][1], ins[2][1], outs[0][1], outs[1][1], outs[2][1])
    L.scalars([b[1] for b in ins[3:]], [b[1] for b in outs[3:]])
    torch.cuda.synchronize()
    skew = form == "pw_skew"
    want = list(P.momentum(H[0], H[1], H[2], skew=skew)) + [P.scalar(H[0], H[1], H[2], q, skew=skew) for q in H[3:]]
    for (buf, view), w_, nm in zip(outs, want, ["su", "sv", "sw"] + names[3:]):
        gc.check(cfg, view, w_, nm)
        gc.check_halo_untouched(cfg, view, nm)
        g = buf.cpu().numpy()
        assert np.all(g[:G] == gc.SENTINEL) and np.all(g[G + n:] == gc.SENTINEL), f"{nm}: guard written"
    L.close()


# ---------------------------------------------------------------------------
# monc_adv_tendencies: the whole step in one call (fused launch where it fits)
# ---------------------------------------------------------------------------
def run_tendencies(cfg, nq, form="flux", fuse=True, tuning=None, accumulate=False):
    cfgq = dataclasses.replace(cfg, nq=nq)
    P, L = gc.make_pair(cfgq)
    L.set_form(form)
    L.set_fuse(fuse)
    if tuning:
        L.set_tuning(**tuning)
    U, V, W = [synth.field(cfgq, n) for n in "uvw"]
    names = synth.field_names(cfgq)
    Q = [synth.field(cfgq, n) for n in names]
    du, dv, dw = (gc.to_dev(a, L) for a in (U, V, W))
    dq = [gc.to_dev(a, L) for a in Q]
    outs = gc.fresh_out(L, 3 + nq)
    skew = form == "pw_skew"
    want = list(P.momentum(U, V, W, skew=skew)) + [P.scalar(U, V, W, q, skew=skew) for q in Q]
    reps = 1
    if accumulate:
        for o in outs:
            h = cfgq.halo
            o[h:h + cfgq.nx, h:h + cfgq.ny] = 0.0
        L.set_accumulate(True)
        reps = 2
    for _ in range(reps):
        L.tendencies(du, dv, dw, outs[0], outs[1], outs[2], dq, outs[3:])
    torch.cuda.synchronize()
    plan = L.describe_plan()
    for o, w_, n in zip(outs, want, ["su", "sv", "sw"] + names):
        gc.check(cfgq, o, reps * w_, n)
        gc.check_halo_untouched(cfgq, o, n)
    L.close()
    return plan


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("form", ["flux", "pw_skew"])
def test_tendencies_fused(dtype, form):
    # several y tiles, z tiles and x chunks with ragged tails; every scalar count 1..10
    cfg = gc.custom_cfg(21, 19, 200, dtype=dtype, cid=310)
    for nq, tuning in ((1, None), (3, dict(xchunk=8)), (4, dict(xchunk=5, tile_y=2, stages=3)),
                       (7, dict(xchunk=8, warps=2)), (10, dict(xchunk=6))):
        plan = run_tendencies(cfg, nq, form=form, tuning=tuning)
        assert "tma_fused" in plan, plan
    # nothing to fuse: the momentum launch alone; fusing switched off: two launches, same results
    assert "tma_fused" not in run_tendencies(cfg, 0, form=form)
    assert "tma_fused" not in run_tendencies(cfg, 4, form=form, fuse=False)
    # more scalars than the fused launch's one group of 10: the rest in a scalars launch of their own
    plan = run_tendencies(cfg, 13, form=form)
    assert "tma_fused(momentum+scalars) group=10" in plan and "; tma_scalars group=3" in plan, plan


def test_tendencies_accumulate_and_shapes():
    run_tendencies(gc.custom_cfg(9, 5, 64, cid=311), 5, accumulate=True)
    run_tendencies(gc.custom_cfg(3, 1, 4, cid=312), 2)            # ny = 1, one vector per column
    run_tendencies(gc.custom_cfg(5, 9, 37, cid=313), 2)           # odd nz: generic kernels, two launches
    run_tendencies(gc.custom_cfg(6, 10, 160, halo=1, cid=314), 4)  # halo 1, 2.5 warps per column


def test_tendencies_errors():
    cfg = gc.custom_cfg(8, 8, 16, nq=2, cid=315)
    P, L = gc.make_pair(cfg)
    d = [torch.zeros(L.shape, device="cuda", dtype=L.torch_dtype) for _ in range(5)]
    o = gc.fresh_out(L, 5)
    with pytest.raises(binding.MoncAdvError):  # output aliases an input
        L.tendencies(d[0], d[1], d[2], o[0], o[1], o[2], d[3:], [o[3], d[0]])
    with pytest.raises(binding.MoncAdvError):  # outputs not distinct
        L.tendencies(d[0], d[1], d[2], o[0], o[1], o[2], d[3:], [o[3], o[0]])
    L.tendencies(d[0], d[1], d[2], o[0], o[1], o[2], d[3:], o[3:])
    L.scalars(d[3:], o[3:])  # the wind is bound by tendencies
    torch.cuda.synchronize()
    L.close()


# ---------------------------------------------------------------------------
# the paper's work-scaling experiment: the flux
# arithmetic evaluated n times on the same bytes gives the result of n = 1, bitwise
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_work_scale_is_the_identity_bitwise(dtype):
    cfg = gc.custom_cfg(19, 13, 136, nq=6, dtype=dtype, cid=320)
    P, L = gc.make_pair(cfg)
    names = ["u", "v", "w"] + synth.field_names(cfg)
    H = [synth.field(cfg, n) for n in names]
    d = [gc.to_dev(a, L) for a in H]
    res = {}
    for n in (1, 3, 16):
        L.set_work_scale(n)
        two, fused = gc.fresh_out(L, len(names)), gc.fresh_out(L, len(names))
        L.momentum(d[0], d[1], d[2], two[0], two[1], two[2])
        L.scalars(d[3:], two[3:])
        L.tendencies(d[0], d[1], d[2], fused[0], fused[1], fused[2], d[3:], fused[3:])
        torch.cuda.synchronize()
        assert "tma_fused" in L.describe_plan()
        res[n] = (two, fused)
    want = list(P.momentum(H[0], H[1], H[2])) + [P.scalar(H[0], H[1], H[2], q) for q in H[3:]]
    for o, w_, nm in zip(res[16][1], want, names):
        gc.check(cfg, o, w_, nm)
        gc.check_halo_untouched(cfg, o, nm)
    for n in (3, 16):
        for a, b in zip(res[1][0] + res[1][1], res[n][0] + res[n][1]):
            assert torch.equal(a, b), f"work scale {n} changed a result"
    # the knob is for the flux form, overwrite mode, TMA kernels only
    for bad in (lambda: L.set_form("pw_skew"), lambda: L.set_accumulate(True), lambda: L.set_variant("march"),
                lambda: L.set_work_scale(0), lambda: L.set_work_scale(65)):
        with pytest.raises(binding.MoncAdvError) as e:
            bad()
        assert e.value.code == binding.EINVAL
    L.set_work_scale(1)
    L.set_form("pw_skew")
    with pytest.raises(binding.MoncAdvError):
        L.set_work_scale(2)
    L.close()
    # a shape the TMA kernels do not take (odd nz): the compute call refuses while n > 1
    cfg2 = gc.custom_cfg(5, 4, 9, dtype=dtype, cid=321)
    P2, L2 = gc.make_pair(cfg2)
    L2.set_work_scale(4)
    z = [torch.zeros(L2.shape, device="cuda", dtype=L2.torch_dtype) for _ in range(6)]
    with pytest.raises(binding.MoncAdvError) as e:
        L2.momentum(*z)
    assert e.value.code == binding.EINVAL
    L2.close()
