"""Shared helpers of the GPU parity tests: build the same problem for the CPU
oracle and for the CUDA library from the same seeded inputs, and compare."""
import dataclasses

import numpy as np
import torch

import oracle
from paper_2009_12850_b200 import binding, synth

# BASELINE.json north_star: fp64 <= 1e-12, fp32 <= 2e-5, relative to the
# field's max |tendency| (taken over the oracle's interior values)
TOL = {"f64": 1e-12, "f32": 2e-5}


def custom_cfg(nx, ny, nz, halo=2, nq=0, dtype="f64", cid=100):
    return synth.Config(cid, nx, ny, nz, halo=halo, nq=nq, dtype=dtype)


def make_pair(cfg, dx=synth.DX, dy=synth.DY):
    g = synth.grid(cfg.nz)
    P = oracle.Problem(cfg.nx, cfg.ny, cfg.nz, cfg.halo, dx, dy, g["dz"], g["dzn"], g["rho"], g["rhon"])
    L = binding.MoncAdv(cfg.nx, cfg.ny, cfg.nz, cfg.halo, dx, dy, g["dz"], g["dzn"], g["rho"],
                        g["rhon"], dtype=cfg.dtype)
    return P, L


def to_dev(a, L):
    return torch.from_numpy(a).to(device="cuda", dtype=L.torch_dtype).contiguous()


def interior(cfg, a):
    h = cfg.halo
    return a[h:h + cfg.nx, h:h + cfg.ny]


def check(cfg, got, want, name, tol=None):
    """got: torch tensor (device or host) or ndarray, full array; want: oracle full array."""
    if isinstance(got, torch.Tensor):
        got = got.detach().cpu().numpy()
    gi = interior(cfg, got).astype(np.float64)
    wi = interior(cfg, want)
    scale = np.max(np.abs(wi))
    err = np.max(np.abs(gi - wi)) / max(scale, 1e-300)
    tol = TOL[cfg.dtype] if tol is None else tol
    assert np.all(np.isfinite(gi)), f"{name}: non-finite output"
    assert err <= tol, f"{name}: max rel err {err:.3e} > {tol:.1e} (scale {scale:.3e})"
    return err


SENTINEL = -777.25


def fresh_out(L, n=1):
    return [torch.full(L.shape, SENTINEL, device="cuda", dtype=L.torch_dtype) for _ in range(n)]


def check_halo_untouched(cfg, t, name):
    a = t.detach().cpu().numpy()
    h = cfg.halo
    m = np.ones(a.shape, bool)
    m[h:h + cfg.nx, h:h + cfg.ny] = False
    assert np.all(a[m] == SENTINEL), f"{name}: output halo was written"


def sample_points(cfg, n, rng):
    """Random interior points plus every structural edge: k = 0, 1, nz-2, nz-1,
    warp/vector boundaries in z, first/last columns and planes."""
    h = cfg.halo
    ii = rng.integers(h, h + cfg.nx, n)
    jj = rng.integers(h, h + cfg.ny, n)
    kk = rng.integers(0, cfg.nz, n)
    ks = [0, 1, 2, cfg.nz - 2, cfg.nz - 1] + [k for b in (32, 64, 128, 192) for k in (b - 1, b, b + 1) if k < cfg.nz]
    m = n // 4
    kk[:m] = np.array(ks)[rng.integers(0, len(ks), m)]
    ii[m:2 * m] = np.array([h, h + 1, h + cfg.nx - 2, h + cfg.nx - 1])[rng.integers(0, 4, m)]
    jj[2 * m:3 * m] = np.array([h, h + 1, h + cfg.ny - 2, h + cfg.ny - 1])[rng.integers(0, 4, m)]
    return ii, jj, kk


def check_sampled(cfg, P, name, got, U, V, W, Q, ii, jj, kk, scale, tol=None):
    if isinstance(got, torch.Tensor):
        g = got[torch.from_numpy(ii).to(got.device), torch.from_numpy(jj).to(got.device),
                torch.from_numpy(kk).to(got.device)].cpu().numpy().astype(np.float64)
    else:
        g = got[ii, jj, kk].astype(np.float64)
    want = P.points(name if name in ("su", "sv", "sw") else "sq", U, V, W, Q, ii, jj, kk)
    err = np.max(np.abs(g - want)) / scale
    tol = TOL[cfg.dtype] if tol is None else tol
    assert np.all(np.isfinite(g))
    assert err <= tol, f"{name}: sampled max rel err {err:.3e} > {tol:.1e}"
    return err
