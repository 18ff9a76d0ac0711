"""Seeded synthetic inputs for BASELINE.json's configs.

This module serves BOTH the CPU oracle (via tests/bench) and the CUDA library.
It holds none of the advection arithmetic: only the grid profiles the caller
hands to `monc_adv_create`, a counter-based random generator, the value
distributions of the configs and the periodic halo fill (SURVEY.md 8(c).4 item
10: the caller fills halos).  numpy only; never imports the CUDA binding or
the oracle.

The paper measures on MONC's "tank" bubble case, which
needs the full model and is not available; these fields stand in for it
(DESIGN.md "Input recipe").
"""
from __future__ import annotations

import dataclasses
from concurrent.futures import ThreadPoolExecutor
import os

import numpy as np

BASE_SEED = 200912850
DX = DY = 50.0
FIELD_ID = {"u": 0, "v": 1, "w": 2, "theta": 3}  # q_m -> 3 + m

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)


@dataclasses.dataclass(frozen=True)
class Config:
    """One row of BASELINE.json `configs` (sizes per SURVEY.md 8 table)."""
    cid: int
    nx: int
    ny: int
    nz: int
    halo: int = 2
    nq: int = 0
    dtype: str = "f64"
    seed_cid: int | None = None  # config 3 reuses config 2's fields
    steps: int = 1

    @property
    def seed(self) -> int:
        return BASE_SEED + (self.cid if self.seed_cid is None else self.seed_cid)

    @property
    def shape(self):
        return (self.nx + 2 * self.halo, self.ny + 2 * self.halo, self.nz)

    @property
    def points(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def elems(self) -> int:
        s = self.shape
        return s[0] * s[1] * s[2]


CONFIGS = {
    0: Config(0, 16, 16, 32),
    1: Config(1, 256, 256, 128),
    2: Config(2, 512, 512, 256, nq=10),
    3: Config(3, 512, 512, 256, nq=10, dtype="f32", seed_cid=2),
    4: Config(4, 1024, 1024, 160, nq=4, steps=20),
}


# ----------------------------------------------------------------------------
# grid profiles (SURVEY.md 8(d) "Grid")
# ----------------------------------------------------------------------------
def grid(nz: int) -> dict:
    """Stretched vertical grid and anelastic density profiles, index K-1.

    z_1 = 0, dz_K = 20 r^(K-2) for K = 2..nz with r = 3^(1/(nz-2)) (20 m -> 60 m),
    zn_K = (z_K + z_{K-1})/2, zn_1 = -zn_2, dzn_K = zn_K - zn_{K-1},
    dz_1 = dz_2, dzn_1 = dzn_2, rho = 1.2 exp(-z/8000), rhon = 1.2 exp(-zn/8000).
    """
    assert nz >= 3
    r = 3.0 ** (1.0 / (nz - 2))
    dz = np.empty(nz)
    dz[1:] = 20.0 * r ** np.arange(nz - 1)
    dz[0] = dz[1]
    z = np.zeros(nz)
    z[1:] = np.cumsum(dz[1:])
    zn = np.empty(nz)
    zn[1:] = 0.5 * (z[1:] + z[:-1])
    zn[0] = -zn[1]
    dzn = np.empty(nz)
    dzn[1:] = zn[1:] - zn[:-1]
    dzn[0] = dzn[1]
    rho = 1.2 * np.exp(-z / 8000.0)
    rhon = 1.2 * np.exp(-zn / 8000.0)
    return dict(z=z, zn=zn, dz=dz, dzn=dzn, rho=rho, rhon=rhon)


# ----------------------------------------------------------------------------
# counter-based generator (splitmix64 finaliser), keyed by
# (seed, stream, field_id, interior linear index, draw)
# ----------------------------------------------------------------------------
def _mix(x: np.ndarray) -> np.ndarray:
    x = (x ^ (x >> np.uint64(30))) * _C1
    x = (x ^ (x >> np.uint64(27))) * _C2
    return x ^ (x >> np.uint64(31))


def _key(seed: int, stream: int, field_id: int) -> np.uint64:
    with np.errstate(over="ignore"):
        k = _mix(np.uint64(seed) * _GOLD + np.uint64(1))
        k = _mix(k ^ (np.uint64(stream) * _C1 + np.uint64(field_id) * _C2 + _GOLD))
    return k


def _uniform_range(key: np.uint64, lo: int, hi: int, draw: int) -> np.ndarray:
    """53-bit uniforms in [0,1) for interior linear indices lo..hi-1."""
    with np.errstate(over="ignore"):
        idx = np.arange(lo, hi, dtype=np.uint64)
        z = _mix(key + (idx * np.uint64(2) + np.uint64(draw) + np.uint64(1)) * _GOLD)
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def _chunks(n: int, chunk: int = 1 << 21):
    return [(lo, min(n, lo + chunk)) for lo in range(0, n, chunk)]


def _parallel_fill(n: int, fn) -> np.ndarray:
    out = np.empty(n)
    parts = _chunks(n)

    def work(p):
        out[p[0]:p[1]] = fn(p[0], p[1])

    if len(parts) == 1:
        work(parts[0])
    else:
        with ThreadPoolExecutor(max_workers=min(len(parts), os.cpu_count() or 1, 32)) as ex:
            list(ex.map(work, parts))
    return out


def uniform01(seed: int, stream: int, field_id: int, n: int) -> np.ndarray:
    key = _key(seed, stream, field_id)
    return _parallel_fill(n, lambda lo, hi: _uniform_range(key, lo, hi, 0))


def normal01(seed: int, stream: int, field_id: int, n: int) -> np.ndarray:
    """Standard normals by Box-Muller from two keyed uniforms per index."""
    key = _key(seed, stream, field_id)

    def fn(lo, hi):
        u1 = _uniform_range(key, lo, hi, 0)
        u2 = _uniform_range(key, lo, hi, 1)
        return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)

    return _parallel_fill(n, fn)


# ----------------------------------------------------------------------------
# fields
# ----------------------------------------------------------------------------
def fill_halo_periodic(f: np.ndarray, h: int) -> np.ndarray:
    """Periodic wrap in x and y, all levels. In place."""
    nx = f.shape[0] - 2 * h
    ny = f.shape[1] - 2 * h
    f[:h] = f[nx:nx + h]
    f[nx + h:] = f[h:2 * h]
    f[:, :h] = f[:, ny:ny + h]
    f[:, ny + h:] = f[:, h:2 * h]
    return f


def embed(interior: np.ndarray, h: int) -> np.ndarray:
    """[nx,ny,nz] interior -> [nx+2h, ny+2h, nz] with periodic halos."""
    nx, ny, nz = interior.shape
    f = np.empty((nx + 2 * h, ny + 2 * h, nz))
    f[h:h + nx, h:h + ny] = interior
    return fill_halo_periodic(f, h)


def field_names(cfg: Config):
    """Scalar field names of a config: theta, q1, q2, ... (SURVEY.md 8(d) 'Fields')."""
    return ["theta"] + [f"q{m}" for m in range(1, cfg.nq)] if cfg.nq > 0 else []


def _fid(name: str) -> int:
    return FIELD_ID[name] if name in FIELD_ID else 3 + int(name[1:])


def interior_field(cfg: Config, name: str) -> np.ndarray:
    """u, v ~ U(-5,5); w ~ U(-1,1) with w = 0 at K = 1 and K = nz;
    theta ~ N(0, sd 0.5); q_m ~ |N(0, sd 1e-3)|."""
    n = cfg.points
    shp = (cfg.nx, cfg.ny, cfg.nz)
    fid = _fid(name)
    if name in ("u", "v"):
        f = (uniform01(cfg.seed, 0, fid, n) * 10.0 - 5.0).reshape(shp)
    elif name == "w":
        f = (uniform01(cfg.seed, 0, fid, n) * 2.0 - 1.0).reshape(shp)
        f[:, :, 0] = 0.0
        f[:, :, -1] = 0.0
    elif name == "theta":
        f = (0.5 * normal01(cfg.seed, 0, fid, n)).reshape(shp)
    else:
        f = np.abs(1e-3 * normal01(cfg.seed, 0, fid, n)).reshape(shp)
    return f


def field(cfg: Config, name: str) -> np.ndarray:
    """Full array with periodic halos, float64, C order [NXH, NYH, nz]."""
    return embed(interior_field(cfg, name), cfg.halo)


def perturb(cfg: Config, name: str, f: np.ndarray, step: int, sd: float = 0.01) -> np.ndarray:
    """Config 4 time loop: f += sd * N(0,1) on interior points, keyed by
    (seed, 1000 + step, field, index); re-zero w at K = 1, nz; re-fill halos.
    In place on a full (halo'd) array."""
    h = cfg.halo
    n = cfg.points
    d = normal01(cfg.seed, 1000 + step, _fid(name), n).reshape(cfg.nx, cfg.ny, cfg.nz)
    inner = f[h:h + cfg.nx, h:h + cfg.ny]
    inner += sd * d
    if name == "w":
        inner[:, :, 0] = 0.0
        inner[:, :, -1] = 0.0
    return fill_halo_periodic(f, h)
