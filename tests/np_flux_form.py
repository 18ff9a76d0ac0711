"""Independent numpy restatement of the advection definition (pin P8).

Written separately from oracle/monc_adv_oracle.cpp and in a different shape:
it works on PERIODIC INTERIOR arrays [nx, ny, nz] (np.roll, no halos), in
physical quantities (dx, dz, dzn, rho, rhon -- not the tzc/tzd coefficients),
and first fills whole face-flux arrays, then differences them:

    s_phi = -(1/rho_c) [ d_x(U phibar^x) + d_y(V phibar^y) + d_z(rho W phibar^z) ]

("Equivalently, with anelastic mass-flux notation").  phibar
is the two-point arithmetic mean at the face, (U, V, W) the advecting velocity
averaged to that face, rho_c = rhon_K for u, v, q and rho_K for w.  Horizontal
terms carry no density (8(c).4 item 6); the flux through z_nz is dropped
(8(c).4 item 7).  Test infrastructure only.
"""
import numpy as np


def _xm(a):  # value at i-1
    return np.roll(a, 1, axis=0)


def _xp(a):  # value at i+1
    return np.roll(a, -1, axis=0)


def _ym(a):
    return np.roll(a, 1, axis=1)


def _yp(a):
    return np.roll(a, -1, axis=1)


def _zp(a):  # value at K+1 (last level gets garbage that callers never use)
    return np.roll(a, -1, axis=2)


def _dz_lower_upper(F_top, rho_c_thick):
    """-(F[K] - F[K-1]) / rho_c_thick for K >= 2, with F[nz] := 0; K = 1 -> 0.
    F_top[..., k] is the flux through the TOP face of level k (0-based)."""
    F = F_top.copy()
    F[:, :, -1] = 0.0
    out = np.zeros_like(F)
    out[:, :, 1:] = -(F[:, :, 1:] - F[:, :, :-1]) / rho_c_thick[1:]
    return out


def scalar(u, v, w, q, dx, dy, dz, rho, rhon):
    Fx = u * 0.5 * (q + _xp(q))          # east face of cell i
    Fy = v * 0.5 * (q + _yp(q))          # north face
    Fz = rho * w * 0.5 * (q + _zp(q))    # top face z_K
    s = -(Fx - _xm(Fx)) / dx - (Fy - _ym(Fy)) / dy + _dz_lower_upper(Fz, rhon * dz)
    s[:, :, 0] = 0.0
    return s


def momentum(u, v, w, dx, dy, dz, dzn, rho, rhon):
    nz = u.shape[2]
    # ---- u: control volume centred on x_{i+1/2}; x faces at cell centres i, i+1
    FxU_c = (0.5 * (_xm(u) + u)) ** 2                       # at centre i
    FyU = 0.5 * (v + _xp(v)) * 0.5 * (u + _yp(u))           # at (i+1/2, j+1/2)
    FzU = rho * 0.5 * (w + _xp(w)) * 0.5 * (u + _zp(u))     # at (i+1/2, z_K)
    su = (-(_xp(FxU_c) - FxU_c) / dx - (FyU - _ym(FyU)) / dy
          + _dz_lower_upper(FzU, rhon * dz))
    su[:, :, 0] = 0.0
    # ---- v
    FyV_c = (0.5 * (_ym(v) + v)) ** 2                       # at centre j
    FxV = 0.5 * (u + _yp(u)) * 0.5 * (v + _xp(v))           # at (i+1/2, j+1/2)
    FzV = rho * 0.5 * (w + _yp(w)) * 0.5 * (v + _zp(v))
    sv = (-(_yp(FyV_c) - FyV_c) / dy - (FxV - _xm(FxV)) / dx
          + _dz_lower_upper(FzV, rhon * dz))
    sv[:, :, 0] = 0.0
    # ---- w: control volume between zn_K and zn_{K+1}, thickness dzn_{K+1}, density rho_K
    FxW = 0.5 * (u + _zp(u)) * 0.5 * (w + _xp(w))           # at (i+1/2, z_K)
    FyW = 0.5 * (v + _zp(v)) * 0.5 * (w + _yp(w))
    FzW_low = np.zeros_like(w)                              # at zn_K: rhon_K ((w_{K-1}+w_K)/2)^2
    FzW_low[:, :, 1:] = rhon[1:] * (0.5 * (w[:, :, :-1] + w[:, :, 1:])) ** 2
    sw = np.zeros_like(w)
    k = slice(1, nz - 1)
    kp = slice(2, nz)
    sw[:, :, k] = (-(FxW - _xm(FxW))[:, :, k] / dx - (FyW - _ym(FyW))[:, :, k] / dy
                   - (FzW_low[:, :, kp] - FzW_low[:, :, k]) / (rho[k] * dzn[kp]))
    return su, sv, sw


def divergence(u, v, w, dx, dy, dz, rho, rhon):
    """Discrete anelastic divergence of cell (i,j,K), K >= 2:
    D = d_x u + d_y v + d_z(rho w)/(rhon dz); level K = 1 returned as 0."""
    D = (u - _xm(u)) / dx + (v - _ym(v)) / dy
    m = rho * w
    D[:, :, 1:] += (m[:, :, 1:] - m[:, :, :-1]) / (rhon * dz)[1:]
    D[:, :, 0] = 0.0
    return D


def nondivergent_wind(rng, nx, ny, nz, dx, dy, dz, rho, rhon, amp=1.0):
    """Discretely non-divergent periodic wind from three staggered stream
    functions (SURVEY.md 8(c).5 pin P2); every delta is a backward difference.
    Returns interior arrays with w = 0 at K = 1 and K = nz."""
    psi = rng.standard_normal((nx, ny, nz)) * amp * dx
    chi = rng.standard_normal((nx, ny, nz)) * amp * dz.mean()
    xi = rng.standard_normal((nx, ny, nz)) * amp * dz.mean()
    for s in (chi, xi):
        s[:, :, 0] = 0.0
        s[:, :, -1] = 0.0
    u = -(psi - _ym(psi)) / dy
    v = (psi - _xm(psi)) / dx
    w = np.zeros((nx, ny, nz))
    dk = np.zeros((nx, ny, nz))
    dk[:, :, 1:] = chi[:, :, 1:] - chi[:, :, :-1]
    v -= dk / (rhon * dz)
    w += (chi - _ym(chi)) / (rho * dy)
    dk = np.zeros((nx, ny, nz))
    dk[:, :, 1:] = xi[:, :, 1:] - xi[:, :, :-1]
    u -= dk / (rhon * dz)
    w += (xi - _xm(xi)) / (rho * dx)
    return u, v, w
