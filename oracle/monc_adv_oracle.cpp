/*
 * oracle/monc_adv_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU definition of MONC's advection source
 * terms: the computation arxiv 2009.12850 offloads to the GPU (PAPER.md:49,
 * 75, 83, 97: "advection source terms" of u, v, w, theta and the q fields by
 * the Piacsek-Williams centred scheme).  PAPER.md prints no equation; the
 * definition below is the one fixed in SURVEY.md section 8(c).2 / DESIGN.md
 * "Readings" (flux form, centred differences, Arakawa C grid, anelastic
 * reference density, stretched vertical grid) and every function cites the
 * block of 8(c).2 it writes out.
 *
 * Rules this file obeys:
 *   - fp64 only, triple loops, one output point at a time, evaluated in the
 *     order the formulas are written (each parenthesis, the products, the
 *     difference, then X + Y + Z left to right); built with
 *     -ffp-contract=off so no FMA contraction changes that order.
 *   - shares no code, header, table or constant with the CUDA path under
 *     paper_2009_12850_b200/csrc; neither imports the other.
 *   - only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 *     --impl reference legs may load it.
 *   - the optional `nthreads` argument splits the OUTER x loop over OpenMP
 *     threads; every output point is still computed by the same scalar
 *     expression, so results are bitwise independent of the thread count.
 *
 * Parity pins (tests/test_oracle_pins.py, -m "not gpu"): constant fields,
 * closed forms, first-moment and quadratic conservation, the exact 4x4x6
 * worked example (tests/golden/), an independent numpy flux-array
 * formulation, x<->y symmetry and translation invariance.  The PW "skew"
 * variant is pinned by the flux/skew identity and its own checksums.
 *
 * Layout: F[i][j][k] in C order, k (z) fastest,
 * NXH = nx + 2h, NYH = ny + 2h, linear index (i*NYH + j)*nz + k, interior
 * i in [h, h+nx), j in [h, h+ny).  Level K = k + 1 in the 1-based notation
 * of SURVEY.md 8(c).2.
 */
#include <cstddef>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct Grid {
  int nx, ny, nz, h;
  long nyh;
  double cx, cy; /* 1/(4dx), 1/(4dy): SURVEY.md 8(c).2 "Coefficients" */
  inline long at(long i, long j, long k) const { return (i * nyh + j) * (long)nz + k; }
};

inline Grid make_grid(int nx, int ny, int nz, int h, double dx, double dy) {
  return Grid{nx, ny, nz, h, (long)ny + 2 * h, 1.0 / (4.0 * dx), 1.0 / (4.0 * dy)};
}

/* One output point each.  (i, j) are array indices (halo offset included),
 * k is 0-based: K = k + 1.  `skew` selects the Piacsek-Williams advective
 * ("skew") variant of SURVEY.md 8(c).4 item 4 / 8(f) NEXT-1: the centre value
 * is dropped from every advected-quantity parenthesis; skew = 0 is the flux
 * form that BASELINE.json's north_star names. */

/* SURVEY.md 8(c).2 block "su", K = 2..nz. */
inline double su_at(const Grid &g, const double *tzc1, const double *tzc2, const double *u,
                    const double *v, const double *w, int i, int j, int k, int skew) {
  if (k == 0) return 0.0;
  const long c = g.at(i, j, k);
  const long im = g.at(i - 1, j, k), ip = g.at(i + 1, j, k);
  const long jm = g.at(i, j - 1, k), jp = g.at(i, j + 1, k);
  const long km = c - 1, kp = c + 1;
  const double uc = skew ? 0.0 : u[c];
  const double X = g.cx * ((u[im] + u[c]) * (u[im] + uc) - (u[c] + u[ip]) * (uc + u[ip]));
  const double Y = g.cy * ((v[jm] + v[g.at(i + 1, j - 1, k)]) * (u[jm] + uc) -
                           (v[c] + v[ip]) * (uc + u[jp]));
  double Z = tzc1[k] * (w[km] + w[ip - 1]) * (u[km] + uc);
  if (k < g.nz - 1) Z = Z - tzc2[k] * (w[c] + w[ip]) * (uc + u[kp]);
  return X + Y + Z;
}

/* SURVEY.md 8(c).2 block "sv", K = 2..nz. */
inline double sv_at(const Grid &g, const double *tzc1, const double *tzc2, const double *u,
                    const double *v, const double *w, int i, int j, int k, int skew) {
  if (k == 0) return 0.0;
  const long c = g.at(i, j, k);
  const long im = g.at(i - 1, j, k), ip = g.at(i + 1, j, k);
  const long jm = g.at(i, j - 1, k), jp = g.at(i, j + 1, k);
  const long km = c - 1, kp = c + 1;
  const double vc = skew ? 0.0 : v[c];
  const double Y = g.cy * ((v[jm] + v[c]) * (v[jm] + vc) - (v[c] + v[jp]) * (vc + v[jp]));
  const double X = g.cx * ((u[im] + u[g.at(i - 1, j + 1, k)]) * (v[im] + vc) -
                           (u[c] + u[jp]) * (vc + v[ip]));
  double Z = tzc1[k] * (w[km] + w[jp - 1]) * (v[km] + vc);
  if (k < g.nz - 1) Z = Z - tzc2[k] * (w[c] + w[jp]) * (vc + v[kp]);
  return Y + X + Z;
}

/* SURVEY.md 8(c).2 block "sw", K = 2..nz-1; 0 at K = 1 and K = nz. */
inline double sw_at(const Grid &g, const double *tzd1, const double *tzd2, const double *u,
                    const double *v, const double *w, int i, int j, int k, int skew) {
  if (k == 0 || k > g.nz - 2) return 0.0;
  const long c = g.at(i, j, k);
  const long im = g.at(i - 1, j, k), ip = g.at(i + 1, j, k);
  const long jm = g.at(i, j - 1, k), jp = g.at(i, j + 1, k);
  const long km = c - 1, kp = c + 1;
  const double wc = skew ? 0.0 : w[c];
  const double X = g.cx * ((u[im] + u[im + 1]) * (w[im] + wc) - (u[c] + u[kp]) * (wc + w[ip]));
  const double Y = g.cy * ((v[jm] + v[jm + 1]) * (w[jm] + wc) - (v[c] + v[kp]) * (wc + w[jp]));
  const double Z =
      tzd1[k] * (w[km] + w[c]) * (w[km] + wc) - tzd2[k] * (w[c] + w[kp]) * (wc + w[kp]);
  return X + Y + Z;
}

/* SURVEY.md 8(c).2 block "sq", K = 2..nz: scalar at cell centres, advecting
 * velocities already on the faces (hence 2cx, 2cy, 2tzc). */
inline double sq_at(const Grid &g, const double *tzc1, const double *tzc2, const double *u,
                    const double *v, const double *w, const double *q, int i, int j, int k,
                    int skew) {
  if (k == 0) return 0.0;
  const long c = g.at(i, j, k);
  const long im = g.at(i - 1, j, k), ip = g.at(i + 1, j, k);
  const long jm = g.at(i, j - 1, k), jp = g.at(i, j + 1, k);
  const long km = c - 1, kp = c + 1;
  const double qc = skew ? 0.0 : q[c];
  const double X = 2.0 * g.cx * (u[im] * (q[im] + qc) - u[c] * (qc + q[ip]));
  const double Y = 2.0 * g.cy * (v[jm] * (q[jm] + qc) - v[c] * (qc + q[jp]));
  double Z = 2.0 * tzc1[k] * w[km] * (q[km] + qc);
  if (k < g.nz - 1) Z = Z - 2.0 * tzc2[k] * w[c] * (qc + q[kp]);
  return X + Y + Z;
}

}  // namespace

extern "C" {

/* SURVEY.md 8(c).2 "Coefficients".  Inputs are indexed K-1 (length nz).
 *   tzc1_K = rho_{K-1} / (4 rhon_K dz_K)       tzc2_K = rho_K / (4 rhon_K dz_K)        K = 2..nz
 *   tzd1_K = rhon_K / (4 rho_K dzn_{K+1})      tzd2_K = rhon_{K+1} / (4 rho_K dzn_{K+1})  K = 2..nz-1
 * all other entries 0. */
void oracle_coefficients(int nz, const double *dz, const double *dzn, const double *rho,
                         const double *rhon, double *tzc1, double *tzc2, double *tzd1,
                         double *tzd2) {
  for (int k = 0; k < nz; ++k) tzc1[k] = tzc2[k] = tzd1[k] = tzd2[k] = 0.0;
  for (int k = 1; k <= nz - 1; ++k) {
    tzc1[k] = rho[k - 1] / (4.0 * rhon[k] * dz[k]);
    tzc2[k] = rho[k] / (4.0 * rhon[k] * dz[k]);
  }
  for (int k = 1; k <= nz - 2; ++k) {
    tzd1[k] = rhon[k] / (4.0 * rho[k] * dzn[k + 1]);
    tzd2[k] = rhon[k + 1] / (4.0 * rho[k] * dzn[k + 1]);
  }
}

/* Momentum tendencies over the whole interior.
 * Every interior point, all K, is overwritten (zeros at the levels 8(c).2
 * lists); output halos are not touched (8(c).4 item 9). */
void oracle_momentum(int nx, int ny, int nz, int h, double dx, double dy, const double *tzc1,
                     const double *tzc2, const double *tzd1, const double *tzd2,
                     const double *u, const double *v, const double *w, double *su, double *sv,
                     double *sw, int skew, int nthreads) {
  const Grid g = make_grid(nx, ny, nz, h, dx, dy);
  (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for num_threads(nthreads > 0 ? nthreads : 1) schedule(static)
#endif
  for (int i = h; i < h + nx; ++i)
    for (int j = h; j < h + ny; ++j)
      for (int k = 0; k < nz; ++k) {
        const long c = g.at(i, j, k);
        su[c] = su_at(g, tzc1, tzc2, u, v, w, i, j, k, skew);
        sv[c] = sv_at(g, tzc1, tzc2, u, v, w, i, j, k, skew);
        sw[c] = sw_at(g, tzd1, tzd2, u, v, w, i, j, k, skew);
      }
}

/* One scalar's tendency over the whole interior. */
void oracle_scalar(int nx, int ny, int nz, int h, double dx, double dy, const double *tzc1,
                   const double *tzc2, const double *u, const double *v, const double *w,
                   const double *q, double *sq, int skew, int nthreads) {
  const Grid g = make_grid(nx, ny, nz, h, dx, dy);
  (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for num_threads(nthreads > 0 ? nthreads : 1) schedule(static)
#endif
  for (int i = h; i < h + nx; ++i)
    for (int j = h; j < h + ny; ++j)
      for (int k = 0; k < nz; ++k)
        sq[g.at(i, j, k)] = sq_at(g, tzc1, tzc2, u, v, w, q, i, j, k, skew);
}

/* The same definition at n sampled points, for parity checks at sizes where
 * a full pass is too slow.  which: 0 = su, 1 = sv, 2 = sw, 3 = sq (q must
 * then be non-NULL).  ii/jj are array indices (halo offset included), kk is
 * 0-based. */
void oracle_points(int which, int nx, int ny, int nz, int h, double dx, double dy,
                   const double *tzc1, const double *tzc2, const double *tzd1,
                   const double *tzd2, const double *u, const double *v, const double *w,
                   const double *q, int skew, long n, const int *ii, const int *jj,
                   const int *kk, double *out) {
  const Grid g = make_grid(nx, ny, nz, h, dx, dy);
  for (long p = 0; p < n; ++p) {
    const int i = ii[p], j = jj[p], k = kk[p];
    if (which == 0) out[p] = su_at(g, tzc1, tzc2, u, v, w, i, j, k, skew);
    else if (which == 1) out[p] = sv_at(g, tzc1, tzc2, u, v, w, i, j, k, skew);
    else if (which == 2) out[p] = sw_at(g, tzd1, tzd2, u, v, w, i, j, k, skew);
    else out[p] = sq_at(g, tzc1, tzc2, u, v, w, q, i, j, k, skew);
  }
}

int oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
