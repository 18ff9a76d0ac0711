// monc_adv_kernels.cuh -- sm_100a kernels for MONC's advection source terms.
//
// Definition implemented: SURVEY.md 8(c).2 / DESIGN.md "Definition" (flux-form
// centred advection on the Arakawa C grid, z-fastest layout).  The paper
// runs "the advection kernel ... for the entirety of the field
// (each column at the same time)"; these kernels are that step, re-designed
// for B200: an HBM-bound stencil, so the design goal is algorithmic DRAM
// traffic (every input read once, every output written once) with enough
// bytes in flight, not flops.  No tensor cores: there is no dense contraction.
//
// Two families:
//   generic_*  one thread per output point, direct loads.  Always valid (any
//              nz, both forms); the fallback and the "naive" baseline.
//   march_*    the fast path.  lane <-> z (16-byte vectors, coalesced along
//              MONC's fastest axis), warp <-> (column j, 32-vector z chunk),
//              block marches a chunk of x planes.  Values that an x-neighbour
//              step needs again stay in registers (raw E-plane values and the
//              three x-face fluxes), vertical neighbours come from warp
//              shuffles, y neighbours from L1 (adjacent warps load the same
//              lines).  Every face flux is computed once per thread: the
//              nine flux differences of the momentum equations need only six
//              distinct products because the off-diagonal ones are shared
//              (FxV == FyU, FxW == FzU, FyW == FzV).  The arithmetic of one x
//              step (momentum_faces) is shared with the TMA kernels.
//
// This header shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace monc {

constexpr int kMaxScalars = 64;
constexpr int kWarpsPerBlock = 8;   // maximum / default
constexpr int kDefaultPrefetch = 0;  // planes; 0 = off

template <typename T>
struct KParams {
  int nx, ny, nz, h;
  int nyh;          // ny + 2h
  long long plane;  // nyh * nz elements
  int ia, ib;       // output x range [ia, ib), array indices
  int xc;           // x planes marched per block
  int l2hint;       // TMA kernels: L2 eviction hint of the input copies (0 none, 1 evict_last, 2 evict_first)
  int colgroup;     // tma_scalars: columns per row of the tensor view (1; 2 or 4 when nz is ragged)
  int wzc;          // warps (z chunks of 32 vectors) per column
  int units;        // ny * wzc
  int accumulate;   // 0: overwrite, 1: add into outputs
  int skew;         // generic kernels only: PW skew form
  int prefetch;     // march kernels: L2 prefetch distance in planes (0 = off)
  int work;         // TMA kernels, WS instantiations: evaluations of the flux arithmetic per point
  T zero;           // 0, as a run-time value: x + zero * r is x, but no compiler can know it
  T cx, cy;         // 1/(4dx), 1/(4dy)
  const T *tzc1, *tzc2, *tzd1, *tzd2;  // device tables, length nz padded with zeros to whole vectors + one; tzc2[nz-1] = 0
};

template <typename T>
struct ScalarPtrs {
  const T *q[kMaxScalars];
  T *sq[kMaxScalars];
};

// ---------------------------------------------------------------------------
// 16-byte vectors along z
// ---------------------------------------------------------------------------
template <typename T> struct VecOf;
template <> struct VecOf<double> { static constexpr int NK = 2; };
template <> struct VecOf<float> { static constexpr int NK = 4; };

template <typename T>
struct Vec {
  T v[VecOf<T>::NK];
};

__device__ __forceinline__ Vec<double> ld_vec(const double *p) {
  const double2 t = __ldg(reinterpret_cast<const double2 *>(p));
  Vec<double> r;
  r.v[0] = t.x; r.v[1] = t.y;
  return r;
}
__device__ __forceinline__ Vec<float> ld_vec(const float *p) {
  const float4 t = __ldg(reinterpret_cast<const float4 *>(p));
  Vec<float> r;
  r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w;
  return r;
}
__device__ __forceinline__ Vec<double> ld_vec_rw(const double *p) {
  const double2 t = *reinterpret_cast<const double2 *>(p);
  Vec<double> r;
  r.v[0] = t.x; r.v[1] = t.y;
  return r;
}
__device__ __forceinline__ Vec<float> ld_vec_rw(const float *p) {
  const float4 t = *reinterpret_cast<const float4 *>(p);
  Vec<float> r;
  r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w;
  return r;
}
// streaming (evict-first) stores: tendencies are never re-read by the kernel
__device__ __forceinline__ void st_vec(double *p, const Vec<double> &a) {
  __stcs(reinterpret_cast<double2 *>(p), make_double2(a.v[0], a.v[1]));
}
__device__ __forceinline__ void st_vec(float *p, const Vec<float> &a) {
  __stcs(reinterpret_cast<float4 *>(p), make_float4(a.v[0], a.v[1], a.v[2], a.v[3]));
}

template <typename T>
__device__ __forceinline__ Vec<T> ld_or_zero(const T *p, bool act) {
  Vec<T> r;
#pragma unroll
  for (int e = 0; e < VecOf<T>::NK; ++e) r.v[e] = T(0);
  if (act) r = ld_vec(p);
  return r;
}

constexpr unsigned kFull = 0xffffffffu;

// Work scaling: repetition r of a point's arithmetic reads x + zero * r
// (zero is a kernel parameter equal to 0: the value is x, but neither nvcc nor ptxas
// can hoist the arithmetic out of the repetition loop), and `consume` makes every
// repetition's results needed where they are produced, so they cannot be sunk out of
// it either.
template <typename T>
__device__ __forceinline__ Vec<T> same_value(const Vec<T> &a, const T zero, const int r) {
  Vec<T> o;
#pragma unroll
  for (int e = 0; e < VecOf<T>::NK; ++e) o.v[e] = zero * (T)r + a.v[e];
  return o;
}
__device__ __forceinline__ void consume(const double x) { asm volatile("" ::"d"(x)); }
__device__ __forceinline__ void consume(const float x) { asm volatile("" ::"f"(x)); }
template <typename T>
__device__ __forceinline__ void consume(const Vec<T> &a) {
#pragma unroll
  for (int e = 0; e < VecOf<T>::NK; ++e) consume(a.v[e]);
}


// TMA-issued L2 prefetch of a contiguous run (bytes % 16 == 0, 16-B aligned)
__device__ __forceinline__ void prefetch_l2_bulk(const void *p, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// value one level above each element: r[e] = a[e+1]; the last comes from the
// next lane's first element, or (warp's last lane) from `edge`.
template <typename T>
__device__ __forceinline__ Vec<T> shift_up(const Vec<T> &a, int lane, T edge) {
  constexpr int NK = VecOf<T>::NK;
  Vec<T> r;
#pragma unroll
  for (int e = 0; e + 1 < NK; ++e) r.v[e] = a.v[e + 1];
  T nxt = __shfl_down_sync(kFull, a.v[0], 1);
  r.v[NK - 1] = (lane == 31) ? edge : nxt;
  return r;
}
// flux one level below each element: r[e] = f[e-1]; the first comes from the
// previous lane's last element, or (warp's first lane) from `edge`.
template <typename T>
__device__ __forceinline__ Vec<T> shift_down(const Vec<T> &f, int lane, T edge) {
  constexpr int NK = VecOf<T>::NK;
  Vec<T> r;
#pragma unroll
  for (int e = 1; e < NK; ++e) r.v[e] = f.v[e - 1];
  T prv = __shfl_up_sync(kFull, f.v[NK - 1], 1);
  r.v[0] = (lane == 0) ? edge : prv;
  return r;
}

// values of one x plane a thread carries to the next x step: u, v, w at its
// column and v at the column to the south
template <typename T>
struct PlaneRegs {
  Vec<T> u, v, vs, w;
};
// the three x-face fluxes carried to the next x step
template <typename T>
struct XFlux {
  Vec<T> xx, xy, xz;
};

// ---------------------------------------------------------------------------
// One x step of the fused momentum update for a thread's NK levels (SURVEY.md
// 8(c).2 blocks su/sv/sw): centre plane RC, east plane RE, the centre plane's
// south/north/upper neighbours, the west-face terms FW carried from the
// previous step, and the three vertical fluxes b_* through the face below the
// thread's first level that a shuffle cannot provide (lane 0; unused elsewhere).
// Returns the tendencies of the centre plane and, in FE, the east-face terms
// the next step needs as its west.
// ---------------------------------------------------------------------------
template <typename T, bool SKEW>
__device__ __forceinline__ void momentum_faces(
    const PlaneRegs<T> &RC, const PlaneRegs<T> &RE, const XFlux<T> &FW, XFlux<T> &FE,
    const Vec<T> &uS, const Vec<T> &uN, const Vec<T> &vN, const Vec<T> &wS, const Vec<T> &wN,
    const Vec<T> &uCu, const Vec<T> &vCu, const Vec<T> &wCu, const Vec<T> &vSu, const T b_xz,
    const T b_yz, const T b_zz, const Vec<T> &c1, const Vec<T> &c2, const Vec<T> &d1, const Vec<T> &d2,
    const T cx, const T cy, const int lane, Vec<T> &ou, Vec<T> &ov, Vec<T> &ow) {
  constexpr int NK = VecOf<T>::NK;
  if (SKEW) {
    // Piacsek-Williams skew form (R4): the advected parenthesis holds the
    // neighbour's value only, so a face carries two products, A*phi_far for the
    // point on this side and A*phi_near for the point across the face (handed on
    // through FE in x, by shuffle in z), with the advecting sums A shared.
    Vec<T> su_t, sv_t, sw_t, pu_t, pv_t, pw_t, ry, rv, rwy;
#pragma unroll
    for (int e = 0; e < NK; ++e) {
      const T axu = RC.u.v[e] + RE.u.v[e];     // advects u through the east face
      const T axv = RC.u.v[e] + uN.v[e];       // advects v through the east face
      const T axw = RC.u.v[e] + uCu.v[e];      // advects w through the east face
      const T ayu_n = RC.v.v[e] + RE.v.v[e], ayu_s = RC.vs.v[e] + RE.vs.v[e];
      const T ayv_n = RC.v.v[e] + vN.v[e], ayv_s = RC.vs.v[e] + RC.v.v[e];
      const T ayw_n = RC.v.v[e] + vCu.v[e], ayw_s = RC.vs.v[e] + vSu.v[e];
      const T azu = RC.w.v[e] + RE.w.v[e];     // advects u through the top face
      const T azv = RC.w.v[e] + wN.v[e];
      const T azw = RC.w.v[e] + wCu.v[e];
      ry.v[e] = cx * (FW.xx.v[e] - axu * RE.u.v[e]) + cy * (ayu_s * uS.v[e] - ayu_n * uN.v[e]);
      rv.v[e] = cx * (FW.xy.v[e] - axv * RE.v.v[e]) + cy * (ayv_s * RC.vs.v[e] - ayv_n * vN.v[e]);
      rwy.v[e] = cx * (FW.xz.v[e] - axw * RE.w.v[e]) + cy * (ayw_s * wS.v[e] - ayw_n * wN.v[e]);
      FE.xx.v[e] = axu * RC.u.v[e];
      FE.xy.v[e] = axv * RC.v.v[e];
      FE.xz.v[e] = axw * RC.w.v[e];
      su_t.v[e] = azu * uCu.v[e]; pu_t.v[e] = azu * RC.u.v[e];
      sv_t.v[e] = azv * vCu.v[e]; pv_t.v[e] = azv * RC.v.v[e];
      sw_t.v[e] = azw * wCu.v[e]; pw_t.v[e] = azw * RC.w.v[e];
    }
    const Vec<T> fu_b = shift_down(pu_t, lane, b_xz);
    const Vec<T> fv_b = shift_down(pv_t, lane, b_yz);
    const Vec<T> fw_b = shift_down(pw_t, lane, b_zz);
#pragma unroll
    for (int e = 0; e < NK; ++e) {
      ou.v[e] = ry.v[e] + (c1.v[e] * fu_b.v[e] - c2.v[e] * su_t.v[e]);
      ov.v[e] = rv.v[e] + (c1.v[e] * fv_b.v[e] - c2.v[e] * sv_t.v[e]);
      ow.v[e] = rwy.v[e] + (d1.v[e] * fw_b.v[e] - d2.v[e] * sw_t.v[e]);
    }
  } else {
    // six distinct face fluxes:
    //   fxx (u_i+u_i+1)^2            fyy (v_j+v_j+1)^2           fzz (w_K+w_K+1)^2
    //   fxy (u_j+u_j+1)(v_i+v_i+1)   fxz (u_K+u_K+1)(w_i+w_i+1)  fyz (v_K+v_K+1)(w_j+w_j+1)
    // (FyU == FxV, FzU == FxW, FzV == FyW up to the constant)
    Vec<T> fyz_n, fzz_t, ry, rv, rwy;
#pragma unroll
    for (int e = 0; e < NK; ++e) {
      const T a = RC.u.v[e] + RE.u.v[e];
      FE.xx.v[e] = a * a;
      FE.xy.v[e] = (RC.u.v[e] + uN.v[e]) * (RC.v.v[e] + RE.v.v[e]);
      const T fxy_se = (uS.v[e] + RC.u.v[e]) * (RC.vs.v[e] + RE.vs.v[e]);
      FE.xz.v[e] = (RC.u.v[e] + uCu.v[e]) * (RC.w.v[e] + RE.w.v[e]);
      const T bn = RC.v.v[e] + vN.v[e], bs = RC.vs.v[e] + RC.v.v[e];
      fyz_n.v[e] = (RC.v.v[e] + vCu.v[e]) * (RC.w.v[e] + wN.v[e]);
      const T fyz_s = (RC.vs.v[e] + vSu.v[e]) * (wS.v[e] + RC.w.v[e]);
      const T g = RC.w.v[e] + wCu.v[e];
      fzz_t.v[e] = g * g;
      ry.v[e] = cy * (fxy_se - FE.xy.v[e]);
      rwy.v[e] = cy * (fyz_s - fyz_n.v[e]);
      rv.v[e] = cx * (FW.xy.v[e] - FE.xy.v[e]) + cy * (bs * bs - bn * bn);
    }
    const Vec<T> fxz_b = shift_down(FE.xz, lane, b_xz);
    const Vec<T> fyz_b = shift_down(fyz_n, lane, b_yz);
    const Vec<T> fzz_b = shift_down(fzz_t, lane, b_zz);
#pragma unroll
    for (int e = 0; e < NK; ++e) {
      ou.v[e] = cx * (FW.xx.v[e] - FE.xx.v[e]) + ry.v[e] + (c1.v[e] * fxz_b.v[e] - c2.v[e] * FE.xz.v[e]);
      ov.v[e] = rv.v[e] + (c1.v[e] * fyz_b.v[e] - c2.v[e] * fyz_n.v[e]);
      ow.v[e] = cx * (FW.xz.v[e] - FE.xz.v[e]) + rwy.v[e] + (d1.v[e] * fzz_b.v[e] - d2.v[e] * fzz_t.v[e]);
    }
  }
}

// ---------------------------------------------------------------------------
// march_momentum: fused su, sv, sw (SURVEY.md 8(a) row a1, 8(c).2 blocks su/sv/sw)
//
// EDGES = columns span several warps (nz > 32 vectors): lane 31 / lane 0 of a
// warp read the few scalars of the neighbouring z chunk that a shuffle cannot
// provide.  Lanes above the column top are clamped onto the last vector: they
// load valid data, take part in the shuffles and store nothing.
// ---------------------------------------------------------------------------
template <typename T, bool EDGES>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
march_momentum(const KParams<T> p, const T *__restrict__ u, const T *__restrict__ v,
               const T *__restrict__ w, T *__restrict__ su, T *__restrict__ sv,
               T *__restrict__ sw) {
  constexpr int NK = VecOf<T>::NK;
  const int lane = threadIdx.x & 31;
  const int unit = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (unit >= p.units) return;  // warp-uniform
  const int jr = unit / p.wzc;
  const int zc = unit - jr * p.wzc;
  const int k0r = (zc * 32 + lane) * NK;
  const bool act = k0r < p.nz;
  const int k0 = act ? k0r : p.nz - NK;  // clamp: finite data, never stored
  const bool top_edge = EDGES && act && lane == 31 && (k0 + NK < p.nz);
  const bool bot_edge = EDGES && act && lane == 0 && zc > 0;
  const int i0 = p.ia + blockIdx.y * p.xc;
  const int i1 = min(p.ib, i0 + p.xc);
  const int nz = p.nz;
  const long long plane = p.plane;

  // per-level coefficients, kept in registers for the whole march
  const Vec<T> c1 = ld_vec(p.tzc1 + k0), c2 = ld_vec(p.tzc2 + k0);
  const Vec<T> d1 = ld_vec(p.tzd1 + k0), d2 = ld_vec(p.tzd2 + k0);
  const T cx = p.cx, cy = p.cy;

  const long long c0 = ((long long)(i0 - 1) * p.nyh + (jr + p.h)) * nz + k0;  // (i0-1, j, k0)
  const T *pu = u + c0, *pv = v + c0, *pw = w + c0;
  T *qu = su + c0, *qv = sv + c0, *qw = sw + c0;
  // values of the centre plane that the previous step already loaded
  PlaneRegs<T> RC, RE;
  RC.u = ld_vec(pu); RC.v = ld_vec(pv); RC.vs = ld_vec(pv - nz); RC.w = ld_vec(pw);
  // x-face fluxes on the west side, carried from the previous step
  XFlux<T> FW, FE;
#pragma unroll
  for (int e = 0; e < NK; ++e) FW.xx.v[e] = FW.xy.v[e] = FW.xz.v[e] = T(0);
  const int pf = p.prefetch;
  // one lane per warp asks the TMA unit to pull this warp's 32 vectors of
  // plane i+pf into L2 (DRAM latency then overlaps the steps in between)
  const bool pf_lane = pf > 0 && lane == 0;
  const unsigned pf_bytes = (unsigned)(min(32 * NK, nz - k0r) * (int)sizeof(T));

#pragma unroll 1
  for (int i = i0 - 1; i < i1; ++i) {
    const Vec<T> uS = ld_vec(pu - nz), uN = ld_vec(pu + nz);
    const Vec<T> vN = ld_vec(pv + nz);
    const Vec<T> wS = ld_vec(pw - nz), wN = ld_vec(pw + nz);
    RE.u = ld_vec(pu + plane); RE.v = ld_vec(pv + plane);
    RE.vs = ld_vec(pv + plane - nz); RE.w = ld_vec(pw + plane);
    if (pf_lane && i + pf <= i1) {  // pull plane i+pf of this column towards L2
      prefetch_l2_bulk(pu + pf * plane, pf_bytes); prefetch_l2_bulk(pv + pf * plane, pf_bytes);
      prefetch_l2_bulk(pw + pf * plane, pf_bytes);
    }
    // z-chunk edges: one lane each reads the few scalars a shuffle cannot give
    T e_u = T(0), e_v = T(0), e_w = T(0), e_vs = T(0);
    T b_xz = T(0), b_yz = T(0), b_zz = T(0);
    if (EDGES) {
      if (top_edge) {
        e_u = __ldg(pu + NK); e_v = __ldg(pv + NK);
        e_w = __ldg(pw + NK); e_vs = __ldg(pv - nz + NK);
      }
      if (bot_edge) {
        const T ub = __ldg(pu - 1), vb = __ldg(pv - 1), wb = __ldg(pw - 1);
        const T web = __ldg(pw + plane - 1), wnb = __ldg(pw + nz - 1);
        b_xz = (ub + RC.u.v[0]) * (wb + web);
        b_yz = (vb + RC.v.v[0]) * (wb + wnb);
        b_zz = (wb + RC.w.v[0]) * (wb + RC.w.v[0]);
      }
    }
    const Vec<T> uCu = shift_up(RC.u, lane, e_u), vCu = shift_up(RC.v, lane, e_v);
    const Vec<T> wCu = shift_up(RC.w, lane, e_w), vSu = shift_up(RC.vs, lane, e_vs);

    Vec<T> ou, ov, ow;
    momentum_faces<T, false>(RC, RE, FW, FE, uS, uN, vN, wS, wN, uCu, vCu, wCu, vSu, b_xz, b_yz, b_zz,
                             c1, c2, d1, d2, cx, cy, lane, ou, ov, ow);
    if (k0 == 0) { ou.v[0] = T(0); ov.v[0] = T(0); ow.v[0] = T(0); }  // level K = 1: no tendency
    if (k0 + NK == nz) ow.v[NK - 1] = T(0);                            // level K = nz: sw = 0
    if (i >= i0 && act) {
      if (p.accumulate) {
        const Vec<T> au = ld_vec_rw(qu), av = ld_vec_rw(qv), aw = ld_vec_rw(qw);
#pragma unroll
        for (int e = 0; e < NK; ++e) { ou.v[e] += au.v[e]; ov.v[e] += av.v[e]; ow.v[e] += aw.v[e]; }
      }
      st_vec(qu, ou); st_vec(qv, ov); st_vec(qw, ow);
    }
    // rotate: east becomes centre, its x-face terms the next step's west
    RC = RE;
    FW = FE;
    pu += plane; pv += plane; pw += plane;
    qu += plane; qv += plane; qw += plane;
  }
}

// ---------------------------------------------------------------------------
// march_scalars<G>: G scalars per thread share one read of the wind
// (SURVEY.md 8(a) row a2, 8(c).2 block sq; PAPER.md:83 wind shared by kernels)
// ---------------------------------------------------------------------------
template <typename T, int G>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
march_scalars(const KParams<T> p, const ScalarPtrs<T> ptrs, const int nq, const int ngroups,
              const T *__restrict__ u, const T *__restrict__ v, const T *__restrict__ w) {
  constexpr int NK = VecOf<T>::NK;
  const int lane = threadIdx.x & 31;
  const int grp = blockIdx.x % ngroups;  // group index fastest: co-scheduled blocks share the wind in L2
  const int unit = (blockIdx.x / ngroups) * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (unit >= p.units) return;
  const int s0 = grp * G;
  const int cnt = min(G, nq - s0);
  const int jr = unit / p.wzc;
  const int zc = unit - jr * p.wzc;
  const int k0r = (zc * 32 + lane) * NK;
  const bool act = k0r < p.nz;
  const int k0 = act ? k0r : p.nz - NK;  // clamp: finite data, never stored
  const bool top_edge = act && lane == 31 && (k0 + NK < p.nz);
  const bool bot_edge = act && lane == 0 && zc > 0;
  const int i0 = p.ia + blockIdx.y * p.xc;
  const int i1 = min(p.ib, i0 + p.xc);
  const int nz = p.nz;
  const long long plane = p.plane;

  Vec<T> c1 = ld_vec(p.tzc1 + k0), c2 = ld_vec(p.tzc2 + k0);
#pragma unroll
  for (int e = 0; e < NK; ++e) { c1.v[e] *= T(2); c2.v[e] *= T(2); }
  const T cx2 = T(2) * p.cx, cy2 = T(2) * p.cy;

  long long c = ((long long)(i0 - 1) * p.nyh + (jr + p.h)) * nz + k0;
  Vec<T> qC[G], fx_w[G];
#pragma unroll
  for (int s = 0; s < G; ++s) {
    qC[s] = ld_vec(ptrs.q[s0 + (s < cnt ? s : 0)] + c);
#pragma unroll
    for (int e = 0; e < NK; ++e) fx_w[s].v[e] = T(0);
  }
  const int pf = p.prefetch;
  const bool pf_lane = pf > 0 && lane == 0;
  const unsigned pf_bytes = (unsigned)(min(32 * NK, nz - k0r) * (int)sizeof(T));

#pragma unroll 1
  for (int i = i0 - 1; i < i1; ++i, c += plane) {
    const Vec<T> uC = ld_vec(u + c), vC = ld_vec(v + c);
    const Vec<T> vS = ld_vec(v + c - nz), wC = ld_vec(w + c);
    const T wb = bot_edge ? __ldg(w + c - 1) : T(0);
    if (pf_lane && i + pf <= i1) {
      if (grp == 0) {
        prefetch_l2_bulk(u + c + pf * plane, pf_bytes); prefetch_l2_bulk(v + c + pf * plane, pf_bytes);
        prefetch_l2_bulk(w + c + pf * plane, pf_bytes);
      }
#pragma unroll
      for (int s = 0; s < G; ++s)
        if (s < cnt) prefetch_l2_bulk(ptrs.q[s0 + s] + c + (pf + 1) * plane, pf_bytes);
    }
#pragma unroll
    for (int s = 0; s < G; ++s) {
      if (s < cnt) {  // block-uniform
        const T *__restrict__ q = ptrs.q[s0 + s];
        const Vec<T> qE = ld_vec(q + c + plane);
        const Vec<T> qS = ld_vec(q + c - nz), qN = ld_vec(q + c + nz);
        const T e_q = top_edge ? __ldg(q + c + NK) : T(0);
        const T b_z = bot_edge ? wb * (__ldg(q + c - 1) + qC[s].v[0]) : T(0);
        const Vec<T> qCu = shift_up(qC[s], lane, e_q);
        Vec<T> fz_t, fx_e, hy;
#pragma unroll
        for (int e = 0; e < NK; ++e) {
          fx_e.v[e] = uC.v[e] * (qC[s].v[e] + qE.v[e]);
          hy.v[e] = cy2 * (vS.v[e] * (qS.v[e] + qC[s].v[e]) - vC.v[e] * (qC[s].v[e] + qN.v[e]));
          fz_t.v[e] = wC.v[e] * (qC[s].v[e] + qCu.v[e]);
        }
        const Vec<T> fz_b = shift_down(fz_t, lane, b_z);
        if (i >= i0 && act) {
          T *sq = ptrs.sq[s0 + s];
          Vec<T> o;
#pragma unroll
          for (int e = 0; e < NK; ++e) {
            T x = cx2 * (fx_w[s].v[e] - fx_e.v[e]) + hy.v[e] +
                  (c1.v[e] * fz_b.v[e] - c2.v[e] * fz_t.v[e]);
            if (k0 + e == 0) x = T(0);
            o.v[e] = x;
          }
          if (p.accumulate) {
            const Vec<T> a = ld_vec_rw(sq + c);
#pragma unroll
            for (int e = 0; e < NK; ++e) o.v[e] += a.v[e];
          }
          st_vec(sq + c, o);
        }
        fx_w[s] = fx_e;
        qC[s] = qE;
      }
    }
  }
}

// ---------------------------------------------------------------------------
// generic kernels: one thread per interior point, formulas as written
// ---------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
generic_momentum(const KParams<T> p, const T *__restrict__ u, const T *__restrict__ v,
                 const T *__restrict__ w, T *__restrict__ su, T *__restrict__ sv,
                 T *__restrict__ sw) {
  const long long n = (long long)(p.ib - p.ia) * p.ny * p.nz;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const int k = (int)(t % p.nz);
  const long long r = t / p.nz;
  const int j = (int)(r % p.ny) + p.h;
  const int i = (int)(r / p.ny) + p.ia;
  const long long nz = p.nz, pl = p.plane;
  const long long c = ((long long)i * p.nyh + j) * nz + k;
  T xu = T(0), xv = T(0), xw = T(0);
  if (k > 0) {
    const T uc = u[c], vc = v[c], wc = w[c];
    const T ua = p.skew ? T(0) : uc, va = p.skew ? T(0) : vc, wa = p.skew ? T(0) : wc;
    const bool top = (k == p.nz - 1);
    const T c1 = p.tzc1[k], c2 = p.tzc2[k];
    {
      const T X = p.cx * ((u[c - pl] + uc) * (u[c - pl] + ua) - (uc + u[c + pl]) * (ua + u[c + pl]));
      const T Y = p.cy * ((v[c - nz] + v[c + pl - nz]) * (u[c - nz] + ua) -
                          (vc + v[c + pl]) * (ua + u[c + nz]));
      T Z = c1 * (w[c - 1] + w[c + pl - 1]) * (u[c - 1] + ua);
      if (!top) Z -= c2 * (wc + w[c + pl]) * (ua + u[c + 1]);
      xu = X + Y + Z;
    }
    {
      const T Y = p.cy * ((v[c - nz] + vc) * (v[c - nz] + va) - (vc + v[c + nz]) * (va + v[c + nz]));
      const T X = p.cx * ((u[c - pl] + u[c - pl + nz]) * (v[c - pl] + va) -
                          (uc + u[c + nz]) * (va + v[c + pl]));
      T Z = c1 * (w[c - 1] + w[c + nz - 1]) * (v[c - 1] + va);
      if (!top) Z -= c2 * (wc + w[c + nz]) * (va + v[c + 1]);
      xv = Y + X + Z;
    }
    if (!top) {
      const T X = p.cx * ((u[c - pl] + u[c - pl + 1]) * (w[c - pl] + wa) -
                          (uc + u[c + 1]) * (wa + w[c + pl]));
      const T Y = p.cy * ((v[c - nz] + v[c - nz + 1]) * (w[c - nz] + wa) -
                          (vc + v[c + 1]) * (wa + w[c + nz]));
      const T Z = p.tzd1[k] * (w[c - 1] + wc) * (w[c - 1] + wa) -
                  p.tzd2[k] * (wc + w[c + 1]) * (wa + w[c + 1]);
      xw = X + Y + Z;
    }
  }
  if (p.accumulate) { xu += su[c]; xv += sv[c]; xw += sw[c]; }
  su[c] = xu; sv[c] = xv; sw[c] = xw;
}

template <typename T>
__global__ void __launch_bounds__(256)
generic_scalars(const KParams<T> p, const ScalarPtrs<T> ptrs, const T *__restrict__ u,
                const T *__restrict__ v, const T *__restrict__ w) {
  const long long n = (long long)(p.ib - p.ia) * p.ny * p.nz;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const T *__restrict__ q = ptrs.q[blockIdx.y];
  T *__restrict__ sq = ptrs.sq[blockIdx.y];
  const int k = (int)(t % p.nz);
  const long long r = t / p.nz;
  const int j = (int)(r % p.ny) + p.h;
  const int i = (int)(r / p.ny) + p.ia;
  const long long nz = p.nz, pl = p.plane;
  const long long c = ((long long)i * p.nyh + j) * nz + k;
  T x = T(0);
  if (k > 0) {
    const T qc = q[c];
    const T qa = p.skew ? T(0) : qc;
    const T X = T(2) * p.cx * (u[c - pl] * (q[c - pl] + qa) - u[c] * (qa + q[c + pl]));
    const T Y = T(2) * p.cy * (v[c - nz] * (q[c - nz] + qa) - v[c] * (qa + q[c + nz]));
    T Z = T(2) * p.tzc1[k] * w[c - 1] * (q[c - 1] + qa);
    if (k < p.nz - 1) Z -= T(2) * p.tzc2[k] * w[c] * (qa + q[c + 1]);
    x = X + Y + Z;
  }
  if (p.accumulate) x += sq[c];
  sq[c] = x;
}

}  // namespace monc
