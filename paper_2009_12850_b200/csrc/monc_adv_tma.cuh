// monc_adv_tma.cuh -- TMA-staged x-marching kernels (sm_100a): the default path.
//
// Data movement.  A thread block owns a y tile of full or partial columns and
// marches a chunk of x planes.  At fixed x such a tile is staged into a ring of
// shared-memory slots by the TMA unit (tma_momentum: ONE contiguous 1-D bulk
// copy per field per plane, cp.async.bulk / SASS UBLKCP; tma_scalars: ONE
// tensor-map box copy per field per plane, cp.async.bulk.tensor / UTMALDG),
// completing on mbarriers and running several planes ahead of the consumers.
// DRAM latency is hidden by the ring depth instead of by occupancy; y
// neighbours and z-chunk edges are plain shared-memory reads, vertical face
// fluxes travel between lanes by warp shuffle, x-face fluxes are carried in
// registers from one plane to the next, so every face flux is computed once.
//
// The x march of the fused momentum update exists ONCE (momentum_march): it is
// the consumer loop of tma_momentum and the momentum role of the fused launch.
#pragma once
#include "monc_adv_kernels.cuh"

#include <cuda.h>  // CUtensorMap (type only; the encoder is fetched at run time)

#include <cstdint>
#include <type_traits>

namespace monc {

constexpr int kTmaMaxConsumerWarps = 16;
constexpr int kTmaThreads = kTmaMaxConsumerWarps * 32;
// accumulate mode holds the three old tendencies of a point as well (and the work-scaled
// variant every input of a step across its repetitions): with 128 registers
// per thread (16 warps) the march spills inside its loop and the local-memory loads sit
// on every step's critical path (2.3 x slower, measured); 14 warps leave 144 registers
constexpr int kTmaMaxConsumerWarpsAcc = 14;
constexpr int tma_momentum_max_warps(bool acc) { return acc ? kTmaMaxConsumerWarpsAcc : kTmaMaxConsumerWarps; }

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
#ifndef MONC_ADV_WAIT_HINT
#define MONC_ADV_WAIT_HINT 1  // try_wait with a suspend-time hint (measured against the plain form: DESIGN.md 7.2)
#endif
// Wait for the phase with parity `parity` of an mbarrier, called by ALL 32 lanes of a converged
// warp.  The lanes leave the spin loop TOGETHER (vote.sync.all on the try_wait results): the
// result of try_wait is per lane, and lanes that left a plain spin loop at different
// iterations stay diverged afterwards -- the compiler sees straight-line inline asm, assumes
// convergence and turns the __syncwarp() before a slot release into a NOP, so that lane 0's
// group could release a ring slot while the other group had not yet issued its last shared-
// memory read of it (seen as one launch in ~50 at config 2 reading a plane's u four planes late:
// DESIGN.md 11).
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1, P2;\n"
      "LAB_WAIT:\n"
#if MONC_ADV_WAIT_HINT
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1, 2000;\n"  // suspend for up to 2 us per attempt
#else
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
#endif
      "vote.sync.all.pred P2, P1, 0xffffffff;\n"
      "@P2 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(bar), "r"(parity)
      : "memory");
}
// the same wait for a single lane (tma_momentum's refilling lane, inside a divergent branch)
__device__ __forceinline__ void mbar_wait_one(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(bar), "r"(parity)
      : "memory");
}
// global -> shared bulk copy (bytes % 16 == 0, both addresses 16-B aligned)
__device__ __forceinline__ void tma_load_1d(uint32_t dst, const void *src, uint32_t bytes,
                                            uint32_t bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
      ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
      : "memory");
}

// the same copy with an L2 eviction-priority hint for the lines it reads
__device__ __forceinline__ void tma_load_1d_hint(uint32_t dst, const void *src, uint32_t bytes,
                                                 uint32_t bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
      ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy)
      : "memory");
}
// Input tiles are read by two to four blocks each (the halo rows and z-halo vectors of the
// neighbouring tiles) at times that drift apart during a march: asking L2 to evict them last
// keeps more of the re-reads out of DRAM (+1.7 % sustained on the fused config-2 launch;
// evict_first costs 5-10 %: DESIGN.md 7.1).  0 = no hint.
__device__ __forceinline__ uint64_t l2_policy(const int hint) {
  uint64_t pol = 0;
  if (hint == 1) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  if (hint == 2) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}

// Programmatic dependent launch (PDL): a kernel launched with the programmatic
// stream-serialisation attribute may start while its predecessor in the stream
// drains.  pdl_launch_dependents() lets the successor's blocks be scheduled as
// soon as this grid's blocks have all started; pdl_wait() blocks until the
// predecessor has completed and its writes are visible -- everything before it
// must touch only memory no kernel writes (the coefficient tables).
__device__ __forceinline__ void pdl_launch_dependents() {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ---------------------------------------------------------------------------
// Checked build (-DMONC_ADV_CHECKED=1 -> libmonc_adv_checked.so; tests/test_gpu_checked.py).
// compute-sanitizer is closed on the pool this library is developed on, so the
// ring protocol is shaken out from the inside instead:
//   poison  every ring slot is filled with NaN before each TMA refill (and the whole
//           ring at kernel start): a value read from a slot location the copy did not
//           write, or from a slot released too early and already poisoned for the
//           next plane, reaches an output as NaN and fails the parity tests
//           (initcheck / racecheck on the ring, by construction of the data);
//   jitter  every warp sleeps a pseudo-random 0..2 us before it reads a slot, before
//           it releases one and (producers) before a refill, so that orderings the
//           undisturbed schedule never produces are exercised.
// Results are bitwise those of the normal build (same arithmetic).
// ---------------------------------------------------------------------------
#ifndef MONC_ADV_CHECKED
#define MONC_ADV_CHECKED 0
#endif

__device__ __forceinline__ void chk_jitter(const unsigned salt) {
#if MONC_ADV_CHECKED
  unsigned x = (unsigned)clock64() * 2654435761u + salt * 40503u + blockIdx.x * 9176u + (threadIdx.x >> 5) * 7919u;
  x ^= x >> 15; x *= 2246822519u; x ^= x >> 13;
  if (x & 1u) __nanosleep(x & 2047u);
#endif
}
// NaN-fill `bytes` bytes of shared memory at `dst` with the `nthr` threads that call it
// (thread `tid` of them), then order the generic-proxy stores before later async-proxy
// (TMA) writes to the same locations
__device__ __forceinline__ void chk_poison(const uint32_t dst, const uint32_t bytes, const int tid, const int nthr) {
#if MONC_ADV_CHECKED
  for (uint32_t o = 8u * tid; o + 8u <= bytes; o += 8u * nthr)
    asm volatile("st.shared.b64 [%0], %1;" ::"r"(dst + o), "l"(0x7ff8dead7ff8deadull) : "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
#endif
}

// ---------------------------------------------------------------------------
// Shared-memory loads by 32-bit shared-window address with a compile-time byte
// offset folded into the instruction ([R + imm]): the consumers' address
// arithmetic is then a handful of 32-bit adds per plane.
// ---------------------------------------------------------------------------
template <int OFF>
__device__ __forceinline__ Vec<double> lds_at(uint32_t a, const double *) {
  Vec<double> r;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(r.v[0]), "=d"(r.v[1]) : "r"(a), "n"(OFF));
  return r;
}
template <int OFF>
__device__ __forceinline__ Vec<float> lds_at(uint32_t a, const float *) {
  Vec<float> r;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];"
               : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]) : "r"(a), "n"(OFF));
  return r;
}
template <int OFF>
__device__ __forceinline__ double lds1_at(uint32_t a, const double *) {
  double r;
  asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(r) : "r"(a), "n"(OFF));
  return r;
}
template <int OFF>
__device__ __forceinline__ float lds1_at(uint32_t a, const float *) {
  float r;
  asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(r) : "r"(a), "n"(OFF));
  return r;
}
// r[e] = a[e+1]; the last element is the scalar `top` (level k0 + NK)
template <typename T>
__device__ __forceinline__ Vec<T> up_with(const Vec<T> &a, const T top) {
  constexpr int NK = VecOf<T>::NK;
  Vec<T> r;
#pragma unroll
  for (int e = 0; e + 1 < NK; ++e) r.v[e] = a.v[e + 1];
  r.v[NK - 1] = top;
  return r;
}
// r[e] = a[e-1]; the first element is the scalar `bot` (level k0 - 1)
template <typename T>
__device__ __forceinline__ Vec<T> down_with(const Vec<T> &a, const T bot) {
  constexpr int NK = VecOf<T>::NK;
  Vec<T> r;
#pragma unroll
  for (int e = 1; e < NK; ++e) r.v[e] = a.v[e - 1];
  r.v[0] = bot;
  return r;
}
// accumulate mode: the old tendencies of the plane two steps ahead are pulled into L2 now, so
// that the read-modify-write of that step finds them there (a DRAM miss on every step's critical
// path made the accumulating launches 2-3.5 x slower than the overwriting ones)
__device__ __forceinline__ void prefetch_l2(const void *p) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
// Element-wise global access for the threads whose 16-byte vector is not whole or not
// aligned in the caller's array (nz not a multiple of the vector: DESIGN.md 6.8)
template <typename T>
__device__ __forceinline__ void st_elems(T *p, const Vec<T> &a, const int nlo, const int nhi) {
#pragma unroll
  for (int e = 0; e < VecOf<T>::NK; ++e)
    if (e >= nlo && e < nhi) __stcs(p + e, a.v[e]);
}
template <typename T>
__device__ __forceinline__ Vec<T> ld_elems_rw(const T *p, const int nlo, const int nhi) {
  Vec<T> r;
#pragma unroll
  for (int e = 0; e < VecOf<T>::NK; ++e) r.v[e] = (e >= nlo && e < nhi) ? p[e] : T(0);
  return r;
}
// NK consecutive elements from an address that is element-aligned only (ragged nz: a
// neighbour row's levels are not vector-aligned with the centre row's)
__device__ __forceinline__ Vec<double> lds_elems(uint32_t a, const double *tag) {
  Vec<double> r;
  r.v[0] = lds1_at<0>(a, tag); r.v[1] = lds1_at<8>(a, tag);
  return r;
}
__device__ __forceinline__ Vec<float> lds_elems(uint32_t a, const float *tag) {
  Vec<float> r;
  if ((a & 7u) == 0) {
    // warp-uniform (the lanes are 16 bytes apart): two 8-byte loads are conflict-free at that
    // stride, four 4-byte loads are 4-way bank conflicts each
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(r.v[0]), "=f"(r.v[1]) : "r"(a));
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+8];" : "=f"(r.v[2]), "=f"(r.v[3]) : "r"(a));
  } else {
    r.v[0] = lds1_at<0>(a, tag); r.v[1] = lds1_at<4>(a, tag); r.v[2] = lds1_at<8>(a, tag); r.v[3] = lds1_at<12>(a, tag);
  }
  return r;
}
// a neighbour row's vector: one 16-byte load, or element by element when RAG
template <bool RAG, typename T>
__device__ __forceinline__ Vec<T> lds_row(uint32_t a, const T *tag) {
  if constexpr (RAG) return lds_elems(a, tag);
  else return lds_at<0>(a, tag);
}
// a neighbour row at a compile-time byte offset OFF (aligned columns: the offset folds into the
// instruction) or, RAG, at the warp's run-time offset `rs` (row stride +- the shift between the rows)
template <bool RAG, int OFF, typename T>
__device__ __forceinline__ Vec<T> lds_nb(uint32_t a, uint32_t rs, const T *tag) {
  if constexpr (RAG) return lds_elems(OFF < 0 ? a - rs : a + rs, tag);
  else return lds_at<OFF>(a, tag);
}
// coefficient vector of levels k0 .. k0+NK-1; RAG: element by element, 0 outside the column
template <bool RAG, typename T>
__device__ __forceinline__ Vec<T> ld_coef(const T *tz, const int k0, const int nz) {
  if constexpr (!RAG) {
    return ld_vec(tz + k0);
  } else {
    Vec<T> r;
#pragma unroll
    for (int e = 0; e < VecOf<T>::NK; ++e) r.v[e] = (k0 + e >= 0 && k0 + e < nz) ? __ldg(tz + k0 + e) : T(0);
    return r;
  }
}
// x & m bit by bit (m = 0 or ~0): forces an exact +0 without a predicate, so the
// "no tendency at this level" rule costs a logic op instead of a compare + select
__device__ __forceinline__ double keep_if(double x, int m) {
  return __hiloint2double(__double2hiint(x) & m, __double2loint(x) & m);
}
__device__ __forceinline__ float keep_if(float x, int m) {
  return __int_as_float(__float_as_int(x) & m);
}

// ---------------------------------------------------------------------------
// momentum_march: the x march of one warp over its column chunk, fed by a ring
// of staged planes.  Used by tma_momentum (every consumer warp) and by the
// momentum role of the fused launch (tma_scalars<.., MOM = true>).
//
// Ring protocol: full[s] at bar0 + 8 s completes when the plane in slot s has
// landed; the warp reads a plane when it lands (as the east plane; the values
// it needs again stay in registers) and once more one step later (as the centre
// plane: south/north/upper neighbours), then releases the slot with ONE arrival
// (lane 0) on empty[s] at bar0 + 8 (nstages + s).  `after_release()` runs right
// after that arrival in every step but the first (tma_momentum's refilling lane;
// nothing in the fused launch).
//
// Slot layout, in bytes: field f of stage s at s * sbytes + f * fb, rows rsb
// apart; a0 = shared address of u(this column, k0) in stage 0.  The x loop is
// unrolled by two with the register sets of the centre and east planes (and of
// the west/east x fluxes) swapping roles, so the plane rotation costs no moves.
// ---------------------------------------------------------------------------
template <typename T>
struct MarchArgs {
  uint32_t a0, fb, sbytes, rsb, bar0;
  uint32_t rsbS, rsbN;  // bytes back to the south row / on to the north row (rsb; shifted by whole elements when RAG)
  int nstages, nsteps, lane;
  int work;  // WS: evaluations of the arithmetic per step (results identical)
  T zero;    // WS: 0 as a run-time value (same_value)
  bool act, bot_edge;
  bool vst;        // all NK levels of the thread's vector exist (it is 16-byte aligned by construction)
  int nlo, nhi;    // elements [nlo, nhi) of the vector are levels of the column (0, NK unless nz is ragged)
  int first_elem;  // element that is level K = 1 (no tendency), -1 if none
  int last_elem;   // element that is level K = nz (sw = 0), -1 if none
  T *su, *sv, *sw;            // output arrays (kernel parameters: re-read from the constant bank, not kept in registers)
  long long c0, plane;        // element offset of (i0, j, k0); elements per x plane
  T cx, cy;
  Vec<T> c1, c2, d1, d2;
};

template <typename T, bool ACC, bool SKEW, bool WS, bool RAG, typename AfterRelease>
__device__ __forceinline__ void momentum_march(const MarchArgs<T> &m, AfterRelease &&after_release) {
  constexpr int NK = VecOf<T>::NK;
  constexpr int SZ = (int)sizeof(T);
  constexpr int UP = NK * SZ;  // byte offset of the level above a vector's last element
  const T *const tag = nullptr;
  const uint32_t a0 = m.a0, fb = m.fb, sbytes = m.sbytes, bar0 = m.bar0;
  const uint32_t rsbS = RAG ? m.rsbS : m.rsb, rsbN = RAG ? m.rsbN : m.rsb;
  const int nstages = m.nstages, lane = m.lane;
  const bool bot_edge = m.bot_edge;
  long long c = m.c0;

  mbar_wait(bar0, 0);  // plane i0-1
  PlaneRegs<T> RA, RB;
  XFlux<T> FA, FB;
  RA.u = lds_at<0>(a0, tag);
  RA.v = lds_at<0>(a0 + fb, tag);
  RA.vs = lds_row<RAG>(a0 + fb - rsbS, tag);
  RA.w = lds_at<0>(a0 + 2 * fb, tag);
#pragma unroll
  for (int e = 0; e < NK; ++e) FA.xx.v[e] = FA.xy.v[e] = FA.xz.v[e] = T(0);

  int sC = 0, sE = 1 % nstages;
  uint32_t parE = (nstages == 1) ? 1 : 0;
  uint32_t pC = a0, pE = a0 + (uint32_t)sE * sbytes;

  // one x step: centre plane in RC (registers) / stage sC, east plane arriving in stage sE.
  // The first step (plane i0-1 as the centre) only builds the x-face terms: no store.
  bool first = true;
  int left = m.nsteps;  // steps left, the running one included
  auto step = [&](const PlaneRegs<T> &RC, PlaneRegs<T> &RE, const XFlux<T> &FW, XFlux<T> &FE) {
    // accumulate: what the tendencies are added to is read from global memory; issue those
    // loads first so that their latency overlaps the wait for the plane and the arithmetic
    Vec<T> au, av, aw;
    if (ACC && m.act && left >= 3) {  // this step updates plane c (nothing, the first step), two steps on: c + 2 planes (c + 1)
      const long long ahead = c + (first ? 1 : 2) * m.plane;
      prefetch_l2(m.su + ahead); prefetch_l2(m.sv + ahead); prefetch_l2(m.sw + ahead);
      if (first) { prefetch_l2(m.su + c); prefetch_l2(m.sv + c); prefetch_l2(m.sw + c); }
    }
    if (ACC) {
#pragma unroll
      for (int e = 0; e < NK; ++e) au.v[e] = av.v[e] = aw.v[e] = T(0);
      if (!first) {
        if (m.vst) { au = ld_vec_rw(m.su + c); av = ld_vec_rw(m.sv + c); aw = ld_vec_rw(m.sw + c); }
        else if (RAG && m.act) {
          au = ld_elems_rw(m.su + c, m.nlo, m.nhi); av = ld_elems_rw(m.sv + c, m.nlo, m.nhi);
          aw = ld_elems_rw(m.sw + c, m.nlo, m.nhi);
        }
      }
    }
    mbar_wait(bar0 + 8 * sE, parE);  // plane i+1 has landed
    chk_jitter(1);
    const uint32_t pCv = pC + fb, pCw = pCv + fb, pEv = pE + fb;
    const Vec<T> uS = lds_row<RAG>(pC - rsbS, tag), uN = lds_row<RAG>(pC + rsbN, tag);
    const Vec<T> vN = lds_row<RAG>(pCv + rsbN, tag);
    const Vec<T> wS = lds_row<RAG>(pCw - rsbS, tag), wN = lds_row<RAG>(pCw + rsbN, tag);
    RE.u = lds_at<0>(pE, tag);
    RE.v = lds_at<0>(pEv, tag);
    RE.vs = lds_row<RAG>(pEv - rsbS, tag);
    RE.w = lds_at<0>(pEv + fb, tag);
    const Vec<T> uCu = up_with(RC.u, lds1_at<UP>(pC, tag)), vCu = up_with(RC.v, lds1_at<UP>(pCv, tag));
    const Vec<T> wCu = up_with(RC.w, lds1_at<UP>(pCw, tag));
    const Vec<T> vSu = up_with(RC.vs, lds1_at<UP>(pCv - rsbS, tag));
    T b_xz = T(0), b_yz = T(0), b_zz = T(0);
    if (bot_edge) {  // the level below this warp's first: fluxes a shuffle cannot provide
      const T ub = lds1_at<-SZ>(pC, tag), vb = lds1_at<-SZ>(pCv, tag), wb = lds1_at<-SZ>(pCw, tag);
      const T web = lds1_at<-SZ>(pEv + fb, tag), wnb = lds1_at<-SZ>(pCw + rsbN, tag);
      if (SKEW) {
        b_xz = ub * (wb + web);
        b_yz = vb * (wb + wnb);
        b_zz = wb * (wb + RC.w.v[0]);
      } else {
        b_xz = (ub + RC.u.v[0]) * (wb + web);
        b_yz = (vb + RC.v.v[0]) * (wb + wnb);
        b_zz = (wb + RC.w.v[0]) * (wb + RC.w.v[0]);
      }
    }
    Vec<T> ou, ov, ow;
    if constexpr (WS) {
      // the paper's work-scaling experiment: the same arithmetic m.work
      // times on the same bytes; every evaluation gives the same result
#pragma unroll 1
      for (int r = 0; r < m.work; ++r) {
        PlaneRegs<T> Rc;
        Rc.u = same_value(RC.u, m.zero, r); Rc.v = same_value(RC.v, m.zero, r);
        Rc.vs = same_value(RC.vs, m.zero, r); Rc.w = same_value(RC.w, m.zero, r);
        momentum_faces<T, SKEW>(Rc, RE, FW, FE, uS, uN, vN, wS, wN, uCu, vCu, wCu, vSu, b_xz, b_yz, b_zz,
                                m.c1, m.c2, m.d1, m.d2, m.cx, m.cy, lane, ou, ov, ow);
        consume(ou); consume(ov); consume(ow); consume(FE.xx); consume(FE.xy); consume(FE.xz);
      }
    } else {
      momentum_faces<T, SKEW>(RC, RE, FW, FE, uS, uN, vN, wS, wN, uCu, vCu, wCu, vSu, b_xz, b_yz, b_zz, m.c1,
                              m.c2, m.d1, m.d2, m.cx, m.cy, lane, ou, ov, ow);
    }
    // this warp is done with the centre plane's slot
    chk_jitter(2);
    __syncwarp();
    if (lane == 0) mbar_arrive(bar0 + 8 * (nstages + sC));
    if (!first) {
      after_release();
      if (RAG) {
        if (m.first_elem >= 0 || m.last_elem >= 0) {
#pragma unroll
          for (int e = 0; e < NK; ++e) {
            if (e == m.first_elem) { ou.v[e] = T(0); ov.v[e] = T(0); ow.v[e] = T(0); }
            if (e == m.last_elem) ow.v[e] = T(0);
          }
        }
      } else {
        if (m.first_elem == 0) { ou.v[0] = T(0); ov.v[0] = T(0); ow.v[0] = T(0); }
        if (m.last_elem == NK - 1) ow.v[NK - 1] = T(0);
      }
      if (m.act) {
        T *qu = m.su + c, *qv = m.sv + c, *qw = m.sw + c;
        if (ACC) {
#pragma unroll
          for (int e = 0; e < NK; ++e) { ou.v[e] += au.v[e]; ov.v[e] += av.v[e]; ow.v[e] += aw.v[e]; }
        }
        if (!RAG || m.vst) { st_vec(qu, ou); st_vec(qv, ov); st_vec(qw, ow); }
        else { st_elems(qu, ou, m.nlo, m.nhi); st_elems(qv, ov, m.nlo, m.nhi); st_elems(qw, ow, m.nlo, m.nhi); }
      }
      c += m.plane;
    }
    first = false;
    sC = sE;
    pC = pE;
    pE += sbytes;
    if (++sE == nstages) { sE = 0; parE ^= 1; pE = a0; }
  };
#pragma unroll 1
  while (true) {
    step(RA, RB, FA, FB);
    if (--left == 0) break;
    step(RB, RA, FB, FA);
    if (--left == 0) break;
  }
}

// ---------------------------------------------------------------------------
// tma_momentum<T, ACC, SKEW>: fused su, sv, sw (SURVEY.md 8(a) row a1, 8(c).2 blocks
// su/sv/sw) from a TMA-fed shared-memory ring.
//
// One block = `ty` full columns x a chunk of xc planes; warp <-> (column, 32-vector
// z chunk).  A stage holds the u, v, w tiles of one plane, rows [jr0-1, jr0+ty]:
// at fixed x that is ONE contiguous run of (ty+2)*nz elements per field, so one
// 1-D bulk copy per field fills it.  There is no dedicated producer warp (a 17th
// warp would cap the block at 96 registers per thread): lane 0 of the last warp
// refills, one step late, the slot every warp has released, so the ring runs
// nstages-2 planes ahead.
//
// dynamic shared memory: nstages * 3 * (ty+2) * nz elements, then 2*nstages
// mbarriers.
// ---------------------------------------------------------------------------
template <typename T, bool ACC, bool SKEW, bool WS = false>
__global__ void __launch_bounds__(tma_momentum_max_warps(ACC || WS) * 32, 1)
tma_momentum(const KParams<T> p, const int ty, const int nstages, const T *__restrict__ u,
             const T *__restrict__ v, const T *__restrict__ w, T *__restrict__ su,
             T *__restrict__ sv, T *__restrict__ sw) {
  constexpr int NK = VecOf<T>::NK;
  constexpr int SZ = (int)sizeof(T);
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int nz = p.nz;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int fieldsz = (ty + 2) * nz;  // elements of one field in one stage
  const int stagesz = 3 * fieldsz;
  T *tiles = reinterpret_cast<T *>(smem_raw);
  const uint32_t bar0 = smem_u32(smem_raw + (size_t)nstages * stagesz * sizeof(T));
  // full[s] at bar0 + 8 s, empty[s] at bar0 + 8 (nstages + s)
  const int jr0 = blockIdx.x * ty;
  if (jr0 >= p.ny) return;  // grid padded to whole thread-block clusters
  const int ncol = min(ty, p.ny - jr0);
  const int i0 = p.ia + blockIdx.y * p.xc;
  const int i1 = min(p.ib, i0 + p.xc);
  const int nsteps = i1 - i0 + 1;  // consumer steps: planes i0-1 .. i1-1
  const int ncw = ncol * p.wzc;    // consumer warps that have a column

  if (threadIdx.x == 0) {
    for (int s = 0; s < nstages; ++s) {
      mbar_init(bar0 + 8 * s, 1);
      mbar_init(bar0 + 8 * (nstages + s), ncw);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  chk_poison(smem_u32(smem_raw), (uint32_t)(nstages * stagesz * SZ), threadIdx.x, blockDim.x);
  __syncthreads();

  pdl_launch_dependents();
  if (warp >= ncw) return;
  // coefficient tables are written once at create: safe to read before pdl_wait
  const int col = warp / p.wzc;
  const int zc = warp - col * p.wzc;
  const int k0r = (zc * 32 + lane) * NK;
  MarchArgs<T> m;
  m.act = k0r < nz;
  const int k0 = m.act ? k0r : nz - NK;  // clamp: finite data, never stored
  m.c1 = ld_vec(p.tzc1 + k0); m.c2 = ld_vec(p.tzc2 + k0);
  m.d1 = ld_vec(p.tzd1 + k0); m.d2 = ld_vec(p.tzd2 + k0);
  pdl_wait();  // the fields may have been written by the previous kernel in the stream
  // ---------------- producer role: lane 0 of the last warp ----------------
  const bool producer = (warp == ncw - 1) && lane == 0;
  const uint32_t tile_bytes = (uint32_t)((ncol + 2) * nz * SZ);
  const uint32_t t0 = smem_u32(tiles);
  const uint32_t fb = (uint32_t)(fieldsz * SZ), sb = 3u * fb;
  long long g_next = ((long long)(i0 - 1) * p.nyh + (jr0 + p.h - 1)) * nz;  // next plane to load
  const uint64_t l2pol = l2_policy(p.l2hint);
  int to_issue = nsteps + 1, s_next = 0;  // planes i0-1 .. i1
  uint32_t par_next = 0;  // parity of the empty-phase the next refill of slot s_next waits for
  auto issue_plane = [&]() {
    const uint32_t full = bar0 + 8 * s_next;
    mbar_expect_tx(full, 3 * tile_bytes);
    const uint32_t dst = t0 + (uint32_t)s_next * sb;
    if (p.l2hint) {
      tma_load_1d_hint(dst, u + g_next, tile_bytes, full, l2pol);
      tma_load_1d_hint(dst + fb, v + g_next, tile_bytes, full, l2pol);
      tma_load_1d_hint(dst + 2 * fb, w + g_next, tile_bytes, full, l2pol);
    } else {
      tma_load_1d(dst, u + g_next, tile_bytes, full);
      tma_load_1d(dst + fb, v + g_next, tile_bytes, full);
      tma_load_1d(dst + 2 * fb, w + g_next, tile_bytes, full);
    }
    g_next += p.plane;
    --to_issue;
    if (++s_next == nstages) s_next = 0;
  };
  if (producer) {
    const int first = min(nstages, nsteps + 1);
    for (int n = 0; n < first; ++n) issue_plane();
  }

  // ---------------- consumers: warp <-> (column, z chunk) ----------------
  m.a0 = t0 + (uint32_t)(((col + 1) * nz + k0) * SZ);  // u(column, k0) in stage 0
  m.fb = fb; m.sbytes = sb; m.rsb = (uint32_t)(nz * SZ); m.bar0 = bar0;
  m.nstages = nstages; m.nsteps = nsteps; m.lane = lane;
  m.work = p.work; m.zero = p.zero;
  m.bot_edge = m.act && lane == 0 && zc > 0;
  m.vst = m.act; m.nlo = 0; m.nhi = NK;  // this kernel takes whole, aligned vectors only (nz % NK == 0)
  m.first_elem = k0 == 0 ? 0 : -1;
  m.last_elem = (k0 + NK == nz) ? NK - 1 : -1;
  m.rsbS = m.rsbN = (uint32_t)(nz * SZ);
  m.c0 = ((long long)i0 * p.nyh + (jr0 + col + p.h)) * nz + k0;  // (i0, j, k0)
  m.su = su; m.sv = sv; m.sw = sw;
  m.plane = p.plane;
  m.cx = p.cx; m.cy = p.cy;
  momentum_march<T, ACC, SKEW, WS, false>(m, [&]() {
    if (producer && to_issue > 0) {
      // slot of plane i-1: every warp released it during the previous step
      mbar_wait_one(bar0 + 8 * (nstages + s_next), par_next);
      chk_jitter(3);
      chk_poison(t0 + (uint32_t)s_next * sb, sb, 0, 1);
      issue_plane();
      if (s_next == 0) par_next ^= 1;
    }
  });
}

// ---------------------------------------------------------------------------
// Tensor-map TMA (cp.async.bulk.tensor, SASS UTMALDG): one instruction moves a
// (z, y) box of one x plane of one field, strided rows and all, and fills
// out-of-range elements (levels below 0 / above nz-1, rows past the array)
// with zeros.  Descriptors are encoded on the host per plan (the field
// pointers are call arguments) and passed as __grid_constant__ parameters.
// ---------------------------------------------------------------------------
constexpr int kMaxScalarsPerLaunch = 20;  // 23 descriptors of 128 B stay below the 4 KB parameter limit

struct alignas(64) TensorMaps {
  CUtensorMap m[3 + kMaxScalarsPerLaunch];  // u, v, w, then the scalars of this launch
};
template <typename T>
struct SqPtrs {
  T *sq[kMaxScalarsPerLaunch];
};
// outputs of the momentum role of the fused launch (MOM = true)
template <typename T>
struct MomPtrs {
  T *su, *sv, *sw;
};

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *map, int c0, int c1,
                                            int c2, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
      " [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
      : "memory");
}
// the same copy with an L2 eviction-priority hint for the lines it reads
__device__ __forceinline__ void tma_load_3d_hint(uint32_t dst, const CUtensorMap *map, int c0, int c1,
                                                 int c2, uint32_t bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3, %4}], [%5], %6;"
      ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar), "l"(policy)
      : "memory");
}
__device__ __forceinline__ void prefetch_tensormap(const CUtensorMap *map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// ---------------------------------------------------------------------------
// tma_scalars<T, GW, ACC, SKEW, MOM>: batched scalar tendencies (SURVEY.md 8(a) row a2, 8(c).2
// block sq; PAPER.md:83 wind shared by kernels).
//
// A block owns a (y, z) tile of `ty` columns x ZB = 32*NK levels (one 16-byte
// vector per lane), advects gb = GW*ss scalars of one group and marches a chunk of
// x planes.  A stage of the ring holds, for u, v, w and the gb scalars, the box
// rows [jr0-1, jr0+ty] x levels [kb0-NK, kb0+ZB+NK) of ONE plane: one tensor-map
// TMA copy per field, issued by a dedicated producer warp (lanes 0..2+gb),
// completing on the stage's `full` mbarrier.  Elements outside the array are
// zero-filled by the TMA unit: they are read (the top level's upper neighbour)
// but multiplied by a zero coefficient.  The row stride is the compile-time
// constant kRowBytes = 34 vectors for both dtypes, so the y and z neighbours of
// a value are immediate offsets from one register.
//
// Consumer warp <-> (column, scalar split): `ss` warps share one column chunk
// and take GW scalars each, so the warp count (latency hiding) does not shrink
// when the tile is made small enough for a deep ring.
//
// Every plane is touched in exactly ONE consumer step (so S-1 of the S stages
// can be in flight).  When plane i lands a thread forms, once for its GW scalars,
// the advecting velocities of the four faces of plane i scaled by their
// coefficients (2cx u, 2cy v, 2tzc1 w below, 2tzc2 w) and then, per scalar, the y
// and z flux differences P of plane i and the x flux f through the face between
// planes i-1 and i: A = P + f is carried to the next step, where subtracting that
// step's f completes sq(i), which is stored.  Two values per scalar stay in
// registers from one plane to the next (q and A).
//
// MOM = true is the fused launch behind monc_adv_tendencies: each
// column chunk gets one more consumer warp, whose role is the momentum update
// (su, sv, sw) of that chunk from the SAME staged wind tiles (momentum_march), so
// u, v, w are read from DRAM once for the whole step.  It needs a plane twice
// (east, then centre), so it releases a slot one step after the scalar warps do.
// Requires one scalar group.
//
// dynamic shared memory: nstages * (3+gb) field tiles of fieldsz elements
// ((ty+2) rows of kRowBytes, rounded up to 128 B), then 2*nstages mbarriers.
// ---------------------------------------------------------------------------
// 15 consumer warps + the producer warp = 512 threads: 128 registers per thread
constexpr int kScalarConsumerWarps = 15;
constexpr int kScalarThreads = (kScalarConsumerWarps + 1) * 32;
constexpr int kRowBytes = 34 * 16;  // 32 vectors of the tile + one vector of z halo on each side
// Ragged nz (tma_scalars, RAG): the tensor view holds G columns per row; the columns j = c mod G
// of a tile ("class" c) are one box of ceil(rows / G) box rows, staged in a class block of its
// own (128-byte aligned: a tensor copy's destination must be): bytes of one class block / field
__host__ __device__ constexpr int ragged_class_rows(int rows, int g) { return (rows + g - 1) / g; }
__host__ __device__ constexpr int ragged_class_bytes(int rows, int g) {
  return (ragged_class_rows(rows, g) * kRowBytes + 127) / 128 * 128;
}
// bytes of one field tile of `rows` rows in a ring stage
__host__ __device__ constexpr int scalar_field_bytes(int rows, int g, bool rag) {
  return rag ? g * ragged_class_bytes(rows, g) : (rows * kRowBytes + 127) / 128 * 128;
}
// z tiles of 32 vectors per column; a ragged column's levels are shifted by up to NK-1
// elements against its vectors (tma_scalars, RAG)
__host__ __device__ constexpr int scalar_z_tiles(int nz, int nk, int g, bool rag) {
  int shift = 0;  // the largest (c nz) mod NK over the classes c < G
  if (rag)
    for (int c = 1; c < g; ++c) shift = (c * (nz % nk)) % nk > shift ? (c * (nz % nk)) % nk : shift;
  return (nz + shift + 32 * nk - 1) / (32 * nk);
}

// The scalar role of one warp: GW scalars (mycnt of them live when !FULL) of one
// column chunk over the block's planes.
template <typename T, int GW, bool ACC, bool SKEW, bool FULL, bool WS, bool RAG>
__device__ __forceinline__ void scalar_march(const uint32_t a0, const uint32_t fb, const uint32_t sbytes,
                                             const uint32_t rsbS, const uint32_t rsbN, const uint32_t q0off, const uint32_t bar0, const int nstages,
                                             const int nplanes, const int mycnt, const int work, const T zero,
                                             const int lane,
                                             const bool act, const bool vst, const int nlo, const int nhi,
                                             const bool bot_edge, const int (&keep)[VecOf<T>::NK],
                                             T *const *__restrict__ sqp, const long long c0,
                                             const long long plane, const Vec<T> &c1, const Vec<T> &c2,
                                             const T cx2, const T cy2) {
  constexpr int NK = VecOf<T>::NK;
  constexpr int SZ = (int)sizeof(T);
  constexpr int UP = NK * SZ;
  const T *const tag = nullptr;
  // carried per scalar: q of the previous plane (two register sets that swap roles in
  // the x loop unrolled by two, so the rotation costs no moves) and A = P + f of it
  Vec<T> QA[GW], QB[GW], CA[GW];
  Vec<T> UA, UB;  // 2cx u of the previous plane (the face between it and the arriving one): swap like q
#pragma unroll
  for (int e = 0; e < NK; ++e) UA.v[e] = T(0);
#pragma unroll
  for (int s = 0; s < GW; ++s) {
#pragma unroll
    for (int e = 0; e < NK; ++e) QA[s].v[e] = CA[s].v[e] = T(0);
  }
  int st = 0;
  uint32_t par = 0, pA = a0;
  long long c = c0;
  int togo = nplanes;  // steps left, this one included

  auto step = [&](auto store_tag, const Vec<T> (&QP)[GW], Vec<T> (&QN)[GW], const Vec<T> &ux, Vec<T> &un) {
    constexpr bool STORE = decltype(store_tag)::value;
    if (ACC && act && togo >= 3) {
      // a storing step updates plane c and pulls plane c + 2 in; the two steps before the first
      // store (c = c0 in both) pull in the planes the first two stores update
      const long long ahead = STORE ? c + 2 * plane : c + (nplanes - togo) * plane;
#pragma unroll
      for (int s = 0; s < GW; ++s)
        if (FULL || s < mycnt) prefetch_l2(sqp[s] + ahead);
    }
    mbar_wait(bar0 + 8 * st, par);  // the next plane has landed
    chk_jitter(4);
    const uint32_t pV = pA + fb, pW = pV + fb;
    Vec<T> vs = lds_nb<RAG, -kRowBytes>(pV, rsbS, tag), vn = lds_at<0>(pV, tag);
    Vec<T> wt = lds_at<0>(pW, tag);
    Vec<T> wl = down_with(wt, lds1_at<-SZ>(pW, tag));  // w one level below each element
    un = lds_at<0>(pA, tag);  // read now: the slot's release must not wait for it
#pragma unroll
    for (int e = 0; e < NK; ++e) {
      vs.v[e] *= cy2; vn.v[e] *= cy2;
      wl.v[e] *= c1.v[e]; wt.v[e] *= c2.v[e];
      un.v[e] *= cx2;
    }
    uint32_t pQ = pA + q0off;
#pragma unroll
    for (int s = 0; s < GW; ++s) {
      if (FULL || s < mycnt) {  // warp-uniform
        QN[s] = lds_at<0>(pQ, tag);
        const Vec<T> &q = QN[s];
        const Vec<T> qS = lds_nb<RAG, -kRowBytes>(pQ, rsbS, tag), qN = lds_nb<RAG, kRowBytes>(pQ, rsbN, tag);
        const T qtop = lds1_at<UP>(pQ, tag);  // the level above the thread's last
        // the level below the thread's first: lane 0 reads it, the others get it by shuffle
        const T qb = bot_edge ? lds1_at<-SZ>(pQ, tag) : T(0);
        Vec<T> o, can;
        // o: the previous plane's tendency, complete; can: this plane's A.  qc is the centre
        // vector the arithmetic reads (q itself, or an opaque copy when the work is repeated)
        auto evaluate = [&](const Vec<T> &qc) {
          const Vec<T> qU = up_with(qc, qtop);
          if (SKEW) {
            // Piacsek-Williams skew form (R4): the advected parenthesis holds the
            // far value only, so each face contributes the neighbour's value times the
            // (scaled) advecting velocity
            const T prv = __shfl_up_sync(kFull, qc.v[NK - 1], 1);
            const Vec<T> qD = down_with(qc, lane == 0 ? qb : prv);
#pragma unroll
            for (int e = 0; e < NK; ++e) {
              T y = vn.v[e] * qN.v[e];
              y = vs.v[e] * qS.v[e] - y;
              y = wl.v[e] * qD.v[e] + y;
              y = y - wt.v[e] * qU.v[e];
              o.v[e] = CA[s].v[e] - ux.v[e] * qc.v[e];
              can.v[e] = y + ux.v[e] * QP[s].v[e];
            }
          } else {
            Vec<T> g;
#pragma unroll
            for (int e = 0; e < NK; ++e) g.v[e] = qc.v[e] + qU.v[e];
            const T prv = __shfl_up_sync(kFull, g.v[NK - 1], 1);
            const Vec<T> gD = down_with(g, lane == 0 ? qb + qc.v[0] : prv);
#pragma unroll
            for (int e = 0; e < NK; ++e) {
              T y = vn.v[e] * (qc.v[e] + qN.v[e]);
              y = vs.v[e] * (qS.v[e] + qc.v[e]) - y;
              y = wl.v[e] * gD.v[e] + y;
              y = y - wt.v[e] * g.v[e];  // P: the y and z flux differences of this plane
              const T sx = QP[s].v[e] + qc.v[e];
              o.v[e] = CA[s].v[e] - ux.v[e] * sx;  // minus the flux through the face between the two planes
              can.v[e] = y + ux.v[e] * sx;
            }
          }
        };
        if constexpr (WS) {
          // the same arithmetic `work` times on the same bytes, same result
#pragma unroll 1
          for (int r = 0; r < work; ++r) {
            evaluate(same_value(q, zero, r));
            consume(o); consume(can);
          }
        } else {
          evaluate(q);
        }
        CA[s] = can;
        if (STORE) {  // sq of the previous plane is complete
          if (RAG) {  // level K = 1 may be any element of the vector
#pragma unroll
            for (int e = 0; e < NK; ++e) o.v[e] = keep_if(o.v[e], keep[e]);
          } else {
            o.v[0] = keep_if(o.v[0], keep[0]);
          }
          T *sq = sqp[s] + c;  // pointer table lives in the constant bank
          if (ACC) {
            if (act) {
              const Vec<T> a = (!RAG || vst) ? ld_vec_rw(sq) : ld_elems_rw(sq, nlo, nhi);
#pragma unroll
              for (int e = 0; e < NK; ++e) o.v[e] += a.v[e];
            }
          }
          if (RAG) {
            if (vst) st_vec(sq, o);
            else if (act) st_elems(sq, o, nlo, nhi);  // a vector that straddles an end of the column
          } else {
            if (act) st_vec(sq, o);  // nothing but the store under the predicate
          }
        }
        pQ += fb;
      }
    }
    // this warp is done with the slot
    chk_jitter(5);
    __syncwarp();
    if (lane == 0) mbar_arrive(bar0 + 8 * (nstages + st));
    if (STORE) c += plane;
    --togo;
    pA += sbytes;
    if (++st == nstages) { st = 0; par ^= 1; pA = a0; }
  };
  // plane i0-1 only leaves q and u behind, plane i0 the first A; from then on every
  // plane completes the tendencies of the one before it
  step(std::false_type{}, QA, QB, UA, UB);
  step(std::false_type{}, QB, QA, UB, UA);
  int left = nplanes - 2;
#pragma unroll 1
  while (left > 0) {
    step(std::true_type{}, QA, QB, UA, UB);
    if (--left == 0) break;
    step(std::true_type{}, QB, QA, UB, UA);
    --left;
  }
}

template <typename T, int GW, bool ACC, bool SKEW, bool MOM, bool WS = false, bool RAG = false>
__global__ void __launch_bounds__(kScalarThreads, 1)
tma_scalars(const KParams<T> p, const __grid_constant__ TensorMaps maps, const SqPtrs<T> outs,
            const MomPtrs<T> mo, const int nq, const int ngroups, const int gb, const int ty,
            const int ss, const int nstages, const int fieldsz, const int cl) {
  constexpr int NK = VecOf<T>::NK;
  constexpr int SZ = (int)sizeof(T);
  constexpr int ZB = 32 * NK;                // levels per block tile
  constexpr uint32_t rowb = (uint32_t)kRowBytes;  // bytes between consecutive rows of a tile (of a class block, RAG)
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int nz = p.nz;
  const int lane = threadIdx.x & 31;
  const int warp = __shfl_sync(kFull, (int)(threadIdx.x >> 5), 0);  // tells the compiler it is warp-uniform
  const int rows = ty + 2;
  const int stagesz = (3 + gb) * fieldsz;
  const uint32_t t0 = smem_u32(smem_raw);
  const uint32_t bar0 = t0 + (uint32_t)(nstages * stagesz * SZ);
  // full[s] at bar0 + 8 s, empty[s] at bar0 + 8 (nstages + s)

  // block -> (scalar group, z tile, y tile); group fastest so that the blocks
  // sharing a wind tile run together and the later reads hit L2
  const int grp = blockIdx.x % ngroups;
  const int tile = blockIdx.x / ngroups;
  const int nzt = scalar_z_tiles(nz, NK, p.colgroup, RAG);
  // `cl` consecutive blocks are one thread-block cluster: y-neighbour tiles of the same z
  // tile, co-scheduled on one GPC so that they advance at the same rate and find each
  // other's halo rows in L2 (cl = 1: z tile fastest).  Tiles past the last y tile pad the
  // grid to whole clusters and exit.
  const int cidx = tile / cl, crank = tile - cidx * cl;
  const int zt = cidx % nzt, yt = (cidx / nzt) * cl + crank;
  if (yt * ty >= p.ny) return;
  const int s0 = grp * gb;
  const int cnt = min(gb, nq - s0);  // scalars of this block
  const int jr0 = yt * ty;
  const int ncol = min(ty, p.ny - jr0);
  const int kb0 = zt * ZB;
  const int slive = (cnt + GW - 1) / GW;                   // splits with a scalar
  const int nr = ss + (MOM ? 1 : 0);                       // roles per column
  const int ncw = ncol * (slive + (MOM ? 1 : 0));          // live consumer warps
  const int i0 = p.ia + blockIdx.y * p.xc;
  const int i1 = min(p.ib, i0 + p.xc);
  const int nplanes = i1 - i0 + 2;  // planes i0-1 .. i1
  const int nwarps_c = ty * nr;

  if (threadIdx.x == 0) {
    for (int s = 0; s < nstages; ++s) {
      mbar_init(bar0 + 8 * s, 1);
      mbar_init(bar0 + 8 * (nstages + s), ncw);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  chk_poison(t0, (uint32_t)(nstages * stagesz * SZ), threadIdx.x, blockDim.x);
  __syncthreads();

  pdl_launch_dependents();
  if (warp == nwarps_c) {
    // ---------------- producer warp: one lane per field ----------------
    const int nfld = 3 + cnt;
    const uint32_t box_bytes = (uint32_t)(rows * kRowBytes);
    const CUtensorMap *mymap = &maps.m[lane < 3 ? lane : 3 + s0 + max(0, min(lane - 3, cnt - 1))];
    if (lane < nfld) prefetch_tensormap(mymap);
    pdl_wait();  // the fields may have been written by the previous kernel in the stream
    const uint32_t dst0 = t0 + (uint32_t)(lane * fieldsz * SZ);
    const int G = p.colgroup;
    const uint64_t l2pol = l2_policy(p.l2hint);
    const int jcfirst = jr0 + p.h - 1;  // array column of the tile's first row
    const uint32_t cbs = (uint32_t)ragged_class_bytes(rows, G);
    int s = 0;
    uint32_t par = 1;  // a fresh mbarrier passes a wait on parity 1: the first lap does not block
#pragma unroll 1
    for (int n = 0; n < nplanes; ++n) {
      mbar_wait(bar0 + 8 * (nstages + s), par);  // every consumer warp released the slot
      chk_jitter(6);
      if (n >= nstages) chk_poison(t0 + (uint32_t)(s * stagesz * SZ), (uint32_t)(stagesz * SZ), lane, 32);
      const uint32_t full = bar0 + 8 * s;
      if constexpr (!RAG) {
        if (lane == 0) mbar_expect_tx(full, (uint32_t)nfld * box_bytes);
        __syncwarp();
        if (lane < nfld) {
          if (p.l2hint)
            tma_load_3d_hint(dst0 + (uint32_t)(s * stagesz * SZ), mymap, kb0 - NK, jr0 + p.h - 1, i0 - 1 + n, full, l2pol);
          else
            tma_load_3d(dst0 + (uint32_t)(s * stagesz * SZ), mymap, kb0 - NK, jr0 + p.h - 1, i0 - 1 + n, full);
        }
      } else {
        // ragged nz (a column is not a whole number of 16-byte vectors): the descriptor views G
        // columns as one row (G nz elements: a multiple of 16 bytes), so column j is the elements
        // from (j mod G) nz of row j / G.  One copy per field and class c = j mod G brings that
        // class's columns of the tile (consecutive rows of the view) into its class block.  A copy
        // must start on a 16-byte boundary: it starts at the vector that holds level kb0 - NK of
        // the column, i.e. the class is staged shifted by (c nz) mod NK elements (the consumers know).
        if (lane == 0) mbar_expect_tx(full, (uint32_t)(nfld * G * ragged_class_rows(rows, G) * kRowBytes));
        __syncwarp();
        for (int idx = lane; idx < nfld * G; idx += 32) {
          const int f = idx / G, c = idx - f * G;
          const int e0 = c * nz;  // the column's first level in its row of the view
          const uint32_t dst = t0 + (uint32_t)((s * stagesz + f * fieldsz) * SZ) + (uint32_t)c * cbs;
          const CUtensorMap *map = &maps.m[f < 3 ? f : s0 + f];
          const int cz = e0 - e0 % NK + kb0 - NK, cy = (jcfirst - c + G - 1) / G;
          if (p.l2hint) tma_load_3d_hint(dst, map, cz, cy, i0 - 1 + n, full, l2pol);
          else tma_load_3d(dst, map, cz, cy, i0 - 1 + n, full);
        }
      }
      if (++s == nstages) { s = 0; par ^= 1; }
    }
    return;
  }

  // ---------------- consumers ----------------
  const int col = warp / nr;
  const int sp = warp - col * nr;
  if (col >= ncol) return;
  // RAG: column jc starts mc elements into a 16-byte vector of the array; its threads own the
  // vectors of the ARRAY (so the centre row is vector-aligned in shared memory and the stores
  // are vector-aligned in global memory), i.e. levels shifted down by mc; the neighbour rows
  // are shifted by their own amounts and are read element by element
  const int jc = jr0 + col + p.h;
  const int mc = RAG ? (int)(((long long)jc * nz) % NK) : 0;
  const int k0r = kb0 + lane * NK - mc;
  const int nlo = max(0, -k0r), nhi = min(NK, nz - k0r);  // elements [nlo, nhi) are levels of the column
  const bool act = nhi > nlo;
  const int k0 = RAG ? k0r : (act ? k0r : kb0);  // !RAG: clamp (finite data, never stored)
  const bool bot_edge = act && lane == 0 && k0r > 0;
  const uint32_t fb = (uint32_t)(fieldsz * SZ), sbytes = (uint32_t)(stagesz * SZ);
  // u(column, k0) in stage 0: row col+1 of the box, one vector of z halo before level kb0
  uint32_t a0 = t0 + (uint32_t)(col + 1) * rowb + (uint32_t)((lane + 1) * NK * SZ);
  uint32_t rsbS = rowb, rsbN = rowb;
  if (RAG) {
    // byte offset, in a field tile, of the row of array column j: class block j mod G, then the
    // rows of that class in order; a row's levels sit (j nz) mod NK elements further on
    const int G = p.colgroup, jcfirst = jr0 + p.h - 1;
    const uint32_t cbs = (uint32_t)ragged_class_bytes(rows, G);
    auto row_at = [&](const int j) {
      const int c = j % G;
      return (uint32_t)c * cbs + (uint32_t)(j / G - (jcfirst - c + G - 1) / G) * rowb;
    };
    const int mS = (int)(((long long)(jc - 1) * nz) % NK), mN = (int)(((long long)(jc + 1) * nz) % NK);
    const uint32_t rc = row_at(jc);
    a0 = t0 + rc + (uint32_t)((lane + 1) * NK * SZ);
    rsbS = rc - row_at(jc - 1) - (uint32_t)((mS - mc) * SZ);
    rsbN = row_at(jc + 1) - rc + (uint32_t)((mN - mc) * SZ);
  }
  const long long c0 = ((long long)i0 * p.nyh + (jr0 + col + p.h)) * nz + k0;  // (i0, j, k0)
  const bool vst = nlo == 0 && nhi == NK;  // all NK levels exist
  int keep[NK];  // 0 for the element that is level K = 1 (no tendency), else ~0
#pragma unroll
  for (int e = 0; e < NK; ++e) {
    keep[e] = k0r + e == 0 ? 0 : -1;
    asm volatile("" : "+r"(keep[e]));  // keep it a mask for a logic op: no compare + select per store
  }
  if (MOM && sp == ss) {
    // ---------------- momentum role (fused launch): su, sv, sw of this column chunk
    // from the wind tiles the scalar warps use
    MarchArgs<T> m;
    m.c1 = ld_coef<RAG>(p.tzc1, k0, nz); m.c2 = ld_coef<RAG>(p.tzc2, k0, nz);
    m.d1 = ld_coef<RAG>(p.tzd1, k0, nz); m.d2 = ld_coef<RAG>(p.tzd2, k0, nz);
    m.a0 = a0; m.fb = fb; m.sbytes = sbytes; m.rsb = rowb; m.rsbS = rsbS; m.rsbN = rsbN; m.bar0 = bar0;
    m.nstages = nstages; m.nsteps = nplanes - 1; m.lane = lane;
    m.work = p.work; m.zero = p.zero;
    m.act = act; m.bot_edge = bot_edge;
    m.vst = vst; m.nlo = nlo; m.nhi = nhi;
    m.first_elem = (-k0r >= 0 && -k0r < NK) ? -k0r : -1;
    m.last_elem = (nz - 1 - k0r >= 0 && nz - 1 - k0r < NK) ? nz - 1 - k0r : -1;
    m.su = mo.su; m.sv = mo.sv; m.sw = mo.sw;
    m.c0 = c0; m.plane = p.plane;
    m.cx = p.cx; m.cy = p.cy;
    pdl_wait();
    momentum_march<T, ACC, SKEW, WS, RAG>(m, []() {});
    return;
  }
  if (sp >= slive) return;
  const int sb = sp * GW;              // first scalar (within the block's group) of this warp
  const int mycnt = min(GW, cnt - sb);
  Vec<T> c1 = ld_coef<RAG>(p.tzc1, k0, nz), c2 = ld_coef<RAG>(p.tzc2, k0, nz);
#pragma unroll
  for (int e = 0; e < NK; ++e) { c1.v[e] *= T(2); c2.v[e] *= T(2); }
  const T cx2 = T(2) * p.cx, cy2 = T(2) * p.cy;
  const uint32_t q0off = (uint32_t)(3 + sb) * fb;  // this warp's first scalar
  T *const *sqp = outs.sq + (s0 + sb);
  pdl_wait();  // accumulate mode reads sq, which the previous kernel may have written
  if (mycnt == GW)
    scalar_march<T, GW, ACC, SKEW, true, WS, RAG>(a0, fb, sbytes, rsbS, rsbN, q0off, bar0, nstages, nplanes, mycnt,
                                                  p.work, p.zero, lane, act, vst, nlo, nhi, bot_edge, keep, sqp, c0,
                                                  p.plane, c1, c2, cx2, cy2);
  else
    scalar_march<T, GW, ACC, SKEW, false, WS, RAG>(a0, fb, sbytes, rsbS, rsbN, q0off, bar0, nstages, nplanes, mycnt,
                                                   p.work, p.zero, lane, act, vst, nlo, nhi, bot_edge, keep, sqp, c0,
                                                   p.plane, c1, c2, cx2, cy2);
}

}  // namespace monc
