// monc_adv.cu -- C ABI (include/monc_adv.h) over the sm_100a kernels.
//
// Host side of the library: handle, one-time constant upload,
// kernel launch configuration, and the hybrid asynchronous step (PAPER.md:75-83,
// 99-101): chunked H2D -> kernels -> D2H on separate streams with events.
// No torch types, no CPU compute fallback: if CUDA fails the call fails.
#include "monc_adv.h"
#include "monc_adv_tuning.h"
#include "monc_adv_kernels.cuh"
#include "monc_adv_tma.cuh"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <set>
#include <string>
#include <tuple>
#include <utility>
#include <vector>

using namespace monc;

namespace {
thread_local std::string g_create_error;
}

// default thread-block cluster sizes (y-neighbour tiles co-scheduled on one GPC)
constexpr int kDefaultClusterMomentum = 4;  // single-wave launches only
constexpr int kDefaultClusterScalars = 1;

// geometry of the TMA-staged kernels: TY columns per block, ring depth S
struct TmaPlan {
  bool ok = false;
  int ty = 0, stages = 0, xc = 0, tiles = 0, nchunks = 0;
  int cl = 1;  // thread-block cluster: cl y-neighbour tiles are co-scheduled on one GPC
  bool cl_checked = false;  // the default cluster size has been checked against the device's resident clusters
  size_t smem = 0;
};
// geometry of tma_scalars: ty columns x ss scalar splits = consumer warps per
// block; gb scalars per block (gw per warp); ring depth S.  A stage holds 3 + gb
// field tiles of (ty+2) rows of kRowBytes (each tile rounded up to 128 B).
struct TmaScalarPlan {
  bool ok = false;
  int ty = 0, ss = 0, gb = 0, gw = 0, stages = 0, xc = 0, tiles = 0, nchunks = 0, fieldsz = 0;
  int cl = 1;  // thread-block cluster: cl y-neighbour tiles are co-scheduled on one GPC
  size_t smem = 0;
};
// tensor-map descriptors of one launch, kept while the same arrays come back
// (the chunks of a hybrid step, the rotating buffer sets of a time loop)
struct MapEntry {
  std::vector<const void *> ptrs;  // u, v, w, q[0..n)
  int ty = 0;
  unsigned long stamp = 0;
  TensorMaps maps;
};

struct monc_adv_s {
  int nx = 0, ny = 0, nz = 0, h = 0, dtype = 0;
  int nxh = 0, nyh = 0;
  // tensor-map view of a field for tma_scalars: `colgroup` columns form one row, so that a row
  // is a whole number of 16-byte vectors whatever nz is (1 when nz already is; 2 or 4 when nz is
  // ragged; 0 = no such view: nyh is not a multiple of it, the generic kernels run)
  int colgroup = 1;
  bool plan_only = false;  // a shape without a device behind it (monc_adv_plan_describe)
  double dx = 0, dy = 0;
  size_t elems = 0, esize = 8;
  int device = 0;
  int sm_count = 148;
  void *d_tz[4] = {nullptr, nullptr, nullptr, nullptr};  // tzc1, tzc2, tzd1, tzd2 (dtype)
  std::vector<double> tz_host[4];                        // as stored on the device
  const void *wind[3] = {nullptr, nullptr, nullptr};
  int form = MONC_ADV_FORM_FLUX, accumulate = 0, variant = 0, pdl = 1, fuse = 1, work = 1;
  volatile double zero = 0.0;  // handed to the work-scaled kernels as a run-time 0
  int xchunk = 0, group = 0, prefetch = 0, warps = 0;  // 0 = default
  int stages = 0, tile_y = 0, split = 0;                // TMA kernels, 0 = default
  int cluster = 0;                                      // TMA kernels: y tiles per thread-block cluster, 0 = default
  int l2hint = 1;                                       // TMA kernels: input copies ask L2 to evict them last
  int smem_optin = 0;                                   // max dynamic smem per block
  long launches = 0;
  std::string err;
  std::string plan_mom, plan_sca, plan_text;  // geometry of the last launches
  // launch plans by (planes, scalars, fused); dropped when a tuning knob changes
  std::map<int, TmaPlan> mom_plans;
  std::map<std::tuple<int, int, int>, TmaScalarPlan> sca_plans;
  std::vector<MapEntry> map_cache;
  unsigned long map_clock = 0;
  // ---- async step state
  int nchunks = 0, overlap = 1;  // nchunks 0 = chosen per step (auto_chunks)
  int staged_nq = -1;
  std::vector<void *> d_in, d_out;  // 3+nq each
  cudaStream_t s_in = nullptr, s_k = nullptr, s_out = nullptr;
  cudaEvent_t ev_user = nullptr, ev_in_begin = nullptr, ev_out_begin = nullptr;
  std::vector<cudaEvent_t> ev_h2d, ev_kb, ev_ke, ev_d2h;  // what the host waits on / times (per chunk)
  std::vector<cudaEvent_t> dep_h2d, dep_ke;               // cross-stream dependencies inside a step (per chunk)
  cudaEvent_t dep_join_k = nullptr, dep_join_out = nullptr, ev_done = nullptr;
  // the enqueue of a step with unchanged arguments is captured once into a CUDA graph and replayed
  int use_graph = 1;
  unsigned long epoch = 0;             // bumped by every setter: a graph never outlives a setting
  std::vector<uintptr_t> graph_key;    // arguments + settings of the captured step
  std::vector<uintptr_t> pending_key;  // of the last step that was enqueued eagerly
  cudaGraphExec_t graph_exec = nullptr;
  long graph_launches = 0;             // kernels one replay launches
  std::vector<int> chunk_a, chunk_b;  // interior-relative x ranges of the in-flight step
  bool in_flight = false, have_times = false;
  float times[4] = {0, 0, 0, 0};
};

namespace {

int fail(monc_adv_t h, int code, const std::string &msg) {
  if (h) h->err = msg;
  return code;
}
int cuda_fail(monc_adv_t h, cudaError_t e, const char *what) {
  return fail(h, e == cudaErrorMemoryAllocation ? MONC_ADV_ENOMEM : MONC_ADV_ECUDA,
              std::string(what) + ": " + cudaGetErrorString(e));
}
#define CU(call)                                              \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ != cudaSuccess) return cuda_fail(h, e_, #call);    \
  } while (0)

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// two arrays of `bytes` bytes each share at least one byte
bool ranges_overlap(const void *a, const void *b, size_t bytes) {
  const uintptr_t x = reinterpret_cast<uintptr_t>(a), y = reinterpret_cast<uintptr_t>(b);
  return x < y ? y - x < bytes : x - y < bytes;
}
// first (input, output) or (output, output) pair of whole-field arrays that overlap
const char *find_alias(const std::vector<const void *> &ins, const std::vector<const void *> &outs,
                       size_t bytes) {
  for (size_t b = 0; b < outs.size(); ++b) {
    for (const void *a : ins)
      if (ranges_overlap(a, outs[b], bytes)) return "inputs and outputs must not overlap";
    for (size_t c = 0; c < b; ++c)
      if (ranges_overlap(outs[c], outs[b], bytes)) return "outputs must not overlap each other";
  }
  return nullptr;
}
// host memory the copy engines can read asynchronously: page-locked (cudaMallocHost,
// cudaHostRegister) or managed, over the whole array.  Pageable memory would make
// every "asynchronous" copy a synchronous staged one -- the silent fallback PAPER.md:95
// ran into -- so it is refused.
bool is_pinned_host(const void *p, size_t bytes) {
  for (const char *q : {(const char *)p, (const char *)p + bytes - 1}) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, q) != cudaSuccess) {
      cudaGetLastError();
      return false;
    }
    if (at.type != cudaMemoryTypeHost && at.type != cudaMemoryTypeManaged) return false;
  }
  return true;
}

template <typename T>
KParams<T> make_params(monc_adv_t h, int ia, int ib) {
  KParams<T> p;
  p.nx = h->nx; p.ny = h->ny; p.nz = h->nz; p.h = h->h;
  p.nyh = h->nyh;
  p.plane = (long long)h->nyh * h->nz;
  p.ia = ia; p.ib = ib;
  constexpr int NK = VecOf<T>::NK;
  p.colgroup = std::max(1, h->colgroup);
  p.l2hint = h->l2hint;
  p.wzc = (h->nz / NK + 31) / 32;
  p.units = h->ny * p.wzc;
  p.xc = ib - ia;
  p.accumulate = h->accumulate;
  p.skew = h->form == MONC_ADV_FORM_PW_SKEW;
  p.prefetch = h->prefetch < 0 ? 0 : (h->prefetch == 0 ? kDefaultPrefetch : h->prefetch);
  p.work = h->work;
  p.zero = (T)h->zero;
  p.cx = (T)(1.0 / (4.0 * h->dx));
  p.cy = (T)(1.0 / (4.0 * h->dy));
  p.tzc1 = (const T *)h->d_tz[0]; p.tzc2 = (const T *)h->d_tz[1];
  p.tzd1 = (const T *)h->d_tz[2]; p.tzd2 = (const T *)h->d_tz[3];
  return p;
}

// march kernels need whole 16-byte vectors per column and the flux form
template <typename T>
bool use_march(monc_adv_t h) {
  if (h->variant == 1) return false;
  if (h->form != MONC_ADV_FORM_FLUX) return false;
  return h->nz % VecOf<T>::NK == 0;
}

// planes per block: enough blocks to fill the chip about `waves` times
int pick_xchunk(monc_adv_t h, int nplanes, int blocks_per_plane, int resident_per_sm,
                int multiplicity) {
  if (h->xchunk > 0) return std::min(h->xchunk, nplanes);
  const long slots = (long)h->sm_count * resident_per_sm;
  long want = std::max<long>(1, slots / std::max(1, blocks_per_plane * multiplicity));
  int xc = (int)((nplanes + want - 1) / want);
  xc = std::max(xc, std::min(nplanes, 16));
  return std::min(xc, nplanes);
}

// How many block-times a launch of `blocks` equal blocks (one resident per SM)
// takes.  Measured on B200: a GPC sustains about 16 SMs' worth
// of these streaming kernels.  Up to 8 x 16 = 128 blocks run at the full per-SM
// rate; a single static wave of 129..148 blocks is as slow as its fullest GPC
// (20 SMs on 16 SMs' worth of bandwidth: 1.27 x at 148 blocks).  Several waves of
// short blocks are balanced dynamically: about 1.12 block-times per 148 blocks,
// plus half a block-time for the ragged end.  A single wave that leaves SMs idle
// is charged for them (0.93 x SMs / blocks): under the board's power cap the SM
// clock drops and the per-SM rate, not DRAM, bounds the launch (config 2 momentum,
// 128 blocks x 512 planes against 1024 x 64: 4 % faster in a burst, 6 % slower
// sustained).
double launch_rounds(long blocks, int sm_count) {
  const long full_rate = std::max(1L, (long)sm_count * 128 / 148);
  auto gpc_wave = [&](long b) {
    return b <= full_rate ? 1.0 : 1.0 + 0.27 * (double)(b - full_rate) / (double)(sm_count - full_rate);
  };
  if (blocks <= sm_count) return std::max(gpc_wave(blocks), 0.93 * (double)sm_count / (double)std::max(1L, blocks));
  if (blocks < 2L * sm_count) return 1.12 + gpc_wave(blocks - sm_count);  // a full wave, then a static partial one
  return 1.12 * (double)blocks / (double)sm_count + 0.5;
}

template <typename T>
TmaPlan compute_plan_tma(monc_adv_t h, int nplanes, int fields_per_stage) {
  TmaPlan pl;
  constexpr int NK = VecOf<T>::NK;
  if (h->nz % NK != 0) return pl;
  const int wzc = (h->nz / NK + 31) / 32;
  const int max_warps = tma_momentum_max_warps(h->accumulate != 0 || h->work > 1);
  if (wzc > max_warps) return pl;
  const int tymax = std::min(h->ny, max_warps / wzc);
  const size_t budget = (size_t)std::min(h->smem_optin, 227 * 1024) - 1024;
  const int ty_hi = h->tile_y > 0 ? std::min(h->tile_y, tymax) : tymax;
  const int ty_lo = h->tile_y > 0 ? ty_hi : std::max(1, tymax - 3);
  const int nch_fixed = h->xchunk > 0 ? (nplanes + h->xchunk - 1) / h->xchunk : 0;
  double best = 1e300;
  for (int ty = ty_hi; ty >= ty_lo; --ty) {
    const size_t stage = (size_t)fields_per_stage * (ty + 2) * h->nz * sizeof(T);
    int S = (int)std::min<size_t>(8, budget / (stage + 16));
    // accumulate: every step waits for the old tendencies of its plane (a read-modify-write the ring
    // cannot stage); what hides that latency is many short blocks over several waves and a ring that
    // does not run far ahead of the L2 prefetch of those lines (config 1: 5980 GB/s of real traffic at
    // 4 stages and 16 planes per block against 2690 with the overwriting launch's geometry)
    const bool acc = h->accumulate != 0;
    if (acc) S = std::min(S, 4);
    if (h->stages > 0) S = std::min(S, h->stages);
    if (S < 3) continue;
    const int tiles = (h->ny + ty - 1) / ty;
    // at least four waves of blocks, of at least 8 planes each
    const int nch_acc = std::max(1, std::min((4 * h->sm_count + tiles - 1) / tiles, nplanes / 8));
    const int nch_lo = nch_fixed ? nch_fixed : (acc ? nch_acc : 1);
    const int nch_hi = nch_fixed ? nch_fixed : std::max(nch_lo, nplanes / 4);
    for (int nch = nch_lo; nch <= nch_hi; ++nch) {
      const int xc = (nplanes + nch - 1) / nch;
      const long blocks = (long)tiles * ((nplanes + xc - 1) / xc);
      // time ~ block-times of the launch * (columns per block + the L2/shared-memory
      // cost of its two halo columns) * (planes per block + its two halo planes + the
      // ramp of a deep ring)
      const double rounds = launch_rounds(blocks, h->sm_count);
      const double march = 1.0 + 0.1 * std::min(xc, 256) / 256.0;  // y neighbours drift apart
      const double cost = rounds * (ty + 0.7) * (xc + 4) * (1.0 + 0.02 * (tymax - ty)) * march;
      if (cost < best) {
        best = cost;
        pl.ok = true; pl.ty = ty; pl.stages = S; pl.xc = xc; pl.tiles = tiles;
        pl.nchunks = (nplanes + xc - 1) / xc;
        pl.smem = (size_t)S * (stage + 16);
      }
    }
  }
  if (pl.ok) {
    // a single wave is placed 4 y-neighbour blocks at a time: 16 (or 20) blocks per GPC instead
    // of whatever the block scheduler deals out, +2 % at config 1; several
    // waves gain nothing from it (and clusters of 8 leave most of a GPC idle)
    const bool one_wave = (long)pl.tiles * pl.nchunks <= h->sm_count;
    const int want = h->cluster > 0 ? h->cluster : (one_wave ? kDefaultClusterMomentum : 1);
    pl.cl = std::max(1, std::min(want, pl.tiles));
  }
  return pl;
}

// plans depend on the handle's sizes and tuning knobs and on the call's plane
// count only: computed once, kept on the handle (dropped by set_tuning)
template <typename T>
const TmaPlan &plan_tma(monc_adv_t h, int nplanes) {
  auto it = h->mom_plans.find(nplanes);
  if (it == h->mom_plans.end()) it = h->mom_plans.emplace(nplanes, compute_plan_tma<T>(h, nplanes, 3)).first;
  return it->second;
}

// The dynamic shared-memory limit of a kernel is raised ONCE per device to the
// opt-in maximum (the attribute is per context: setting the exact size of each
// plan before each launch would let two handles lower each other's limit).
template <typename K>
cudaError_t allow_max_smem(monc_adv_t h, K kernel) {
  static std::mutex mu;
  static std::set<std::pair<int, const void *>> done;
  std::lock_guard<std::mutex> lock(mu);
  const auto key = std::make_pair(h->device, reinterpret_cast<const void *>(kernel));
  if (done.count(key)) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin);
  if (e == cudaSuccess) done.insert(key);
  return e;
}

// Launch with the programmatic stream-serialisation attribute (PDL): the kernel
// may begin (barrier set-up, coefficient loads) while its predecessor in the
// stream drains; it calls griddepcontrol.wait before touching any field.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(monc_adv_t h, void (*kernel)(KArgs...), dim3 grid, int cluster, int threads, size_t smem,
                       cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = dim3((unsigned)threads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = h->pdl ? 1 : 0;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (cluster > 1) {
    // `cluster` consecutive blocks in x (y-neighbour tiles) run together on one GPC
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = (unsigned)cluster;
    attr[1].val.clusterDim.y = 1;
    attr[1].val.clusterDim.z = 1;
    cfg.numAttrs = 2;
  }
  cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
  if (e != cudaSuccess && cluster > 1 && e != cudaErrorInvalidResourceHandle) {
    // clusters are a placement hint only (no kernel uses distributed shared memory): if this
    // device or partition cannot co-schedule them, launch the same grid without
    cudaGetLastError();
    cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
  }
  return e;
}

template <typename T>
int run_tma_scalars(monc_adv_t h, KParams<T> p, const T *u, const T *v, const T *w, const void *const *q,
                    void *const *sq, int nq, int ia, int ib, cudaStream_t st, bool *done,
                    const MomPtrs<T> *mo = nullptr);

template <typename T>
int launch_momentum(monc_adv_t h, const T *u, const T *v, const T *w, T *su, T *sv, T *sw,
                    int ia, int ib, cudaStream_t st) {
  if (ib <= ia) return MONC_ADV_OK;
  KParams<T> p = make_params<T>(h, ia, ib);
  TmaPlan pl;
  if (h->variant == 3 || h->variant == 0) pl = plan_tma<T>(h, ib - ia);
  if (h->work > 1 && !pl.ok) return fail(h, MONC_ADV_EINVAL, "momentum: work scaling needs the TMA kernels");
  if (pl.ok) {
    p.xc = pl.xc;
    dim3 grid((pl.tiles + pl.cl - 1) / pl.cl * pl.cl, pl.nchunks);  // padded to whole clusters: the extra blocks exit
    auto go = [&](auto kernel) -> int {
      CU(allow_max_smem(h, kernel));
      if (pl.cl > 1 && h->cluster == 0 && !pl.cl_checked) {
        // the default clusters are worth it only if every cluster of the (padded) grid is resident at
        // once: a GPC of 18 SMs holds 4 clusters of 4, and clusters left over run as a second wave
        // (config 1 with 37 y tiles: 3460 GB/s in clusters of 4 against 5650 without)
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grid;
        cfg.blockDim = dim3((unsigned)(pl.ty * p.wzc * 32));
        cfg.dynamicSmemBytes = pl.smem;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = (unsigned)pl.cl;
        attr[0].val.clusterDim.y = attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        int resident = 0;
        if (cudaOccupancyMaxActiveClusters(&resident, kernel, &cfg) != cudaSuccess) {
          cudaGetLastError();
          resident = 0;
        }
        if ((long)grid.x / pl.cl * grid.y > resident) {
          pl.cl = 1;
          grid.x = (unsigned)pl.tiles;
        }
        TmaPlan &kept = h->mom_plans[ib - ia];  // remembered: the query runs once per plan
        kept.cl = pl.cl;
        kept.cl_checked = true;
      }
      CU(launch_pdl(h, kernel, grid, pl.cl, pl.ty * p.wzc * 32, pl.smem, st, p, pl.ty, pl.stages, u, v, w, su, sv, sw));
      return MONC_ADV_OK;
    };
    const bool skew = h->form == MONC_ADV_FORM_PW_SKEW;
    const int rc = h->work > 1 ? go(tma_momentum<T, false, false, true>)  // checked by work_scale_ok: flux, overwrite
                   : h->accumulate ? (skew ? go(tma_momentum<T, true, true>) : go(tma_momentum<T, true, false>))
                                   : (skew ? go(tma_momentum<T, false, true>) : go(tma_momentum<T, false, false>));
    if (rc != MONC_ADV_OK) return rc;
    char b[160];
    snprintf(b, sizeof b, "tma_momentum ty=%d stages=%d xc=%d grid=%dx%d cluster=%d threads=%d smem=%zu", pl.ty,
             pl.stages, pl.xc, (int)grid.x, pl.nchunks, pl.cl, pl.ty * p.wzc * 32, pl.smem);
    h->plan_mom = b;
  } else {
    if (h->colgroup >= 1 && (h->variant == 0 || h->variant == 3)) {
      // tma_momentum's 1-D bulk copies need whole vectors per column and at most 16 warps per
      // column; the momentum role of the tensor-map kernel, run without scalar warps, takes a
      // ragged nz and columns of any height (z tiles)
      bool done = false;
      const MomPtrs<T> mo{su, sv, sw};
      const int rc = run_tma_scalars<T>(h, p, u, v, w, nullptr, nullptr, 0, ia, ib, st, &done, &mo);
      if (rc != MONC_ADV_OK || done) return rc;
    }
    if (h->variant == 3) return fail(h, MONC_ADV_EINVAL, "momentum: TMA variant does not fit this shape");
    if (use_march<T>(h)) {
      const int wpb = h->warps > 0 ? h->warps : kWarpsPerBlock;
      const int bx = (p.units + wpb - 1) / wpb;
      p.xc = pick_xchunk(h, ib - ia, bx, 16 / wpb, 1);
      dim3 grid(bx, (ib - ia + p.xc - 1) / p.xc);
      if (p.wzc > 1)
        march_momentum<T, true><<<grid, wpb * 32, 0, st>>>(p, u, v, w, su, sv, sw);
      else
        march_momentum<T, false><<<grid, wpb * 32, 0, st>>>(p, u, v, w, su, sv, sw);
      h->plan_mom = "march_momentum xc=" + std::to_string(p.xc);
    } else {
      h->plan_mom = "generic_momentum";
      const long long n = (long long)(ib - ia) * h->ny * h->nz;
      generic_momentum<T><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p, u, v, w, su, sv, sw);
    }
  }
  CU(cudaGetLastError());
  h->launches++;
  return MONC_ADV_OK;
}

// ---- tensor-map encoder, fetched from the driver at first use (no -lcuda link)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                  const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn tensor_map_encoder() {
  static EncodeTiledFn fn = []() -> EncodeTiledFn {
    void *sym = nullptr;
    cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess) {
      cudaGetLastError();
      return nullptr;
    }
    return reinterpret_cast<EncodeTiledFn>(sym);
  }();
  return fn;
}

// descriptor of one field F[NXH][NYH][nz] with a (z, y, x) box of box_z x box_y x 1
// (colgroup G > 1, ragged nz: G columns per row of the view, a box holds the rows of one class of
// columns j mod G of the tile; tma_scalars' producer)
template <typename T>
bool encode_field_map(monc_adv_t h, CUtensorMap *m, const void *base, int box_z, int box_y) {
  EncodeTiledFn enc = tensor_map_encoder();
  if (!enc) return false;
  const int G = std::max(1, h->colgroup);
  const cuuint64_t gdim[3] = {(cuuint64_t)G * h->nz, (cuuint64_t)(h->nyh / G), (cuuint64_t)h->nxh};
  const cuuint64_t gstr[2] = {(cuuint64_t)G * h->nz * sizeof(T), (cuuint64_t)h->nyh * h->nz * sizeof(T)};
  const cuuint32_t box[3] = {(cuuint32_t)box_z, (cuuint32_t)(G > 1 ? ragged_class_rows(box_y, G) : box_y), 1u};
  const cuuint32_t estr[3] = {1u, 1u, 1u};
  const CUtensorMapDataType dt =
      sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
  return enc(m, dt, 3, const_cast<void *>(base), gdim, gstr, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
             CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <typename T>
TmaScalarPlan compute_plan_tma_scalars(monc_adv_t h, int nplanes, int n, bool mom) {
  TmaScalarPlan pl;
  constexpr int NK = VecOf<T>::NK;
  if (h->colgroup == 0 || (!h->plan_only && !tensor_map_encoder())) return pl;
  if (n == 0 && !mom) return pl;
  const size_t budget = (size_t)std::min(h->smem_optin, 227 * 1024) - 1024;
  const int nch_fixed = h->xchunk > 0 ? (nplanes + h->xchunk - 1) / h->xchunk : 0;
  double best = 1e300;
  // Cost model, calibrated on B200:
  // a block step (one plane) takes max(DRAM time of its bytes at this SM's share
  // of HBM bandwidth, the serial time of one warp's gw scalars), stretched when
  // the ring has only two stages, plus a fixed synchronisation cost; a launch takes
  // waves * (planes per block + 4) steps.
  const double sm_gbs = 6200.0 / h->sm_count;
  // n = 0 (momentum only through the momentum role: ragged nz, where tma_momentum's 1-D bulk
  // copies cannot be used): no scalar warps, gb = ss = 0
  for (int gb = std::min(n, 10); gb >= (n == 0 ? 0 : 1); --gb) {
    if (h->group > 0 && gb != std::min(h->group, std::min(n, 10))) continue;
    if (h->group == 0 && gb != std::min(n, 5) && gb != std::min(n, 10)) continue;
    const int ngroups = gb == 0 ? 1 : (n + gb - 1) / gb;
    if (mom && ngroups != 1) continue;  // the momentum role runs once: one group holds every scalar
    for (int ss = (gb == 0 ? 0 : 1); ss <= std::min(gb, 4); ++ss) {
      if (gb > 0 && h->split > 0 && ss != std::min(h->split, std::min(gb, 4))) continue;
      const int gw = gb == 0 ? 1 : (gb + ss - 1) / ss;
      if (gw > 5) continue;
      {
        // one 32-vector z chunk per block tile: the row stride is a compile-time constant
        const int ZB = 32 * NK;
        const int nzt = scalar_z_tiles(h->nz, NK, h->colgroup, h->nz % NK != 0);
        // the momentum role alone (gb = 0) is a chain of dependent steps per warp: two blocks of 7
        // columns and a 4-stage ring per SM hide its latency better than one block of 15 columns and
        // a deep ring (256^2 x 127 fp64: 4350 against 3790 GB/s)
        const int tymax = std::min(h->ny, gb == 0 ? 7 : kScalarConsumerWarps / (ss + (mom ? 1 : 0)));
        if (tymax < 1) continue;
        for (int ty = tymax; ty >= 1; --ty) {
          if (h->tile_y > 0 && ty != std::min(h->tile_y, tymax)) continue;
          const size_t field = (size_t)scalar_field_bytes(ty + 2, h->colgroup, h->nz % NK != 0);
          const size_t stage = (size_t)(3 + gb) * field;
          int S = (int)std::min<size_t>(gb == 0 ? 4 : 8, budget / (stage + 16));
          if (h->stages > 0) S = std::min(S, h->stages);
          if (S < (mom ? 3 : 2)) continue;
          const int tiles = ((h->ny + ty - 1) / ty) * nzt * ngroups;
          // the groups after the first re-read the wind; about half of that hits L2
          const double wind = 3.0 * (1.0 + 0.5 * (ngroups - 1)) / ngroups;
          // inputs: the two halo rows of a tile are re-reads; about 30 % of them miss L2
          // (neighbouring blocks drift apart), fewer per byte in a taller tile
          const double dram_b = ((wind + gb) * (1.0 + 0.6 / ty) + gb + (mom ? 3 : 0)) * ty * ZB * sizeof(T);
          const double t_mem = dram_b / (sm_gbs * 1e3);                            // us
          const double t_warp = std::max(0.15 + 0.25 * gw, mom ? 1.2 : 0.0);         // us; momentum ~ 4 scalars
          const double shallow = S >= 3 ? 1.0 : 1.15;
          const double t_step = std::max(t_mem, t_warp) * shallow + 0.05;
          const int nch_lo = nch_fixed ? nch_fixed : 1;
          const int nch_hi = nch_fixed ? nch_fixed : std::max(1, nplanes / 8);
          for (int nch = nch_lo; nch <= nch_hi; ++nch) {
            const int xc = (nplanes + nch - 1) / nch;
            const long blocks = (long)tiles * ((nplanes + xc - 1) / xc);
            const double waves = launch_rounds(blocks, h->sm_count);
            // +2 halo planes, ~1-2 steps of start-up latency; on a long march the y/z
            // neighbours drift apart (the SMs of a full GPC get less bandwidth each) and
            // their halo re-reads miss L2: config 2 fused, DRAM reads 7.95 GB at xc = 103
            // against 7.09 GB algorithmic; 5 % faster at xc = 32..52
            const double march = 1.0 + 0.0007 * std::min(xc, 512);
            const double cost = waves * (xc + (waves <= 1.3 ? 4 : 3)) * t_step * march;
            if (cost < best) {
              best = cost;
              pl.ok = true; pl.ty = ty; pl.ss = ss; pl.gb = gb; pl.gw = gw; pl.stages = S;
              pl.xc = xc; pl.tiles = tiles;
              pl.nchunks = (nplanes + xc - 1) / xc;
              pl.fieldsz = (int)(field / sizeof(T));
              pl.smem = (size_t)S * (stage + 16);
            }
          }
        }
      }
    }
  }
  if (pl.ok && (pl.gb == 0 || (n + pl.gb - 1) / pl.gb == 1)) {
    // one scalar group: cl y-neighbour tiles (same z tile) form a thread-block cluster; the
    // tile count is padded to whole clusters (the extra blocks exit at once)
    const int nzt = scalar_z_tiles(h->nz, NK, h->colgroup, h->nz % NK != 0), nyt = (h->ny + pl.ty - 1) / pl.ty;
    pl.cl = std::max(1, std::min(h->cluster > 0 ? h->cluster : kDefaultClusterScalars, nyt));
    pl.tiles = (nyt + pl.cl - 1) / pl.cl * pl.cl * nzt;
  }
  return pl;
}

template <typename T>
const TmaScalarPlan &plan_tma_scalars(monc_adv_t h, int nplanes, int n, bool mom) {
  const auto key = std::make_tuple(nplanes, n, mom ? 1 : 0);
  auto it = h->sca_plans.find(key);
  if (it == h->sca_plans.end())
    it = h->sca_plans.emplace(key, compute_plan_tma_scalars<T>(h, nplanes, n, mom)).first;
  return it->second;
}

// Tensor-map descriptors for (u, v, w, q[0..n)) with ty+2 rows per box: encoded
// when first seen, then reused (at most kMapCacheEntries sets, least recently
// used replaced).  Unused slots of the launch repeat the first scalar.
constexpr size_t kMapCacheEntries = 8;
template <typename T>
const TensorMaps *field_maps(monc_adv_t h, const T *u, const T *v, const T *w, const void *const *q, int n,
                             int ty) {
  std::vector<const void *> ptrs = {u, v, w};
  for (int s = 0; s < n; ++s) ptrs.push_back(q[s]);  // (n = 0: q may be NULL)
  for (MapEntry &e : h->map_cache)
    if (e.ty == ty && e.ptrs == ptrs) {
      e.stamp = ++h->map_clock;
      return &e.maps;
    }
  MapEntry *slot = nullptr;
  if (h->map_cache.size() < kMapCacheEntries) {
    h->map_cache.reserve(kMapCacheEntries);
    h->map_cache.emplace_back();
    slot = &h->map_cache.back();
  } else {
    slot = &h->map_cache[0];
    for (MapEntry &e : h->map_cache)
      if (e.stamp < slot->stamp) slot = &e;
  }
  const int RS = kRowBytes / (int)sizeof(T);
  bool ok = true;
  for (int f = 0; f < 3 + kMaxScalarsPerLaunch; ++f) {
    const void *base = f < 3 + n ? ptrs[f] : ptrs[n > 0 ? 3 : 0];
    ok = ok && encode_field_map<T>(h, &slot->maps.m[f], base, RS, ty + 2);
  }
  if (!ok) {
    slot->ptrs.clear();
    slot->stamp = 0;
    return nullptr;
  }
  slot->ptrs = std::move(ptrs);
  slot->ty = ty;
  slot->stamp = ++h->map_clock;
  return &slot->maps;
}

template <typename T, int GW, bool ACC, bool SKEW, bool MOM, bool WS = false, bool RAG = false>
int launch_tma_scalars_k(monc_adv_t h, const KParams<T> &p, const TensorMaps &maps, const SqPtrs<T> &outs,
                         const MomPtrs<T> &mo, int nq, const TmaScalarPlan &pl, cudaStream_t st) {
  CU(allow_max_smem(h, tma_scalars<T, GW, ACC, SKEW, MOM, WS, RAG>));
  dim3 grid(pl.tiles, pl.nchunks);
  const int threads = (pl.ty * (pl.ss + (MOM ? 1 : 0)) + 1) * 32;  // consumers + the producer warp
  CU(launch_pdl(h, tma_scalars<T, GW, ACC, SKEW, MOM, WS, RAG>, grid, pl.cl, threads, pl.smem, st, p, maps, outs, mo, nq,
                pl.gb == 0 ? 1 : (nq + pl.gb - 1) / pl.gb, pl.gb, pl.ty, pl.ss, pl.stages, pl.fieldsz, pl.cl));
  return MONC_ADV_OK;
}

template <typename T, int GW, bool MOM>
int launch_tma_scalars_m(monc_adv_t h, const KParams<T> &p, const TensorMaps &maps, const SqPtrs<T> &outs,
                         const MomPtrs<T> &mo, int nq, const TmaScalarPlan &pl, cudaStream_t st) {
  const bool skew = h->form == MONC_ADV_FORM_PW_SKEW;
  if (h->nz % VecOf<T>::NK != 0) {
    // ragged nz: the RAG instantiations (levels shifted against the vectors, neighbour rows
    // read element by element)
    if (h->work > 1) return fail(h, MONC_ADV_EINVAL, "work scaling needs nz to be a whole number of 16-byte vectors");
    if (h->accumulate)
      return skew ? launch_tma_scalars_k<T, GW, true, true, MOM, false, true>(h, p, maps, outs, mo, nq, pl, st)
                  : launch_tma_scalars_k<T, GW, true, false, MOM, false, true>(h, p, maps, outs, mo, nq, pl, st);
    return skew ? launch_tma_scalars_k<T, GW, false, true, MOM, false, true>(h, p, maps, outs, mo, nq, pl, st)
                : launch_tma_scalars_k<T, GW, false, false, MOM, false, true>(h, p, maps, outs, mo, nq, pl, st);
  }
  if (h->work > 1)  // checked by work_scale_ok: flux form, overwrite
    return launch_tma_scalars_k<T, GW, false, false, MOM, true>(h, p, maps, outs, mo, nq, pl, st);
  if (h->accumulate)
    return skew ? launch_tma_scalars_k<T, GW, true, true, MOM>(h, p, maps, outs, mo, nq, pl, st)
                : launch_tma_scalars_k<T, GW, true, false, MOM>(h, p, maps, outs, mo, nq, pl, st);
  return skew ? launch_tma_scalars_k<T, GW, false, true, MOM>(h, p, maps, outs, mo, nq, pl, st)
              : launch_tma_scalars_k<T, GW, false, false, MOM>(h, p, maps, outs, mo, nq, pl, st);
}

template <typename T, int GW>
int launch_tma_scalars(monc_adv_t h, const KParams<T> &p, const TensorMaps &maps, const SqPtrs<T> &outs,
                       const MomPtrs<T> *mo, int nq, const TmaScalarPlan &pl, cudaStream_t st) {
  if (mo) return launch_tma_scalars_m<T, GW, true>(h, p, maps, outs, *mo, nq, pl, st);
  return launch_tma_scalars_m<T, GW, false>(h, p, maps, outs, MomPtrs<T>{nullptr, nullptr, nullptr}, nq, pl, st);
}

// One launch of tma_scalars per kMaxScalarsPerLaunch scalars.  *done = false
// with MONC_ADV_OK means "does not fit, nothing launched": the caller falls back.
// mo != nullptr: the fused launch (momentum role included); it needs every
// scalar in ONE group of one launch, otherwise nothing is launched.
template <typename T>
int run_tma_scalars(monc_adv_t h, KParams<T> p, const T *u, const T *v, const T *w,
                    const void *const *q, void *const *sq, int nq, int ia, int ib,
                    cudaStream_t st, bool *done, const MomPtrs<T> *mo) {
  *done = false;
  if (mo && nq > 10) return MONC_ADV_OK;
  if (nq == 0 && !mo) return MONC_ADV_OK;
  // (nq = 0 with mo: one launch of the momentum role alone)
  for (int base = 0; base < std::max(nq, 1); base += kMaxScalarsPerLaunch) {
    const int n = std::min(kMaxScalarsPerLaunch, nq - base);
    const TmaScalarPlan &pl = plan_tma_scalars<T>(h, ib - ia, n, mo != nullptr);
    if (!pl.ok) {
      if (base == 0) return MONC_ADV_OK;
      return fail(h, MONC_ADV_ECUDA, "scalars: TMA plan failed after a partial launch");
    }
    const TensorMaps *mp = field_maps<T>(h, u, v, w, n > 0 ? q + base : nullptr, n, pl.ty);
    if (!mp) return fail(h, MONC_ADV_ECUDA, "scalars: cuTensorMapEncodeTiled failed");
    const TensorMaps &maps = *mp;
    SqPtrs<T> outs;
    for (int s = 0; s < kMaxScalarsPerLaunch; ++s) outs.sq[s] = n > 0 ? (T *)sq[base + (s < n ? s : 0)] : nullptr;
    p.xc = pl.xc;
    int rc = MONC_ADV_OK;
    switch (pl.gw) {
      case 1: rc = launch_tma_scalars<T, 1>(h, p, maps, outs, mo, n, pl, st); break;
      case 2: rc = launch_tma_scalars<T, 2>(h, p, maps, outs, mo, n, pl, st); break;
      case 3: rc = launch_tma_scalars<T, 3>(h, p, maps, outs, mo, n, pl, st); break;
      case 4: rc = launch_tma_scalars<T, 4>(h, p, maps, outs, mo, n, pl, st); break;
      default: rc = launch_tma_scalars<T, 5>(h, p, maps, outs, mo, n, pl, st); break;
    }
    if (rc != MONC_ADV_OK) return rc;
    CU(cudaGetLastError());
    h->launches++;
    char b[200];
    snprintf(b, sizeof b, "%s group=%d per_warp=%d split=%d ty=%d stages=%d xc=%d grid=%dx%d cluster=%d "
             "colgroup=%d threads=%d smem=%zu",
             mo ? (n > 0 ? "tma_fused(momentum+scalars)" : "tma_fused(momentum role only)") : "tma_scalars", pl.gb,
             pl.gw, pl.ss, pl.ty, pl.stages, pl.xc, pl.tiles, pl.nchunks, pl.cl, std::max(1, h->colgroup),
             (pl.ty * (pl.ss + (mo ? 1 : 0)) + 1) * 32, pl.smem);
    h->plan_sca = b;
    if (mo) h->plan_mom.clear();
  }
  *done = true;
  return MONC_ADV_OK;
}

template <typename T, int G>
void launch_march_scalars(const KParams<T> &p, const ScalarPtrs<T> &ptrs, int nq, dim3 grid,
                          int wpb, int ngroups, const T *u, const T *v, const T *w,
                          cudaStream_t st) {
  march_scalars<T, G><<<grid, wpb * 32, 0, st>>>(p, ptrs, nq, ngroups, u, v, w);
}

template <typename T>
int launch_scalars(monc_adv_t h, const T *u, const T *v, const T *w, const void *const *q,
                   void *const *sq, int nq, int ia, int ib, cudaStream_t st) {
  if (ib <= ia || nq == 0) return MONC_ADV_OK;
  KParams<T> p = make_params<T>(h, ia, ib);
  ScalarPtrs<T> ptrs;
  for (int n = 0; n < kMaxScalars; ++n) {
    ptrs.q[n] = (const T *)q[n < nq ? n : 0];
    ptrs.sq[n] = (T *)sq[n < nq ? n : 0];
  }
  if (h->variant == 3 || h->variant == 0) {
    bool done = false;
    const int rc = run_tma_scalars<T>(h, p, u, v, w, q, sq, nq, ia, ib, st, &done);
    if (rc != MONC_ADV_OK || done) return rc;
  }
  if (h->variant == 3)
    return fail(h, MONC_ADV_EINVAL, "scalars: TMA variant does not fit this nz / form");
  if (h->work > 1) return fail(h, MONC_ADV_EINVAL, "scalars: work scaling needs the TMA kernels");
  if (use_march<T>(h)) {
    int G = h->group > 0 ? std::min(h->group, 5) : (nq >= 5 ? 5 : nq);
    G = std::min(G, nq);
    const int ngroups = (nq + G - 1) / G;
    const int wpb = h->warps > 0 ? h->warps : kWarpsPerBlock;
    const int bx = (p.units + wpb - 1) / wpb;
    p.xc = pick_xchunk(h, ib - ia, bx, 16 / wpb, ngroups);
    dim3 grid(bx * ngroups, (ib - ia + p.xc - 1) / p.xc);
    switch (G) {
      case 1: launch_march_scalars<T, 1>(p, ptrs, nq, grid, wpb, ngroups, u, v, w, st); break;
      case 2: launch_march_scalars<T, 2>(p, ptrs, nq, grid, wpb, ngroups, u, v, w, st); break;
      case 3: launch_march_scalars<T, 3>(p, ptrs, nq, grid, wpb, ngroups, u, v, w, st); break;
      case 4: launch_march_scalars<T, 4>(p, ptrs, nq, grid, wpb, ngroups, u, v, w, st); break;
      default: launch_march_scalars<T, 5>(p, ptrs, nq, grid, wpb, ngroups, u, v, w, st); break;
    }
    h->plan_sca = "march_scalars group=" + std::to_string(G) + " xc=" + std::to_string(p.xc);
  } else {
    h->plan_sca = "generic_scalars";
    const long long n = (long long)(ib - ia) * h->ny * h->nz;
    dim3 grid((unsigned)((n + 255) / 256), nq);
    generic_scalars<T><<<grid, 256, 0, st>>>(p, ptrs, u, v, w);
  }
  CU(cudaGetLastError());
  h->launches++;
  return MONC_ADV_OK;
}

// whole step from device arrays: one fused launch when the plan allows it, else
// the momentum launch followed by the scalars launch
template <typename T>
int launch_tendencies(monc_adv_t h, const T *u, const T *v, const T *w, T *su, T *sv, T *sw,
                      const void *const *q, void *const *sq, int nq, int ia, int ib, cudaStream_t st) {
  if (nq > 0 && h->fuse && (h->variant == 3 || h->variant == 0)) {
    // the fused launch takes one scalar group (10 scalars); further scalars follow in a scalars
    // launch of their own, which re-reads the wind (24 of 24 + 16 n bytes per point)
    KParams<T> p = make_params<T>(h, ia, ib);
    const MomPtrs<T> mo{su, sv, sw};
    const int nfused = std::min(nq, 10);
    bool done = false;
    const int rc = run_tma_scalars<T>(h, p, u, v, w, q, sq, nfused, ia, ib, st, &done, &mo);
    if (rc != MONC_ADV_OK || (done && nfused == nq)) return rc;
    if (done) {
      const std::string fused_plan = h->plan_sca;
      const int rc2 = launch_scalars<T>(h, u, v, w, q + nfused, sq + nfused, nq - nfused, ia, ib, st);
      h->plan_mom = fused_plan;
      return rc2;
    }
  }
  const int rc = launch_momentum<T>(h, u, v, w, su, sv, sw, ia, ib, st);
  if (rc != MONC_ADV_OK || nq == 0) return rc;
  return launch_scalars<T>(h, u, v, w, q, sq, nq, ia, ib, st);
}

int check_handle(monc_adv_t h) {
  if (!h) return MONC_ADV_EINVAL;
  cudaError_t e = cudaSetDevice(h->device);
  if (e != cudaSuccess) return cuda_fail(h, e, "cudaSetDevice");
  return MONC_ADV_OK;
}

void free_staging(monc_adv_t h) {
  for (void *p : h->d_in) if (p) cudaFree(p);
  for (void *p : h->d_out) if (p) cudaFree(p);
  h->d_in.clear();
  h->d_out.clear();
  h->staged_nq = -1;
}

// Chunk count of a hybrid step when the caller did not fix one.  Both copy engines run
// flat out, D2H one chunk behind H2D, so a step takes T (1 + 1/C) + C c: T = the time of
// one direction's bytes on the host link, c = the fixed cost of a chunk (its copies' set-up,
// events, a kernel launch).  Minimum at C = sqrt(T / c).  Measured on B200 / PCIe Gen5 x16
// (DESIGN.md 7.3): both directions at once move 49.5 GB/s each, c = 15 us + 5 us per copy
// (config 4: 212 ms at C = 8, 201 ms at 32..64; config 2: 158 ms at 8, 151 ms at 32; config 1's shape: 8).
int auto_chunks_for(int nx, int nyh, int nz, size_t esize, int nf_in, int nf_out) {
  const double bytes = (double)std::max(nf_in, nf_out) * (double)nx * nyh * nz * (double)esize;
  const double t_ms = bytes / 49.5e6;
  const double c_ms = 0.015 + 0.005 * (nf_in + nf_out);
  // the power of two nearest to sqrt(T / c): equal slabs copy measurably better than ragged
  // ones (config 2: 150.9 ms at C = 32, 156 ms at 31 and 33), and the minimum is flat
  const double want = std::sqrt(t_ms / c_ms);
  int c = 1;
  while (c < 64 && (double)(2 * c) * (2 * c) <= want * want * 2.0) c *= 2;  // 2c <= want * sqrt(2)
  while (c > nx) c /= 2;
  return std::max(1, c);
}
int auto_chunks(monc_adv_t h, int nf_in, int nf_out) {
  return auto_chunks_for(h->nx, h->nyh, h->nz, h->esize, nf_in, nf_out);
}
int step_chunks(monc_adv_t h, int nf_in, int nf_out) {
  return h->nchunks > 0 ? std::min(h->nchunks, h->nx) : auto_chunks(h, nf_in, nf_out);
}

int ensure_async_objects(monc_adv_t h, int nq, int nchunks) {
  if (!h->s_in) {
    CU(cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking));
    CU(cudaStreamCreateWithFlags(&h->s_k, cudaStreamNonBlocking));
    CU(cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&h->ev_user, cudaEventDisableTiming));
    CU(cudaEventCreate(&h->ev_in_begin));
    CU(cudaEventCreate(&h->ev_out_begin));
    CU(cudaEventCreateWithFlags(&h->dep_join_k, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&h->dep_join_out, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&h->ev_done, cudaEventDisableTiming));
  }
  while ((int)h->ev_h2d.size() < nchunks) {
    cudaEvent_t a, b, c, d;
    CU(cudaEventCreate(&a)); CU(cudaEventCreate(&b));
    CU(cudaEventCreate(&c)); CU(cudaEventCreate(&d));
    h->ev_h2d.push_back(a); h->ev_kb.push_back(b);
    h->ev_ke.push_back(c); h->ev_d2h.push_back(d);
    CU(cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
    h->dep_h2d.push_back(a); h->dep_ke.push_back(b);
  }
  if (h->staged_nq < nq) {
    // grow: keep what exists, add the missing scalar buffers
    const int have = h->staged_nq < 0 ? 0 : 3 + h->staged_nq;
    const int want = 3 + nq;
    h->d_in.resize(want, nullptr);
    h->d_out.resize(want, nullptr);
    const size_t bytes = h->elems * h->esize;
    for (int n = have; n < want; ++n) {
      cudaError_t e = cudaMalloc(&h->d_in[n], bytes);
      if (e == cudaSuccess) e = cudaMalloc(&h->d_out[n], bytes);
      if (e != cudaSuccess) {
        cudaGetLastError();
        free_staging(h);
        return cuda_fail(h, e, "cudaMalloc(staging)");
      }
      // output halos are never written by kernels: define them once
      CU(cudaMemset(h->d_out[n], 0, bytes));
      // input planes beyond halo depth 1 are never copied: define them once
      CU(cudaMemset(h->d_in[n], 0, bytes));
    }
    // the memsets run on the legacy default stream, which the internal (non-blocking)
    // streams do not order against: finish them before any copy or kernel is queued
    CU(cudaDeviceSynchronize());
    h->staged_nq = nq;
  }
  return MONC_ADV_OK;
}

// wait for whatever a failed enqueue left on the internal streams, so that the
// caller's buffers are quiescent and the handle can be used again
void drain_internal_streams(monc_adv_t h) {
  if (h->s_in) cudaStreamSynchronize(h->s_in);
  if (h->s_k) cudaStreamSynchronize(h->s_k);
  if (h->s_out) cudaStreamSynchronize(h->s_out);
  cudaGetLastError();
}

template <typename T>
int step_async_impl(monc_adv_t h, const void *hu, const void *hv, const void *hw,
                    const void *const *hq, int nq, void *hsu, void *hsv, void *hsw,
                    void *const *hsq, bool capture) {
  // capture = the calls below are being captured into a CUDA graph (s_in is the origin
  // stream): events the host waits on or times are then recorded as external event nodes
  // (they fire at every replay), the cross-stream dependencies as ordinary captured events
  auto host_event = [&](cudaEvent_t ev, cudaStream_t st) {
    return capture ? cudaEventRecordWithFlags(ev, st, cudaEventRecordExternal) : cudaEventRecord(ev, st);
  };
  const bool mom = hsu != nullptr;
  const int C = step_chunks(h, 3 + nq, ((mom ? 3 : 0) + nq) * (h->accumulate ? 2 : 1));
  const size_t es = sizeof(T);
  const size_t plane_b = (size_t)h->nyh * h->nz * es;
  const int nf = 3 + nq;
  std::vector<const char *> hin(nf);
  std::vector<char *> hout(nf);
  hin[0] = (const char *)hu; hin[1] = (const char *)hv; hin[2] = (const char *)hw;
  hout[0] = (char *)hsu; hout[1] = (char *)hsv; hout[2] = (char *)hsw;
  for (int n = 0; n < nq; ++n) { hin[3 + n] = (const char *)hq[n]; hout[3 + n] = (char *)hsq[n]; }

  cudaStream_t sin = h->s_in;
  cudaStream_t sk = h->overlap ? h->s_k : h->s_in;
  cudaStream_t sout = h->overlap ? h->s_out : h->s_in;

  h->chunk_a.assign(C, 0);
  h->chunk_b.assign(C, 0);
  for (int c = 0; c < C; ++c) {
    h->chunk_a[c] = (int)((long long)h->nx * c / C);
    h->chunk_b[c] = (int)((long long)h->nx * (c + 1) / C);
  }
  const T *du = (const T *)h->d_in[0], *dv = (const T *)h->d_in[1], *dw = (const T *)h->d_in[2];
  std::vector<const void *> dq(std::max(nq, 1));
  std::vector<void *> dsq(std::max(nq, 1));
  for (int n = 0; n < nq; ++n) { dq[n] = h->d_in[3 + n]; dsq[n] = h->d_out[3 + n]; }

  CU(host_event(h->ev_in_begin, sin));
  // ---- H2D: planes [h-1, h+nx] split so that chunk c's kernels need chunks <= c only
  auto h2d_chunk = [&](int c) -> int {
    const int lo = (c == 0) ? h->h - 1 : h->h + h->chunk_b[c - 1] + 1;
    const int hi = h->h + h->chunk_b[c] + 1;  // exclusive; includes the +1 plane
    const size_t off = (size_t)lo * plane_b, bytes = (size_t)(hi - lo) * plane_b;
    for (int n = 0; n < nf; ++n)
      CU(cudaMemcpyAsync((char *)h->d_in[n] + off, hin[n] + off, bytes, cudaMemcpyHostToDevice, sin));
    if (h->accumulate) {
      // accumulate: the caller's source terms of this slab go up too and the kernels add
      // to them on the device, so what comes back is already combined
      const int ia = h->h + h->chunk_a[c], ib = h->h + h->chunk_b[c];
      const size_t ooff = ((size_t)ia * h->nyh + h->h) * h->nz * es;
      const size_t width = (size_t)h->ny * h->nz * es;
      for (int n = mom ? 0 : 3; n < nf; ++n)
        CU(cudaMemcpy2DAsync((char *)h->d_out[n] + ooff, plane_b, hout[n] + ooff, plane_b, width,
                             (size_t)(ib - ia), cudaMemcpyHostToDevice, sin));
    }
    CU(host_event(h->ev_h2d[c], sin));
    CU(cudaEventRecord(h->dep_h2d[c], sin));
    return MONC_ADV_OK;
  };
  auto compute_chunk = [&](int c) -> int {
    const int ia = h->h + h->chunk_a[c], ib = h->h + h->chunk_b[c];
    if (h->overlap) CU(cudaStreamWaitEvent(sk, h->dep_h2d[c], 0));
    CU(host_event(h->ev_kb[c], sk));
    int rc = MONC_ADV_OK;
    if (mom)
      rc = launch_tendencies<T>(h, du, dv, dw, (T *)h->d_out[0], (T *)h->d_out[1], (T *)h->d_out[2],
                                dq.data(), dsq.data(), nq, ia, ib, sk);
    else if (nq > 0)
      rc = launch_scalars<T>(h, du, dv, dw, dq.data(), dsq.data(), nq, ia, ib, sk);
    if (rc != MONC_ADV_OK) return rc;
    CU(host_event(h->ev_ke[c], sk));
    CU(cudaEventRecord(h->dep_ke[c], sk));
    return MONC_ADV_OK;
  };
  auto d2h_chunk = [&](int c) -> int {
    const int ia = h->h + h->chunk_a[c], ib = h->h + h->chunk_b[c];
    if (h->overlap) CU(cudaStreamWaitEvent(sout, h->dep_ke[c], 0));
    if (c == 0) CU(host_event(h->ev_out_begin, sout));
    // interior columns only: 2-D copy, one row per x plane
    const size_t off = ((size_t)ia * h->nyh + h->h) * h->nz * es;
    const size_t width = (size_t)h->ny * h->nz * es;
    for (int n = mom ? 0 : 3; n < nf; ++n)
      CU(cudaMemcpy2DAsync(hout[n] + off, plane_b, (char *)h->d_out[n] + off, plane_b, width,
                           (size_t)(ib - ia), cudaMemcpyDeviceToHost, sout));
    CU(host_event(h->ev_d2h[c], sout));
    return MONC_ADV_OK;
  };
  int rc;
  if (h->overlap) {
    for (int c = 0; c < C; ++c) {
      if ((rc = h2d_chunk(c)) != MONC_ADV_OK) return rc;
      if ((rc = compute_chunk(c)) != MONC_ADV_OK) return rc;
      if ((rc = d2h_chunk(c)) != MONC_ADV_OK) return rc;
    }
  } else {
    for (int c = 0; c < C; ++c) if ((rc = h2d_chunk(c)) != MONC_ADV_OK) return rc;
    for (int c = 0; c < C; ++c) if ((rc = compute_chunk(c)) != MONC_ADV_OK) return rc;
    for (int c = 0; c < C; ++c) if ((rc = d2h_chunk(c)) != MONC_ADV_OK) return rc;
  }
  if (h->overlap) {
    // the kernel and D2H streams rejoin s_in: s_in is complete when the step is (and a
    // capture needs every forked stream joined before it ends)
    CU(cudaEventRecord(h->dep_join_k, sk));
    CU(cudaEventRecord(h->dep_join_out, sout));
    CU(cudaStreamWaitEvent(sin, h->dep_join_k, 0));
    CU(cudaStreamWaitEvent(sin, h->dep_join_out, 0));
  }
  return MONC_ADV_OK;
}

void drop_graph(monc_adv_t h) {
  if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
  h->graph_exec = nullptr;
  h->graph_key.clear();
}

// Enqueue one hybrid step.  A step whose arguments and settings equal those of the step before
// it is captured into a CUDA graph (all three streams, every copy, launch and event) and from
// then on replayed with ONE cudaGraphLaunch: the enqueue of config 2's 32-chunk step costs the
// host 1.5-1.9 ms call by call (about 900 CUDA calls), a replay a few tens of microseconds
// (DESIGN.md 8).  The first step with new arguments is enqueued call by call (it also fills
// the plan and descriptor caches, so that a capture makes stream calls only).
template <typename T>
int step_async_enqueue(monc_adv_t h, const void *hu, const void *hv, const void *hw, const void *const *hq, int nq,
                       void *hsu, void *hsv, void *hsw, void *const *hsq, cudaStream_t user) {
  std::vector<uintptr_t> key = {(uintptr_t)hu, (uintptr_t)hv, (uintptr_t)hw, (uintptr_t)hsu, (uintptr_t)hsv,
                                (uintptr_t)hsw, (uintptr_t)nq, (uintptr_t)h->epoch};
  for (int n = 0; n < nq; ++n) { key.push_back((uintptr_t)hq[n]); key.push_back((uintptr_t)hsq[n]); }
  cudaStream_t sin = h->s_in;
  if (user) {
    CU(cudaEventRecord(h->ev_user, user));
    CU(cudaStreamWaitEvent(sin, h->ev_user, 0));
  }
  const bool graphs = h->use_graph && h->overlap;
  int rc = MONC_ADV_OK;
  if (graphs && h->graph_exec && key == h->graph_key) {
    CU(cudaGraphLaunch(h->graph_exec, sin));  // chunk ranges, plans: those of the captured step
    h->launches += h->graph_launches;
  } else if (graphs && key == h->pending_key) {
    drop_graph(h);
    const long l0 = h->launches;
    cudaGraph_t graph = nullptr;
    CU(cudaStreamBeginCapture(sin, cudaStreamCaptureModeThreadLocal));
    rc = step_async_impl<T>(h, hu, hv, hw, hq, nq, hsu, hsv, hsw, hsq, true);
    const cudaError_t ec = cudaStreamEndCapture(sin, &graph);  // (ends an invalidated capture too)
    const std::string why = h->err;
    if (rc == MONC_ADV_OK && ec == cudaSuccess && graph &&
        cudaGraphInstantiate(&h->graph_exec, graph, 0) == cudaSuccess) {
      h->graph_launches = h->launches - l0;
      h->graph_key = key;
      cudaGraphDestroy(graph);
      CU(cudaGraphLaunch(h->graph_exec, sin));
    } else {
      // a capture that does not work on this driver is not an error of the step: enqueue it call
      // by call, and do not try again on this handle
      if (graph) cudaGraphDestroy(graph);
      cudaGetLastError();
      h->graph_exec = nullptr;
      h->use_graph = 0;
      h->launches = l0;
      h->err = why;
      rc = step_async_impl<T>(h, hu, hv, hw, hq, nq, hsu, hsv, hsw, hsq, false);
      if (rc != MONC_ADV_OK) return rc;
    }
  } else {
    if (graphs && h->graph_exec) drop_graph(h);
    rc = step_async_impl<T>(h, hu, hv, hw, hq, nq, hsu, hsv, hsw, hsq, false);
    if (rc != MONC_ADV_OK) return rc;
    h->pending_key = key;
  }
  if (user) {
    CU(cudaEventRecord(h->ev_done, sin));
    CU(cudaStreamWaitEvent(user, h->ev_done, 0));
  }
  h->in_flight = true;
  h->have_times = false;
  return MONC_ADV_OK;
}

}  // namespace

// ---------------------------------------------------------------------------
// monc_adv_step_noalloc: the momentum step from pinned host memory with its device staging
// in a file-scope array instead of cudaMalloc'ed buffers (include/monc_adv.h).
//
// g_noalloc_scratch lives in every GPU that loads this library, until exit.  In HOST code
// its name is a host-side stand-in, not a device address: the address kernels and copies
// use is fetched with cudaGetSymbolAddress, once per device, with that device current.
// Every call on a device shares the array (whatever the handle) and finds the last call's
// contents in it; nothing in it has to start at zero, because a call overwrites every byte
// its kernel reads (the three whole input arrays) before the kernel runs and copies back
// only bytes the kernel wrote (interior points of the three tendencies).  Calls that
// overlap on the GPU (two streams, two host threads) race on it.
// ---------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_noalloc_scratch[MONC_ADV_NOALLOC_MAX_BYTES];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_noalloc_mu;
unsigned char *g_noalloc_ptr[kMaxDevices] = {};  // device address of g_noalloc_scratch, per device

// h->device is current (check_handle)
int noalloc_scratch_address(monc_adv_t h, unsigned char **out) {
  if (h->device < 0 || h->device >= kMaxDevices) return fail(h, MONC_ADV_EINVAL, "step_noalloc: device ordinal out of range");
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[h->device]) {
    void *ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
    if (e != cudaSuccess || !ptr) {
      cudaGetLastError();
      return cuda_fail(h, e == cudaSuccess ? cudaErrorInvalidSymbol : e, "cudaGetSymbolAddress(scratch)");
    }
    g_noalloc_ptr[h->device] = static_cast<unsigned char *>(ptr);
  }
  *out = g_noalloc_ptr[h->device];
  return MONC_ADV_OK;
}

template <typename T>
int step_noalloc_impl(monc_adv_t h, unsigned char *scratch, size_t slot, const void *hu, const void *hv,
                      const void *hw, void *hsu, void *hsv, void *hsw, cudaStream_t st) {
  const size_t bytes = h->elems * sizeof(T);
  T *d[6];
  for (int n = 0; n < 6; ++n) d[n] = reinterpret_cast<T *>(scratch + (size_t)n * slot);
  const void *hin[3] = {hu, hv, hw};
  void *hout[3] = {hsu, hsv, hsw};
  for (int n = 0; n < 3; ++n) CU(cudaMemcpyAsync(d[n], hin[n], bytes, cudaMemcpyHostToDevice, st));
  const int rc = launch_momentum<T>(h, d[0], d[1], d[2], d[3], d[4], d[5], h->h, h->h + h->nx, st);
  if (rc != MONC_ADV_OK) return rc;
  // interior columns of the interior planes only: output halos are never written
  const size_t plane_b = (size_t)h->nyh * h->nz * sizeof(T);
  const size_t off = ((size_t)h->h * h->nyh + h->h) * h->nz * sizeof(T);
  const size_t width = (size_t)h->ny * h->nz * sizeof(T);
  for (int n = 0; n < 3; ++n)
    CU(cudaMemcpy2DAsync((char *)hout[n] + off, plane_b, (const char *)d[3 + n] + off, plane_b, width, (size_t)h->nx,
                         cudaMemcpyDeviceToHost, st));
  return MONC_ADV_OK;
}
}  // namespace

extern "C" {

int monc_adv_create(monc_adv_t *out, int nx, int ny, int nz, int halo, double dx, double dy,
                    const double *dz, const double *dzn, const double *rho, const double *rhon,
                    const double *tzc1, const double *tzc2, const double *tzd1,
                    const double *tzd2, int dtype) {
  if (!out) { g_create_error = "out is NULL"; return MONC_ADV_EINVAL; }
  *out = nullptr;
  auto bad = [&](const char *m) { g_create_error = m; return MONC_ADV_EINVAL; };
  if (nx < 1 || ny < 1) return bad("nx, ny must be >= 1");
  if (nz < 3) return bad("nz must be >= 3");
  if (halo < 1) return bad("halo must be >= 1");
  if (!(dx > 0) || !(dy > 0)) return bad("dx, dy must be > 0");
  if (dtype != MONC_ADV_F64 && dtype != MONC_ADV_F32) return bad("dtype must be F64 or F32");
  const int ntz = (tzc1 != nullptr) + (tzc2 != nullptr) + (tzd1 != nullptr) + (tzd2 != nullptr);
  if (ntz != 0 && ntz != 4) return bad("tzc1, tzc2, tzd1, tzd2 must be all given or all NULL");
  if (ntz == 0 && (!dz || !dzn || !rho || !rhon)) return bad("dz, dzn, rho, rhon required when tz arrays are NULL");
  if ((long long)(nx + 2 * halo) * (ny + 2 * halo) * nz > (1LL << 40)) return bad("field too large");

  monc_adv_s *h = new (std::nothrow) monc_adv_s;
  if (!h) { g_create_error = "out of host memory"; return MONC_ADV_ENOMEM; }
  h->nx = nx; h->ny = ny; h->nz = nz; h->h = halo; h->dtype = dtype;
  h->nxh = nx + 2 * halo; h->nyh = ny + 2 * halo;
  h->dx = dx; h->dy = dy;
  h->elems = (size_t)h->nxh * h->nyh * nz;
  h->esize = dtype == MONC_ADV_F64 ? 8 : 4;
  {
    int g = 1;
    while (((size_t)g * nz * h->esize) % 16 != 0) g *= 2;  // 1, 2 or 4
    h->colgroup = h->nyh % g == 0 ? g : 0;
  }
  auto cfail = [&](cudaError_t e, const char *what) {
    g_create_error = std::string(what) + ": " + cudaGetErrorString(e);
    const int code = e == cudaErrorMemoryAllocation ? MONC_ADV_ENOMEM : MONC_ADV_ECUDA;
    for (void *p : h->d_tz) if (p) cudaFree(p);
    delete h;
    return code;
  };
  cudaError_t e = cudaGetDevice(&h->device);
  if (e != cudaSuccess) return cfail(e, "cudaGetDevice");
  e = cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, h->device);
  if (e != cudaSuccess) return cfail(e, "cudaDeviceGetAttribute");
  e = cudaDeviceGetAttribute(&h->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
  if (e != cudaSuccess) return cfail(e, "cudaDeviceGetAttribute");

  // ---- coefficient tables (SURVEY.md 8(c).2 "Coefficients"), fp64 on the host
  for (auto &t : h->tz_host) t.assign(nz, 0.0);
  if (ntz == 4) {
    const double *src[4] = {tzc1, tzc2, tzd1, tzd2};
    for (int a = 0; a < 4; ++a) std::copy(src[a], src[a] + nz, h->tz_host[a].begin());
  } else {
    for (int k = 1; k <= nz - 1; ++k) {
      const double den = 4.0 * rhon[k] * dz[k];
      h->tz_host[0][k] = rho[k - 1] / den;
      h->tz_host[1][k] = rho[k] / den;
    }
    for (int k = 1; k <= nz - 2; ++k) {
      const double den = 4.0 * rho[k] * dzn[k + 1];
      h->tz_host[2][k] = rhon[k] / den;
      h->tz_host[3][k] = rhon[k + 1] / den;
    }
  }
  // entries the definition never uses are pinned to 0 so the kernels need no
  // special case: no tendency at K=1, no flux through the lid z_nz.
  h->tz_host[0][0] = h->tz_host[1][0] = h->tz_host[2][0] = h->tz_host[3][0] = 0.0;
  h->tz_host[1][nz - 1] = 0.0;
  h->tz_host[2][nz - 1] = h->tz_host[3][nz - 1] = 0.0;
  // device tables: zero-padded to whole 16-byte vectors plus one (the last thread of a ragged
  // column reads its whole vector)
  const size_t tz_bytes = ((size_t)nz * h->esize + 15) / 16 * 16 + 16;
  for (int a = 0; a < 4; ++a) {
    e = cudaMalloc(&h->d_tz[a], tz_bytes);
    if (e == cudaSuccess) e = cudaMemset(h->d_tz[a], 0, tz_bytes);
    if (e != cudaSuccess) return cfail(e, "cudaMalloc(constants)");
    if (dtype == MONC_ADV_F64) {
      e = cudaMemcpy(h->d_tz[a], h->tz_host[a].data(), (size_t)nz * 8, cudaMemcpyHostToDevice);
    } else {
      std::vector<float> f(nz);
      for (int k = 0; k < nz; ++k) { f[k] = (float)h->tz_host[a][k]; h->tz_host[a][k] = (double)f[k]; }
      e = cudaMemcpy(h->d_tz[a], f.data(), (size_t)nz * 4, cudaMemcpyHostToDevice);
    }
    if (e != cudaSuccess) return cfail(e, "cudaMemcpy(constants)");
  }
  g_create_error.clear();
  *out = h;
  return MONC_ADV_OK;
}

void monc_adv_destroy(monc_adv_t h) {
  if (!h) return;
  cudaSetDevice(h->device);
  if (h->in_flight) monc_adv_step_wait(h);
  free_staging(h);
  for (void *p : h->d_tz) if (p) cudaFree(p);
  for (auto v : {&h->ev_h2d, &h->ev_kb, &h->ev_ke, &h->ev_d2h})
    for (cudaEvent_t ev : *v) cudaEventDestroy(ev);
  drop_graph(h);
  for (auto v : {&h->dep_h2d, &h->dep_ke})
    for (cudaEvent_t ev : *v) cudaEventDestroy(ev);
  for (cudaEvent_t ev : {h->dep_join_k, h->dep_join_out, h->ev_done})
    if (ev) cudaEventDestroy(ev);
  if (h->ev_user) cudaEventDestroy(h->ev_user);
  if (h->ev_in_begin) cudaEventDestroy(h->ev_in_begin);
  if (h->ev_out_begin) cudaEventDestroy(h->ev_out_begin);
  if (h->s_in) cudaStreamDestroy(h->s_in);
  if (h->s_k) cudaStreamDestroy(h->s_k);
  if (h->s_out) cudaStreamDestroy(h->s_out);
  delete h;
}

int monc_adv_bind_wind(monc_adv_t h, const void *u, const void *v, const void *w) {
  if (!h) return MONC_ADV_EINVAL;
  if (!u || !v || !w) return fail(h, MONC_ADV_EINVAL, "bind_wind: NULL pointer");
  if (!aligned16(u) || !aligned16(v) || !aligned16(w))
    return fail(h, MONC_ADV_EINVAL, "bind_wind: pointers must be 16-byte aligned");
  h->wind[0] = u; h->wind[1] = v; h->wind[2] = w;
  return MONC_ADV_OK;
}

int monc_adv_momentum(monc_adv_t h, const void *u, const void *v, const void *w, void *su,
                      void *sv, void *sw, void *cuda_stream) {
  int rc = check_handle(h);
  if (rc) return rc;
  if (!u || !v || !w || !su || !sv || !sw) return fail(h, MONC_ADV_EINVAL, "momentum: NULL pointer");
  const void *all[6] = {u, v, w, su, sv, sw};
  for (const void *p : all)
    if (!aligned16(p)) return fail(h, MONC_ADV_EINVAL, "momentum: pointers must be 16-byte aligned");
  if (const char *why = find_alias({u, v, w}, {su, sv, sw}, h->elems * h->esize))
    return fail(h, MONC_ADV_EINVAL, std::string("momentum: ") + why);
  h->wind[0] = u; h->wind[1] = v; h->wind[2] = w;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (h->dtype == MONC_ADV_F64)
    return launch_momentum<double>(h, (const double *)u, (const double *)v, (const double *)w,
                                   (double *)su, (double *)sv, (double *)sw, h->h, h->h + h->nx, st);
  return launch_momentum<float>(h, (const float *)u, (const float *)v, (const float *)w,
                                (float *)su, (float *)sv, (float *)sw, h->h, h->h + h->nx, st);
}

int monc_adv_scalars(monc_adv_t h, const void *const *q, void *const *sq, int nq,
                     void *cuda_stream) {
  int rc = check_handle(h);
  if (rc) return rc;
  if (nq < 0 || nq > MONC_ADV_MAX_SCALARS) return fail(h, MONC_ADV_EINVAL, "scalars: nq out of range");
  if (nq == 0) return MONC_ADV_OK;
  if (!q || !sq) return fail(h, MONC_ADV_EINVAL, "scalars: NULL pointer table");
  if (!h->wind[0]) return fail(h, MONC_ADV_ENOWIND, "scalars: no wind bound (call momentum or bind_wind first)");
  std::vector<const void *> ins = {h->wind[0], h->wind[1], h->wind[2]}, outs;
  for (int n = 0; n < nq; ++n) {
    if (!q[n] || !sq[n]) return fail(h, MONC_ADV_EINVAL, "scalars: NULL field pointer");
    if (!aligned16(q[n]) || !aligned16(sq[n]))
      return fail(h, MONC_ADV_EINVAL, "scalars: pointers must be 16-byte aligned");
    ins.push_back(q[n]);
    outs.push_back(sq[n]);
  }
  if (const char *why = find_alias(ins, outs, h->elems * h->esize))
    return fail(h, MONC_ADV_EINVAL, std::string("scalars: ") + why);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (h->dtype == MONC_ADV_F64)
    return launch_scalars<double>(h, (const double *)h->wind[0], (const double *)h->wind[1],
                                  (const double *)h->wind[2], q, sq, nq, h->h, h->h + h->nx, st);
  return launch_scalars<float>(h, (const float *)h->wind[0], (const float *)h->wind[1],
                               (const float *)h->wind[2], q, sq, nq, h->h, h->h + h->nx, st);
}

int monc_adv_tendencies(monc_adv_t h, const void *u, const void *v, const void *w, void *su,
                        void *sv, void *sw, const void *const *q, void *const *sq, int nq,
                        void *cuda_stream) {
  int rc = check_handle(h);
  if (rc) return rc;
  if (!u || !v || !w || !su || !sv || !sw) return fail(h, MONC_ADV_EINVAL, "tendencies: NULL pointer");
  if (nq < 0 || nq > MONC_ADV_MAX_SCALARS) return fail(h, MONC_ADV_EINVAL, "tendencies: nq out of range");
  if (nq > 0 && (!q || !sq)) return fail(h, MONC_ADV_EINVAL, "tendencies: NULL pointer table");
  std::vector<const void *> ins = {u, v, w}, outs = {su, sv, sw};
  for (int n = 0; n < nq; ++n) {
    if (!q[n] || !sq[n]) return fail(h, MONC_ADV_EINVAL, "tendencies: NULL field pointer");
    ins.push_back(q[n]);
    outs.push_back(sq[n]);
  }
  for (const void *p : ins)
    if (!aligned16(p)) return fail(h, MONC_ADV_EINVAL, "tendencies: pointers must be 16-byte aligned");
  for (const void *p : outs)
    if (!aligned16(p)) return fail(h, MONC_ADV_EINVAL, "tendencies: pointers must be 16-byte aligned");
  if (const char *why = find_alias(ins, outs, h->elems * h->esize))
    return fail(h, MONC_ADV_EINVAL, std::string("tendencies: ") + why);
  h->wind[0] = u; h->wind[1] = v; h->wind[2] = w;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (h->dtype == MONC_ADV_F64)
    return launch_tendencies<double>(h, (const double *)u, (const double *)v, (const double *)w, (double *)su,
                                     (double *)sv, (double *)sw, q, sq, nq, h->h, h->h + h->nx, st);
  return launch_tendencies<float>(h, (const float *)u, (const float *)v, (const float *)w, (float *)su,
                                  (float *)sv, (float *)sw, q, sq, nq, h->h, h->h + h->nx, st);
}

int monc_adv_set_fuse(monc_adv_t h, int on) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;  // a captured step never outlives a setting
  h->fuse = on ? 1 : 0;
  return MONC_ADV_OK;
}

int monc_adv_step_async(monc_adv_t h, const void *hu, const void *hv, const void *hw,
                        const void *const *hq, int nq, void *hsu, void *hsv, void *hsw,
                        void *const *hsq, void *cuda_stream) {
  int rc = check_handle(h);
  if (rc) return rc;
  if (h->in_flight) return fail(h, MONC_ADV_EBUSY, "step_async: previous step still in flight (call step_wait)");
  if (nq < 0 || nq > MONC_ADV_MAX_SCALARS) return fail(h, MONC_ADV_EINVAL, "step_async: nq out of range");
  if (!hu || !hv || !hw) return fail(h, MONC_ADV_EINVAL, "step_async: NULL wind pointer");
  const int nout = (hsu != nullptr) + (hsv != nullptr) + (hsw != nullptr);
  if (nout != 0 && nout != 3) return fail(h, MONC_ADV_EINVAL, "step_async: hsu, hsv, hsw must be all given or all NULL");
  if (nout == 0 && nq == 0) return fail(h, MONC_ADV_EINVAL, "step_async: nothing to compute");
  if (nq > 0 && (!hq || !hsq)) return fail(h, MONC_ADV_EINVAL, "step_async: NULL pointer table");
  for (int n = 0; n < nq; ++n)
    if (!hq[n] || !hsq[n]) return fail(h, MONC_ADV_EINVAL, "step_async: NULL field pointer");
  std::vector<const void *> ins = {hu, hv, hw}, outs;
  if (nout) outs = {hsu, hsv, hsw};
  for (int n = 0; n < nq; ++n) { ins.push_back(hq[n]); outs.push_back(hsq[n]); }
  const size_t bytes = h->elems * h->esize;
  if (const char *why = find_alias(ins, outs, bytes))
    return fail(h, MONC_ADV_EINVAL, std::string("step_async: ") + why);
  for (const std::vector<const void *> *v : {&ins, &outs})
    for (const void *p : *v)
      if (!is_pinned_host(p, bytes))
        return fail(h, MONC_ADV_EINVAL, "step_async: every host array must be page-locked (pinned) over its "
                                        "whole length; pageable memory would make the copies synchronous");
  rc = ensure_async_objects(h, nq, step_chunks(h, 3 + nq, ((hsu ? 3 : 0) + nq) * (h->accumulate ? 2 : 1)));
  if (rc) return rc;
  cudaStream_t user = (cudaStream_t)cuda_stream;
  rc = h->dtype == MONC_ADV_F64 ? step_async_enqueue<double>(h, hu, hv, hw, hq, nq, hsu, hsv, hsw, hsq, user)
                                : step_async_enqueue<float>(h, hu, hv, hw, hq, nq, hsu, hsv, hsw, hsq, user);
  if (rc != MONC_ADV_OK) {
    // part of the step may already be queued: let it finish (it touches only the caller's
    // arrays of this call and the staging buffers), then report; the handle stays usable
    const std::string msg = h->err;
    drain_internal_streams(h);
    h->in_flight = false;
    h->err = msg;
  }
  return rc;
}

int monc_adv_step_noalloc(monc_adv_t h, const void *hu, const void *hv, const void *hw, void *hsu, void *hsv,
                          void *hsw, void *cuda_stream) {
  int rc = check_handle(h);
  if (rc) return rc;
  if (!hu || !hv || !hw || !hsu || !hsv || !hsw) return fail(h, MONC_ADV_EINVAL, "step_noalloc: NULL pointer");
  if (h->accumulate) return fail(h, MONC_ADV_EINVAL, "step_noalloc: overwrite mode only (set_accumulate(0))");
  const size_t bytes = h->elems * h->esize;
  const size_t slot = (bytes + 255) / 256 * 256;  // every staged field starts on a 256-byte boundary
  if (6 * slot > (size_t)MONC_ADV_NOALLOC_MAX_BYTES) {
    char b[256];
    snprintf(b, sizeof b, "step_noalloc: 6 staged fields of %zu bytes need %zu bytes, the static scratch holds "
             "MONC_ADV_NOALLOC_MAX_BYTES = %zu (use monc_adv_step_async for larger domains)", bytes, 6 * slot,
             (size_t)MONC_ADV_NOALLOC_MAX_BYTES);
    return fail(h, MONC_ADV_EINVAL, b);
  }
  if (const char *why = find_alias({hu, hv, hw}, {hsu, hsv, hsw}, bytes))
    return fail(h, MONC_ADV_EINVAL, std::string("step_noalloc: ") + why);
  for (const void *p : {hu, hv, hw, (const void *)hsu, (const void *)hsv, (const void *)hsw})
    if (!is_pinned_host(p, bytes))
      return fail(h, MONC_ADV_EINVAL, "step_noalloc: every host array must be page-locked (pinned) over its whole length");
  unsigned char *scratch = nullptr;
  rc = noalloc_scratch_address(h, &scratch);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  return h->dtype == MONC_ADV_F64 ? step_noalloc_impl<double>(h, scratch, slot, hu, hv, hw, hsu, hsv, hsw, st)
                                  : step_noalloc_impl<float>(h, scratch, slot, hu, hv, hw, hsu, hsv, hsw, st);
}

int monc_adv_step_inputs_consumed(monc_adv_t h) {
  int rc = check_handle(h);
  if (rc) return rc;
  if (!h->in_flight) return MONC_ADV_OK;
  CU(cudaEventSynchronize(h->ev_h2d[h->chunk_a.size() - 1]));
  return MONC_ADV_OK;
}

int monc_adv_step_wait_chunk(monc_adv_t h, int c) {
  int rc = check_handle(h);
  if (rc) return rc;
  if (!h->in_flight) return fail(h, MONC_ADV_EINVAL, "step_wait_chunk: no step in flight");
  if (c < 0 || c >= (int)h->chunk_a.size()) return fail(h, MONC_ADV_EINVAL, "step_wait_chunk: chunk out of range");
  CU(cudaEventSynchronize(h->ev_d2h[c]));
  return MONC_ADV_OK;
}

int monc_adv_step_wait(monc_adv_t h) {
  int rc = check_handle(h);
  if (rc) return rc;
  if (!h->in_flight) return MONC_ADV_OK;
  const int C = (int)h->chunk_a.size();
  CU(cudaEventSynchronize(h->ev_d2h[C - 1]));
  CU(cudaStreamSynchronize(h->s_in));
  h->in_flight = false;  // only now: a failed wait leaves the step marked in flight
  float t = 0, ksum = 0;
  CU(cudaEventElapsedTime(&t, h->ev_in_begin, h->ev_h2d[C - 1]));
  h->times[0] = t;
  for (int c = 0; c < C; ++c) {
    CU(cudaEventElapsedTime(&t, h->ev_kb[c], h->ev_ke[c]));
    ksum += t;
  }
  h->times[1] = ksum;
  CU(cudaEventElapsedTime(&t, h->ev_out_begin, h->ev_d2h[C - 1]));
  h->times[2] = t;
  CU(cudaEventElapsedTime(&t, h->ev_in_begin, h->ev_d2h[C - 1]));
  h->times[3] = t;
  h->have_times = true;
  return MONC_ADV_OK;
}

int monc_adv_plan_describe(int nx, int ny, int nz, int halo, int dtype, int nq, int fused, int sm_count,
                           int smem_optin, char *buf, int buflen) {
  if (nx < 1 || ny < 1 || nz < 3 || halo < 1 || nq < 0 || nq > 20 || !buf || buflen < 1 || sm_count < 1 ||
      smem_optin < 1024 || (dtype != MONC_ADV_F64 && dtype != MONC_ADV_F32))
    return MONC_ADV_EINVAL;
  monc_adv_s hs;  // a shape only: no CUDA call is made through it
  monc_adv_t h = &hs;
  h->plan_only = true;
  h->nx = nx; h->ny = ny; h->nz = nz; h->h = halo; h->dtype = dtype;
  h->nxh = nx + 2 * halo; h->nyh = ny + 2 * halo;
  h->esize = dtype == MONC_ADV_F64 ? 8 : 4;
  h->sm_count = sm_count; h->smem_optin = smem_optin;
  int g = 1;
  while (((size_t)g * nz * h->esize) % 16 != 0) g *= 2;
  h->colgroup = h->nyh % g == 0 ? g : 0;
  char b[320];
  const bool f64 = dtype == MONC_ADV_F64;
  std::string text;
  if (!fused || nq == 0) {
    const TmaPlan pm = f64 ? compute_plan_tma<double>(h, nx, 3) : compute_plan_tma<float>(h, nx, 3);
    if (pm.ok) {
      snprintf(b, sizeof b, "tma_momentum ty=%d stages=%d xc=%d grid=%dx%d cluster=%d smem=%zu", pm.ty, pm.stages,
               pm.xc, (pm.tiles + pm.cl - 1) / pm.cl * pm.cl, pm.nchunks, pm.cl, pm.smem);
      text = b;
    } else {
      const TmaScalarPlan pr = f64 ? compute_plan_tma_scalars<double>(h, nx, 0, true)
                                   : compute_plan_tma_scalars<float>(h, nx, 0, true);
      if (pr.ok) {
        snprintf(b, sizeof b, "tma_fused(momentum role only) ty=%d stages=%d xc=%d grid=%dx%d colgroup=%d smem=%zu",
                 pr.ty, pr.stages, pr.xc, pr.tiles, pr.nchunks, h->colgroup, pr.smem);
        text = b;
      } else {
        text = "no TMA plan (momentum)";
      }
    }
  }
  if (nq > 0) {
    const TmaScalarPlan ps = f64 ? compute_plan_tma_scalars<double>(h, nx, std::min(nq, fused ? 10 : nq), fused != 0)
                                 : compute_plan_tma_scalars<float>(h, nx, std::min(nq, fused ? 10 : nq), fused != 0);
    if (ps.ok)
      snprintf(b, sizeof b, "%s group=%d per_warp=%d split=%d ty=%d stages=%d xc=%d grid=%dx%d cluster=%d colgroup=%d smem=%zu",
               fused ? "tma_fused(momentum+scalars)" : "tma_scalars", ps.gb, ps.gw, ps.ss, ps.ty, ps.stages, ps.xc,
               ps.tiles, ps.nchunks, ps.cl, std::max(1, h->colgroup), ps.smem);
    else
      snprintf(b, sizeof b, "no TMA plan (scalars)");
    text += (text.empty() ? "" : "; ") + std::string(b);
  }
  snprintf(buf, (size_t)buflen, "%s", text.c_str());
  return MONC_ADV_OK;
}

int monc_adv_plan_chunks(int nx, int ny, int nz, int halo, int dtype, int nfields_in, int nfields_out) {
  if (nx < 1 || ny < 1 || nz < 1 || halo < 1 || nfields_in < 1 || nfields_out < 1 ||
      (dtype != MONC_ADV_F64 && dtype != MONC_ADV_F32))
    return MONC_ADV_EINVAL;
  return auto_chunks_for(nx, ny + 2 * halo, nz, dtype == MONC_ADV_F64 ? 8 : 4, nfields_in, nfields_out);
}

int monc_adv_step_chunk_count(monc_adv_t h) {
  if (!h) return 0;
  if (h->nchunks > 0) return std::min(h->nchunks, h->nx);
  return (int)h->chunk_a.size();  // automatic: known once a step has been enqueued
}

int monc_adv_step_chunk_range(monc_adv_t h, int c, int *x_begin, int *x_end) {
  if (!h) return MONC_ADV_EINVAL;
  const int C = monc_adv_step_chunk_count(h);
  if (C == 0) return fail(h, MONC_ADV_EINVAL, "step_chunk_range: automatic chunk count and no step enqueued yet");
  if (c < 0 || c >= C || !x_begin || !x_end) return fail(h, MONC_ADV_EINVAL, "step_chunk_range: bad argument");
  *x_begin = (int)((long long)h->nx * c / C);
  *x_end = (int)((long long)h->nx * (c + 1) / C);
  return MONC_ADV_OK;
}

int monc_adv_step_times_ms(monc_adv_t h, float out[4]) {
  if (!h || !out) return MONC_ADV_EINVAL;
  if (!h->have_times) return fail(h, MONC_ADV_EINVAL, "step_times_ms: no completed step");
  for (int a = 0; a < 4; ++a) out[a] = h->times[a];
  return MONC_ADV_OK;
}

int monc_adv_set_chunks(monc_adv_t h, int nchunks) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;  // a captured step never outlives a setting
  if (h->in_flight) return fail(h, MONC_ADV_EBUSY, "set_chunks: step in flight");
  if (nchunks < 0 || nchunks > h->nx) return fail(h, MONC_ADV_EINVAL, "set_chunks: need 0 (automatic) or 1 <= nchunks <= nx");
  h->nchunks = nchunks;
  h->chunk_a.clear();
  h->chunk_b.clear();
  return MONC_ADV_OK;
}

int monc_adv_set_overlap(monc_adv_t h, int on) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;  // a captured step never outlives a setting
  if (h->in_flight) return fail(h, MONC_ADV_EBUSY, "set_overlap: step in flight");
  h->overlap = on ? 1 : 0;
  return MONC_ADV_OK;
}

int monc_adv_set_form(monc_adv_t h, int form) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;  // a captured step never outlives a setting
  if (form != MONC_ADV_FORM_FLUX && form != MONC_ADV_FORM_PW_SKEW)
    return fail(h, MONC_ADV_EINVAL, "set_form: unknown form");
  if (form != MONC_ADV_FORM_FLUX && h->work > 1) return fail(h, MONC_ADV_EINVAL, "set_form: work scaling is on (flux form only)");
  h->form = form;
  return MONC_ADV_OK;
}

int monc_adv_set_accumulate(monc_adv_t h, int on) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;  // a captured step never outlives a setting
  if (on && h->work > 1) return fail(h, MONC_ADV_EINVAL, "set_accumulate: work scaling is on (overwrite mode only)");
  if ((on ? 1 : 0) != h->accumulate) h->mom_plans.clear();  // the accumulating momentum kernel takes fewer warps
  h->accumulate = on ? 1 : 0;
  return MONC_ADV_OK;
}

int monc_adv_set_work_scale(monc_adv_t h, int n) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;  // a captured step never outlives a setting
  if (n < 1 || n > 64) return fail(h, MONC_ADV_EINVAL, "set_work_scale: need 1 <= n <= 64");
  if (n > 1 && (h->form != MONC_ADV_FORM_FLUX || h->accumulate || (h->variant != 0 && h->variant != 3)))
    return fail(h, MONC_ADV_EINVAL, "set_work_scale: needs the flux form, overwrite mode and the TMA kernels");
  if ((n > 1) != (h->work > 1)) h->mom_plans.clear();  // the work-scaled momentum kernel takes fewer warps
  h->work = n;
  return MONC_ADV_OK;
}

int monc_adv_set_cluster(monc_adv_t h, int n) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;  // a captured step never outlives a setting
  if (n < 0 || n > 8) return fail(h, MONC_ADV_EINVAL, "set_cluster: 0 (default) or 1..8");
  h->cluster = n;
  h->mom_plans.clear();
  h->sca_plans.clear();
  return MONC_ADV_OK;
}

int monc_adv_set_l2_hint(monc_adv_t h, int hint) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;  // a captured step never outlives a setting
  if (hint < 0 || hint > 2) return fail(h, MONC_ADV_EINVAL, "set_l2_hint: 0 (none), 1 (evict_last) or 2 (evict_first)");
  h->l2hint = hint;
  return MONC_ADV_OK;
}

int monc_adv_set_graph(monc_adv_t h, int on) {
  if (!h) return MONC_ADV_EINVAL;
  if (h->in_flight) return fail(h, MONC_ADV_EBUSY, "set_graph: step in flight");
  h->epoch++;
  h->use_graph = on ? 1 : 0;
  return MONC_ADV_OK;
}

int monc_adv_graph_state(monc_adv_t h) {
  if (!h || !h->use_graph) return 0;
  return h->graph_exec ? 2 : 1;
}

int monc_adv_set_pdl(monc_adv_t h, int on) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;  // a captured step never outlives a setting
  h->pdl = on ? 1 : 0;
  return MONC_ADV_OK;
}

int monc_adv_set_variant(monc_adv_t h, int variant) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;  // a captured step never outlives a setting
  if (variant < 0 || variant > 3) return fail(h, MONC_ADV_EINVAL, "set_variant: 0..3");
  if (h->work > 1 && variant != 0 && variant != 3)
    return fail(h, MONC_ADV_EINVAL, "set_variant: work scaling is on (TMA kernels only)");
  const int nk = h->dtype == MONC_ADV_F64 ? 2 : 4;
  if (variant == 2 && h->nz % nk != 0)
    return fail(h, MONC_ADV_EINVAL, "set_variant: the direct-load marching kernels need nz % (16/sizeof(dtype)) == 0");
  if (variant == 3 && h->colgroup == 0)
    return fail(h, MONC_ADV_EINVAL, "set_variant: ragged nz needs ny + 2 halo to be a multiple of 2 (fp64, "
                                    "fp32 with even nz) or 4 (fp32 with odd nz) for the TMA kernels");
  h->variant = variant;
  return MONC_ADV_OK;
}

int monc_adv_set_tuning(monc_adv_t h, int xchunk, int group, int prefetch, int warps, int stages,
                        int tile_y, int split) {
  if (!h) return MONC_ADV_EINVAL;
  h->epoch++;
  if (xchunk < 0 || group < 0 || group > 10 || prefetch < -1 || prefetch > 16 || warps < 0 ||
      warps > kWarpsPerBlock || stages < 0 || stages > 8 || tile_y < 0 || split < 0 || split > 4)
    return fail(h, MONC_ADV_EINVAL, "set_tuning: value out of range");
  h->mom_plans.clear();
  h->sca_plans.clear();
  h->split = split;
  h->stages = stages;
  h->tile_y = tile_y;
  h->xchunk = xchunk;
  h->group = group;
  h->prefetch = prefetch;
  h->warps = warps;
  return MONC_ADV_OK;
}

int monc_adv_get_coefficients(monc_adv_t h, double *tzc1, double *tzc2, double *tzd1,
                              double *tzd2) {
  if (!h) return MONC_ADV_EINVAL;
  double *dst[4] = {tzc1, tzc2, tzd1, tzd2};
  for (int a = 0; a < 4; ++a)
    if (dst[a]) std::copy(h->tz_host[a].begin(), h->tz_host[a].end(), dst[a]);
  return MONC_ADV_OK;
}

long monc_adv_launch_count(monc_adv_t h) { return h ? h->launches : 0; }

const char *monc_adv_describe_plan(monc_adv_t h) {
  if (!h) return "";
  h->plan_text = h->plan_mom + (h->plan_mom.empty() || h->plan_sca.empty() ? "" : "; ") + h->plan_sca;
  return h->plan_text.c_str();
}

const char *monc_adv_last_error(monc_adv_t h) {
  return h ? h->err.c_str() : g_create_error.c_str();
}

const char *monc_adv_version(void) {
#if MONC_ADV_CHECKED
  return "monc-adv-b200 0.2 (sm_100a, checked build: poisoned ring slots, jittered schedule)";
#else
  return "monc-adv-b200 0.2 (sm_100a)";
#endif
}

}  // extern "C"
