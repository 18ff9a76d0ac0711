/*
 * monc_adv_tuning.h -- INTERNAL knobs of libmonc_adv.so: kernel family, launch
 * geometry, launch attribute.  For the library's own tests, benchmarks and
 * profiling; not part of the interface a model links against (include/monc_adv.h)
 * and free to change.  The defaults (0 everywhere) are what the library's launch
 * planners choose; results do not depend on any of these.
 */
#ifndef MONC_ADV_TUNING_H
#define MONC_ADV_TUNING_H

#include "monc_adv.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Kernel variant: 0 = auto (default), 1 = generic one-thread-per-point
 * kernels, 2 = x-marching vector kernels with direct global loads, 3 =
 * x-marching kernels fed by a TMA shared-memory ring.  2 needs
 * nz % (16/sizeof(dtype)) == 0 and the flux form; 3 takes a ragged nz too when
 * ny + 2 halo is a multiple of 2 (fp64, fp32 with even nz) or 4 (fp32, odd nz). */
int monc_adv_set_variant(monc_adv_t h, int variant);
/* Tuning knobs of the x-marching kernels; 0 = library default, -1 = off where
 * that makes sense.
 *   xchunk:   planes marched by one thread block;
 *   group:    scalars that share one staged copy of the wind: per thread block
 *             (1..10) in variant 3, per thread (1..5) in variant 2;
 *   prefetch: L2 prefetch distance in planes (-1 = no prefetch), variant 2;
 *   warps:    variant 2: warps per thread block (1..8); ignored by variant 3 (a
 *             block tile is one 32-vector z chunk per column);
 *   stages:   depth of the TMA ring (2..8), variant 3;
 *   tile_y:   columns per thread block, variant 3;
 *   split:    variant 3 scalars: warps that share one column chunk and split
 *             the block's scalars between them (1..4). */
int monc_adv_set_tuning(monc_adv_t h, int xchunk, int group, int prefetch, int warps, int stages,
                        int tile_y, int split);

/* Thread-block cluster size of the TMA kernels (1..8; 0 = library default): that
 * many y-neighbour tiles are launched as one cluster, i.e. co-scheduled on the SMs
 * of one GPC.  No shared-memory traffic crosses the cluster; it only keeps blocks
 * that re-read each other's halo rows running at the same rate. */
int monc_adv_set_cluster(monc_adv_t h, int n);

/* L2 eviction priority the TMA kernels ask for on their input copies: 1 (default)
 * evict_last -- a tile's halo rows are read again by the neighbouring blocks a few
 * steps later --, 0 no hint, 2 evict_first (for measurements). */
int monc_adv_set_l2_hint(monc_adv_t h, int hint);

/* The launch geometry the planners choose for a full-domain call on this shape, as text
 * (the format of monc_adv_describe_plan), for a device with sm_count SMs and smem_optin
 * bytes of opt-in shared memory per block (B200: 148, 232448).  fused != 0: the plan of
 * monc_adv_tendencies (the first 10 scalars); else monc_adv_momentum and, if nq > 0,
 * monc_adv_scalars.  Host arithmetic only: needs no handle and no GPU (the planners'
 * regression tests run on it).  buf receives at most buflen - 1 characters. */
int monc_adv_plan_describe(int nx, int ny, int nz, int halo, int dtype, int nq, int fused, int sm_count,
                           int smem_optin, char *buf, int buflen);

/* 1 (default): a hybrid step whose arguments and settings equal those of the step before it
 * is captured into a CUDA graph and replayed from then on (one cudaGraphLaunch instead of the
 * ~30 CUDA calls of every chunk).  0: every step is enqueued call by call.  Results and the
 * completion calls (step_inputs_consumed / step_wait_chunk / step_wait / step_times_ms) are the
 * same either way. */
int monc_adv_set_graph(monc_adv_t h, int on);
/* 0: graphs are off (set_graph(0), or a capture failed on this driver and the handle fell back
 * to call-by-call enqueues); 1: on, no step captured at the moment; 2: the last step was a
 * captured step (the next one with the same arguments is a replay). */
int monc_adv_graph_state(monc_adv_t h);

/* 1 (default): the TMA kernels are launched with CUDA's programmatic
 * stream-serialisation attribute, so a kernel's set-up overlaps the tail of its
 * predecessor in the stream (it waits for the predecessor's completion before
 * touching any field: results are unchanged).  0: plain stream order. */
int monc_adv_set_pdl(monc_adv_t h, int on);
#ifdef __cplusplus
}
#endif
#endif /* MONC_ADV_TUNING_H */
