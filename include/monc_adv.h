/*
 * monc_adv.h -- C ABI of the B200-native MONC advection source-term library.
 *
 * What it computes.  The computation arxiv 2009.12850 offloads to the GPU:
 * the advection source terms of MONC's prognostic fields ("the advection
 * scheme is the single longest running component"; "run the
 * advection kernel and compute advection source terms for the entirety of the
 * field"; Piacsek-Williams centred scheme).  The
 * paper prints no formula; the definition implemented is the flux-form
 * centred scheme on the Arakawa C grid written out in SURVEY.md 8(c).2 and
 * DESIGN.md "Definition" (BASELINE.json north_star).
 *
 * Layout (all field arrays, host or device): C order F[i][j][k], z (k)
 * fastest, then y, x slowest -- MONC's Fortran F(k,j,i).  NXH = nx + 2*halo,
 * NYH = ny + 2*halo, E = NXH*NYH*nz elements per field, linear index
 * (i*NYH + j)*nz + k.  Interior: i in [halo, halo+nx), j in [halo, halo+ny),
 * all k.  Level K = k+1 in the paper-side 1-based notation.  u sits on the
 * east face of cell i, v on the north face, w on the top face, scalars at the
 * cell centre.
 *
 * Semantics common to every compute call.
 *   - Tendencies are OVERWRITTEN at interior points, all k: su, sv, sq = 0 at
 *     k = 0 and the flux through the top face z_nz is dropped (rigid lid);
 *     sw = 0 at k = 0 and k = nz-1.  With monc_adv_set_accumulate(h, 1) they
 *     are ADDED to what the buffer holds instead (source terms
 *     are additive; combine on the device).
 *   - Halo entries of output arrays are never written.
 *   - Inputs need valid halos to depth 1 in x and y (the library does no halo
 *     exchange: PAPER.md:49 does it in an earlier timestep group).
 *   - No output array may overlap an input array or another output array
 *     (checked over the whole arrays, not only the base pointers: EINVAL).  All
 *     base pointers must be 16-byte aligned.
 *   - Shapes: any nx, ny >= 1, nz >= 3, halo >= 1.  The fast (TMA) kernels take
 *     every nz for which nz * sizeof(dtype) is a multiple of 16 bytes, and a
 *     "ragged" nz (any other) when ny + 2 halo is a multiple of 2 (fp64; fp32
 *     with even nz) or of 4 (fp32 with odd nz), at about 0.9 of the aligned rate
 *     in fp64; the remaining shapes run one-thread-per-point
 *     kernels (about 0.4).  With a ragged nz the value above a column's top level
 *     is read from the neighbouring column and multiplied by a zero coefficient:
 *     inputs must be finite.
 *   - Every call returns MONC_ADV_OK (0) or a negative error code, never
 *     throws or aborts; monc_adv_last_error gives the text of the last
 *     failure on that handle.
 *   - One handle = one device (the one current at create) and one dtype.
 *     Calls on one handle are not thread-safe against each other.
 */
#ifndef MONC_ADV_H
#define MONC_ADV_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct monc_adv_s *monc_adv_t; /* opaque, owned by the library */

enum { MONC_ADV_F64 = 0, MONC_ADV_F32 = 1 };
enum { MONC_ADV_FORM_FLUX = 0, MONC_ADV_FORM_PW_SKEW = 1 };
enum {
  MONC_ADV_OK = 0,
  MONC_ADV_EINVAL = -1,  /* bad argument (sizes, NULL, alignment, nq range) */
  MONC_ADV_ECUDA = -2,   /* a CUDA runtime call failed; see last_error */
  MONC_ADV_ENOMEM = -3,  /* host or device allocation failed */
  MONC_ADV_ENOWIND = -4, /* scalars requested before any wind was bound */
  MONC_ADV_EBUSY = -5    /* step_async while the previous step is in flight */
};
#define MONC_ADV_MAX_SCALARS 64

/*
 * Create a handle and upload the constants ONCE ("share the
 * constants between kernels and copy these across only once (on
 * initialisation)").
 *   nx, ny >= 1, nz >= 3, halo >= 1: interior size and halo width.
 *   dx, dy > 0: horizontal grid spacing (uniform).
 *   dz, dzn, rho, rhon: HOST arrays of nz doubles, index K-1: dz_K = z_K -
 *     z_{K-1}, dzn_K = zn_K - zn_{K-1}, rho_K = rho(z_K), rhon_K = rho(zn_K).
 *   tzc1, tzc2, tzd1, tzd2: HOST arrays of nz doubles or ALL NULL.  If NULL
 *     they are computed:
 *       tzc1_K = rho_{K-1}/(4 rhon_K dz_K), tzc2_K = rho_K/(4 rhon_K dz_K), K=2..nz
 *       tzd1_K = rhon_K/(4 rho_K dzn_{K+1}), tzd2_K = rhon_{K+1}/(4 rho_K dzn_{K+1}), K=2..nz-1
 *     If given, dz/dzn/rho/rhon may be NULL.
 *   dtype: MONC_ADV_F64 (reference path) or MONC_ADV_F32 (PAPER.md:125
 *     precision variant: fp32 storage AND arithmetic; constants are rounded
 *     once from double).
 * The caller keeps ownership of every array passed (they are copied).
 * Errors: EINVAL, ECUDA, ENOMEM; *out is NULL on failure.
 */
int monc_adv_create(monc_adv_t *out, int nx, int ny, int nz, int halo, double dx, double dy,
                    const double *dz, const double *dzn, const double *rho, const double *rhon,
                    const double *tzc1, const double *tzc2, const double *tzd1,
                    const double *tzd2, int dtype);

/* Free the handle, its device constants, staging buffers, streams and events.
 * Waits for an in-flight step.  NULL is ignored. */
void monc_adv_destroy(monc_adv_t h);

/*
 * Momentum tendencies su, sv, sw of (u, v, w) advected by (u, v, w)
 * (one fused kernel).  u, v, w, su, sv, sw: DEVICE
 * pointers to E elements of the handle's dtype.  Asynchronous: enqueued on
 * `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy default
 * stream).  Also BINDS (u, v, w) as the wind used by monc_adv_scalars
 * ("the u, v and w fields are also shared between kernels").
 */
int monc_adv_momentum(monc_adv_t h, const void *u, const void *v, const void *w, void *su,
                      void *sv, void *sw, void *cuda_stream);

/* Bind the advecting wind without computing momentum tendencies.  DEVICE
 * pointers, kept (not copied): the caller keeps them alive and unchanged
 * until the scalar kernels that use them have run. */
int monc_adv_bind_wind(monc_adv_t h, const void *u, const void *v, const void *w);

/*
 * Tendencies sq[n] of nq scalar fields q[n] (theta, moisture, tracers), all
 * advected by the bound wind (one batched kernel pass).
 * q, sq: HOST arrays of nq DEVICE pointers (E elements each).  0 <= nq <=
 * MONC_ADV_MAX_SCALARS; nq = 0 is a no-op.  Asynchronous on `cuda_stream`.
 * Errors: ENOWIND if no wind is bound.
 */
int monc_adv_scalars(monc_adv_t h, const void *const *q, void *const *sq, int nq,
                     void *cuda_stream);

/* The whole step from device arrays in one call (the lower bound
 * of 24 + 24 + 16 nq bytes per point is reached only if u, v, w are read once
 * for momentum AND scalars; "u, v and w ... shared between kernels").
 * Same results (same arithmetic; only the compiler's FMA contraction may differ)
 * as monc_adv_momentum(u, v, w, su, sv, sw) followed by monc_adv_scalars(q, sq,
 * nq); binds (u, v, w) as the wind.  With 1 <= nq <=
 * 10 and a TMA plan that fits, ONE launch does both (the momentum role rides in
 * the scalar kernel's thread blocks and reads the same staged wind tiles);
 * otherwise the two launches are made.  Arguments, layout, ownership and errors
 * as for the two calls; all outputs must be distinct and alias no input. */
int monc_adv_tendencies(monc_adv_t h, const void *u, const void *v, const void *w, void *su,
                        void *sv, void *sw, const void *const *q, void *const *sq, int nq,
                        void *cuda_stream);

/*
 * The paper's hybrid pattern:
 * fields live in PINNED HOST memory; the call enqueues, per x-slab chunk, the
 * H2D copy of the inputs, the kernels on that chunk and the D2H copy of its
 * tendencies, overlapped on internal streams, and RETURNS AT ONCE so the host
 * can run its other dynamics components.  u, v, w are copied once per step
 * and shared by the momentum and scalar kernels.
 *   hu, hv, hw, hq[n]: pinned host inputs, E elements each, valid halos.
 *   hsu, hsv, hsw, hsq[n]: pinned host outputs; only INTERIOR entries are
 *     written.  Default (overwrite): the GPU result lands in this separate
 *     buffer and the host adds it to its own source terms.
 *     With monc_adv_set_accumulate(h, 1) the arrays are IN/OUT: they hold the
 *     host's own source terms, each chunk's slab of them is uploaded with the
 *     fields, the kernels add the advection tendencies on the device
 *      and the combined source terms come back into the same
 *     arrays -- bitwise equal to waiting for the step and adding on the host,
 *     without the extra result buffer PAPER.md:99 needs.  hsu/hsv/hsw may ALL be
 *     NULL to advect scalars only.
 *   hq, hsq: host arrays of nq host pointers (may be NULL when nq = 0).
 *   cuda_stream: work already queued on it is waited for before the first
 *     copy; NULL = no dependency.
 * Device staging buffers (3+nq inputs, 3+nq outputs) are allocated on first
 * use and reused.  Errors: EBUSY if the previous step was not waited for;
 * EINVAL if an array is not page-locked over its whole length (pageable memory
 * would silently turn the asynchronous copies into synchronous ones, the very
 * failure PAPER.md:95 describes) or if arrays overlap.  If a CUDA call fails
 * part-way through the enqueue, what was queued is waited for, the error is
 * returned and no step is in flight: the handle stays usable.
 */
int monc_adv_step_async(monc_adv_t h, const void *hu, const void *hv, const void *hw,
                        const void *const *hq, int nq, void *hsu, void *hsv, void *hsw,
                        void *const *hsq, void *cuda_stream);

/* Block until every H2D copy of the in-flight step is done: the host may then
 * overwrite its input fields. */
int monc_adv_step_inputs_consumed(monc_adv_t h);
/* Block until chunk c's tendencies are in host memory: the host can integrate
 * the source terms of that slab while the later chunks are still streaming back
 * ("overlapping computation with data copying, rather than waiting for the entire
 * data copy").  0 <= c < nchunks. */
int monc_adv_step_wait_chunk(monc_adv_t h, int c);
/* Block until all tendencies of the in-flight step are in host memory and
 * mark the step complete.  No-op if no step is in flight. */
int monc_adv_step_wait(monc_adv_t h);
/* x-range [*x_begin, *x_end) of INTERIOR-relative x indices (0..nx) whose
 * tendencies chunk c delivers. */
int monc_adv_step_chunk_range(monc_adv_t h, int c, int *x_begin, int *x_end);
/* Device time of the last completed step in ms: out[0] = first H2D start to
 * last H2D end, out[1] = sum of kernel times, out[2] = first D2H start to
 * last D2H end, out[3] = whole step (first copy to last copy). */
int monc_adv_step_times_ms(monc_adv_t h, float out[4]);

/* The momentum step from pinned host memory for callers that cannot call cudaMalloc (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid it): this call
 * allocates NOTHING on the device -- no cudaMalloc / cudaFree, no stream or event creation,
 * no allocating library routine.  Its device staging (u, v, w in; su, sv, sw out) is a
 * file-scope device array of MONC_ADV_NOALLOC_MAX_BYTES that every GPU which loads the
 * library holds until exit.  Enqueued on `cuda_stream` (NULL = the default stream) and
 * asynchronous to the host: H2D of the three whole input arrays, the fused su/sv/sw kernel
 * (the kernel monc_adv_momentum launches), D2H of the interior of the three
 * tendencies; the host arrays are the caller's until the stream has drained (synchronise
 * the stream or an event recorded after the call).  Output halos are not written.
 * Limits: six staged fields must fit, 6 * round_up(NXH * NYH * nz * sizeof(dtype), 256)
 * <= MONC_ADV_NOALLOC_MAX_BYTES (the paper's 64 x 64 x 64 sub-domain with halo 2 in fp64
 * fits; BASELINE's configs 1-4 do not: MONC_ADV_EINVAL, nothing enqueued); momentum
 * only; overwrite mode only; host arrays page-locked and not overlapping.
 * The scratch is ONE array per device, shared by every handle and every call, and keeps
 * the last call's contents: nothing in it needs clearing (a call overwrites all it reads
 * before its kernel runs), but two calls that overlap on the GPU -- different streams, or
 * different host threads -- race on it.  Calls on one stream are safe back to back. */
#define MONC_ADV_NOALLOC_MAX_BYTES (16u << 20)
int monc_adv_step_noalloc(monc_adv_t h, const void *hu, const void *hv, const void *hw, void *hsu, void *hsv,
                          void *hsw, void *cuda_stream);

/* Number of x-slab chunks of step_async: 1 <= n <= nx, or 0 (the default) to let
 * the library choose per step from the bytes on the host link and the fixed cost
 * of a chunk (a step takes T (1 + 1/C) + C c). */
int monc_adv_set_chunks(monc_adv_t h, int nchunks);
/* The chunk count an automatic step would take for this shape, nfields_in arrays up and
 * nfields_out arrays down (3 + nq each for a full step; twice nfields_out up with
 * accumulate): the power of two nearest to sqrt(T / c).  Needs no handle and no GPU.
 * Returns the count (>= 1) or MONC_ADV_EINVAL. */
int monc_adv_plan_chunks(int nx, int ny, int nz, int halo, int dtype, int nfields_in, int nfields_out);
/* Chunk count of the step in flight (or of the last one); with a fixed count, that
 * count.  0 = automatic and no step enqueued yet. */
int monc_adv_step_chunk_count(monc_adv_t h);
/* 1 (default): copies and kernels overlap on separate streams.  0: the same
 * work serialised on one stream (H2D all, kernels, D2H all) -- the baseline
 * for the overlap ratio. */
int monc_adv_set_overlap(monc_adv_t h, int on);
/* MONC_ADV_FORM_FLUX (default) or MONC_ADV_FORM_PW_SKEW (PAPER.md:97 names the
 * Piacsek-Williams scheme; the centre value is
 * dropped from every advected-quantity parenthesis).  Both forms run on the
 * generic kernels and on the TMA kernels (variants 1 and 3). */
int monc_adv_set_form(monc_adv_t h, int form);
/* 0 (default): tendencies overwritten.  1: added into the output buffers (device
 * arrays of momentum / scalars / tendencies; host arrays of step_async, see there). */
int monc_adv_set_accumulate(monc_adv_t h, int on);
/* The paper's work-scaling experiment ("we have also scaled the workload
 * of the PW advection scheme to match that of the ULTIMATE scheme ... the GPU times
 * look very similar"; PAPER.md:97 puts ULTIMATE at about 16 x PW): every kernel
 * evaluates the flux arithmetic of a point n times (1 <= n <= 64, default 1) on the
 * same bytes.  Results are identical to n = 1.  Needs the flux form, overwrite mode
 * and the default (TMA) kernels: EINVAL otherwise, and for shapes whose nz is not a
 * multiple of 16 bytes / sizeof(dtype) the compute calls return EINVAL while n > 1. */
int monc_adv_set_work_scale(monc_adv_t h, int n);
/* 1 (default): monc_adv_tendencies and monc_adv_step_async use the fused
 * momentum + scalars launch where it fits.  0: always two launches. */
int monc_adv_set_fuse(monc_adv_t h, int on);
/* Copy the coefficient tables the handle uses to HOST arrays of nz doubles
 * (as stored, i.e. after rounding to fp32 for an F32 handle).  Any pointer
 * may be NULL. */
int monc_adv_get_coefficients(monc_adv_t h, double *tzc1, double *tzc2, double *tzd1,
                              double *tzd2);
/* Kernels launched by this handle since create (the caller's gpu_launches). */
long monc_adv_launch_count(monc_adv_t h);
/* Kernel and launch geometry of the last momentum and scalar launches of this
 * handle (text, for logs and bench records; "" before any launch).  The
 * pointer stays valid until the next call on the handle. */
const char *monc_adv_describe_plan(monc_adv_t h);
/* Text of the last error on this handle ("" if none).  h may be NULL: then the
 * text of the last failed monc_adv_create on this thread. */
const char *monc_adv_last_error(monc_adv_t h);
/* Library version string. */
const char *monc_adv_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MONC_ADV_H */
