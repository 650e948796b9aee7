/*
 * jefi.h -- C ABI of the B200 (sm_100a) library that evaluates the discretised Jefimenko
 * retarded-time sums for E(r,t) and B(r,t) (arxiv 2104.05426, "JefiGPU").
 *
 * What the library computes (Sec. 2.2 Eq. (4)-(6); readings Q1-Q8 of
 * DESIGN.md), per observation point r and evaluation step n (t = t0 + n*dt):
 *
 *   E(r,t) = dV/(4 pi) * sum_cells [ d*( rho/R^3 + rho_dot/(c R^2) ) - J_dot/(c^2 R) ]
 *   B(r,t) = dV/(4 pi) * sum_cells [ ( J/R^3 + J_dot/(c R^2) ) x d ]
 *
 *   d = r - r'_cell, R = |d|; rho, J, rho_dot, J_dot of that cell at the stored step
 *   m = n - floor(R/(c dt) + 0.5)  (Eq. (6): t_r = t - R/c, nearest stored snapshot);
 *   m < 0 contributes zero (the paper's sources vanish before t0);
 *   cells with R < 0.5*min(dx,dy,dz) are skipped (coarse screening);
 *   dV = dx*dy*dz of the source grid.
 *   Powers of c: the weights are exactly d/R^3, d/(c R^2), 1/(c^2 R) for E and 1/R^3, 1/(c R^2)
 *   for B, with NO overall power of c on B (BASELINE.json north_star lists them so).  That is a
 *   chosen convention, not a unit system: Heaviside-Lorentz, the paper's, would put
 *   1/c on B.  The paper and every benchmark config have c = 1, where all conventions agree; a
 *   caller with c != 1 who wants Heaviside-Lorentz B divides B_out by c.  An exact tie in the
 *   retarded step, q = R/(c dt) a half-integer, rounds UP (Q3 says what finite
 *   precision can and cannot decide there).
 *
 * Every step of that path runs in hand-written CUDA kernels; there is no CPU fallback and
 * no other backend.  All pointers named *_dev are DEVICE pointers of the context's dtype,
 * all pointers named *_host are HOST pointers; nothing here is a torch type.  Calls are
 * asynchronous on the given stream unless stated; one context must not be used from two
 * streams at the same time.  Errors are return codes only (nothing is thrown, nothing
 * aborts); argument errors are detected before any launch.
 */
#ifndef JEFI_H
#define JEFI_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct jefi_ctx jefi_ctx;          /* opaque; owned by the library */
typedef void* jefi_stream;                 /* a cudaStream_t (0 = legacy default stream) */

typedef enum {
    JEFI_OK = 0,
    JEFI_ERR_INVALID_ARG = 1,              /* null pointer, n <= 0, dt <= 0, c <= 0, bad range */
    JEFI_ERR_CUDA = 2,                     /* a CUDA runtime call or launch failed; see jefi_last_error */
    JEFI_ERR_OOM = 3,                      /* device allocation failed */
    JEFI_ERR_NO_HISTORY = 4,               /* jefi_fields before jefi_upload_history */
    JEFI_ERR_TIME_RANGE = 5,               /* step outside [0, nsteps-1] or t off the step grid */
    JEFI_ERR_UNSUPPORTED = 6               /* valid request this build does not implement */
} jefi_status;

typedef enum { JEFI_F32 = 0, JEFI_F64 = 1 } jefi_dtype;

/* A regular grid (source and observational regions each have their own sizes
 * and spacings and need not overlap).  origin = CENTRE of cell/point (0,0,0) (PAPER.md:137:
 * 15 cells x 0.4 span [-3,3], so samples are cell centres); index order x fastest:
 * linear index j = (k_z*n[1] + j_y)*n[0] + i_x.  All host fp64. */
typedef struct {
    int32_t n[3];
    double  origin[3];
    double  spacing[3];
} jefi_grid_desc;

/* Observation set.  kind 0: the regular grid `grid` (the paper's case).  kind 1: an explicit
 * list of `npoints` positions, points_dev[npoints][3] of the context dtype, device memory
 * owned by the caller.  The positions belong to the context as a grid does: jefi_create reads
 * them (it sorts the points into spatially compact tiles for the tiled kernel) and every
 * jefi_fields call reads them again; they must stay allocated and UNCHANGED until jefi_destroy.
 * Non-finite positions are JEFI_ERR_INVALID_ARG.  Outputs are always in the caller's order. */
typedef struct {
    int32_t        kind;
    jefi_grid_desc grid;
    int64_t        npoints;
    const void*    points_dev;
} jefi_obs_desc;

/* Stored history: nsteps snapshots m = 0..nsteps-1 at times t0 + m*dt (PAPER.md:231:
 * rho_GPU -> [rho_0 ... rho_lts]).  deriv_mode 0: centred time difference inside the stored
 * history, one-sided at both ends (BASELINE.json north_star (b)); 1: the paper's backward
 * difference (f(t_r) - f(t_r - dt))/dt with f = 0 before step 0.
 * past_mode must be 0 (zero before step 0). */
typedef struct {
    double  t0, dt, c;
    int32_t nsteps;
    int32_t deriv_mode;
    int32_t past_mode;
} jefi_time_desc;

/* Validates the descriptors, selects `device`, and allocates what the one-step calls need on
 * it (the series calls and the *_host uploads add their own buffers on first use, see there and
 * jefi_reserve_series): the packed history (32 bytes (fp32) / 64 bytes (fp64) per (cell, step), plus
 * one all-zero step standing for m < 0), the raw values of the two newest steps (for
 * jefi_append_step), partial-sum scratch, and the device output staging used by
 * jefi_fields_host.  For a regular observation grid no kernel is launched; for a point list
 * (kind 1) the tiling kernels run on the default stream and are waited for.  *out is written
 * only on success.  Synchronous. */
jefi_status jefi_create(const jefi_grid_desc* src, const jefi_obs_desc* obs,
                        const jefi_time_desc* time, jefi_dtype dtype, int device,
                        jefi_ctx** out);

/* Step a1 (pre-pass): reads rho_dev[nsteps][N_s] and J_dev[nsteps][3][N_s] (component planes;
 * the paper's four scalar fields rho, Jx, Jy, Jz), builds d(rho)/dt and dJ/dt and
 * writes the packed records.  The caller may free rho_dev/J_dev once `stream` has passed this
 * call.  May be called again to replace the history. */
jefi_status jefi_upload_history(jefi_ctx* ctx, const void* rho_dev, const void* J_dev,
                                jefi_stream stream);

/* Same, from HOST buffers (pinned for a truly asynchronous copy): copies them into a raw
 * device staging area owned by the context (allocated on first use) and runs the pre-pass on
 * `stream`.  The host-to-device copy itself is enqueued on a stream owned by the context and
 * `stream` waits for it, so in a stepping loop the copy of the next history overlaps the
 * pairwise kernel of the current step.  Consequence: the host buffers must hold their data when
 * this call is made (the copy is not ordered after earlier work on `stream`) and must stay
 * untouched until `stream` has passed this call. */
jefi_status jefi_upload_history_host(jefi_ctx* ctx, const void* rho_host, const void* J_host,
                                     jefi_stream stream);

/* Sliding window.  The paper keeps as many snapshots as the longest light-travel time needs,
 * lts = ceil(d_m/dt), resident on the GPU between calls, while the
 * source solver keeps producing new ones.  jefi_append_step drops the oldest stored
 * step and appends rho_new_dev[N_s], J_new_dev[3][N_s] as the new newest one: afterwards stored
 * step m holds what step m+1 held, t0 has advanced by dt, and nsteps is unchanged (evaluate the
 * new snapshot with step = nsteps-1).  Time derivatives follow deriv_mode: the new step gets
 * (f_new - f_prev)/dt; in centred mode the previous newest step is re-differenced to
 * (f_new - f_prev2)/(2 dt) now that it has a successor, and every other record -- the new oldest
 * one included -- keeps the value it had.  The packed history therefore equals, record for
 * record and bit for bit, the last nsteps records of a pre-pass over the (nsteps+1)-step raw
 * history [old steps..., new step].  Needs a prior jefi_upload_history (JEFI_ERR_NO_HISTORY).
 * One kernel on `stream`.  The stored steps of a cell form a ring inside the context, so the
 * call writes two records per cell -- O(N_s) bytes, whatever the history length. */
jefi_status jefi_append_step(jefi_ctx* ctx, const void* rho_new_dev, const void* J_new_dev,
                             jefi_stream stream);

/* Same from HOST buffers rho_new_host[N_s], J_new_host[3][N_s] (copied on `stream` into a
 * staging area owned by the context, allocated on first use). */
jefi_status jefi_append_step_host(jefi_ctx* ctx, const void* rho_new_host, const void* J_new_host,
                                  jefi_stream stream);

/* Steps a2-a6: E and B at evaluation step `step` (t = t0 + step*dt) for the observation
 * points obs_begin .. obs_begin+obs_count-1 (linear indices into the observation set).
 * E_out_dev / B_out_dev are [3][obs_count] component planes of the context dtype, owned by
 * the caller, fully overwritten, never accumulated into.  obs_count = 0 is a no-op. */
jefi_status jefi_fields(jefi_ctx* ctx, int32_t step, int64_t obs_begin, int64_t obs_count,
                        void* E_out_dev, void* B_out_dev, jefi_stream stream);

/* A time series in one call (the paper evaluates hundreds of snapshots on fixed grids,
 * PAPER.md:213-219; BASELINE.json configs[3] asks for 128 output steps): the fields of
 * step_begin, step_begin+1, ... as step_count calls of jefi_fields would give them (same
 * definition, same tolerances; not the same bits), outputs E_out_dev[step_count][3][obs_count],
 * B_out_dev likewise.  On regular observation grids with at least half a block of steps
 * (block = 6 steps in fp32, 4 in fp64) this runs the time-blocked kernel:
 * the geometry and the retarded lag of a (point, cell) pair do not depend on the evaluation
 * step (Eq. (6)), so a thread computes them once and walks a block of consecutive
 * output steps, whose retarded steps are consecutive stored snapshots; it reads a second copy
 * of the history ("series layout": the raw 16-byte {rho, J/c} record per (cell, step), time
 * differences formed in registers), which the context allocates on the first such call
 * (N_s x (nsteps+3) x 16 B (fp32) / 32 B (fp64); the partial-sum scratch is regrown on that call
 * too, to at most 1 GiB, if the series does not fit it) and rebuilds from the packed history after
 * every jefi_upload_history / jefi_append_step.  One known difference from step_count one-step
 * calls: after a jefi_append_step the rebuilt series layout differences the OLDEST stored step
 * one-sided from the stored values ((f[1] - f[0])/dt in centred mode, f[0]/dt in backward mode),
 * whereas the packed record of that step keeps the derivative it had before the append (see
 * jefi_append_step); only pairs whose retarded step is that oldest step are affected.  Other requests (point lists, one or two steps,
 * windows beyond shared memory) run step_count one-step evaluations.  All launches are enqueued
 * on `stream` back to back; step_count = 0 is a no-op. */
jefi_status jefi_fields_series(jefi_ctx* ctx, int32_t step_begin, int32_t step_count,
                               int64_t obs_begin, int64_t obs_count,
                               void* E_out_dev, void* B_out_dev, jefi_stream stream);

/* Same, results copied to HOST buffers [step_count][3][obs_count] on `stream` through a device
 * staging area owned by the context (allocated on first use, grown when a larger series is
 * asked for).  Returns after enqueueing; synchronise the stream before reading. */
jefi_status jefi_fields_series_host(jefi_ctx* ctx, int32_t step_begin, int32_t step_count,
                                    int64_t obs_begin, int64_t obs_count,
                                    void* E_out_host, void* B_out_host, jefi_stream stream);

/* The series calls above allocate on first use (series layout, a larger partial-sum scratch, the
 * host path's staging), and growing a buffer that earlier launches may still read waits for the
 * whole device (cudaDeviceSynchronize) before freeing it -- so the FIRST series call of a size is
 * not a pure enqueue.  A stepping loop that must stay asynchronous calls jefi_reserve_series once
 * beforehand: it makes those allocations for series of up to max_steps steps on up to max_obs
 * points (host_staging != 0: also the staging of jefi_fields_series_host).  Afterwards
 * jefi_fields_series[_host] within those limits call no cudaMalloc / cudaFree /
 * cudaDeviceSynchronize and jefi_device_bytes stays constant.  Synchronous; may be called again
 * with larger limits (buffers only grow); JEFI_ERR_INVALID_ARG unless 1 <= max_steps <= nsteps and
 * 1 <= max_obs <= N_o; JEFI_ERR_OOM if the layout or the staging does not fit (a scratch that
 * cannot be regrown is not an error: the series then runs in several batches). */
jefi_status jefi_reserve_series(jefi_ctx* ctx, int32_t max_steps, int64_t max_obs, int32_t host_staging);

/* Same for a time t that must lie on the step grid to within 1e-6*dt (the paper
 * evaluates at snapshots only), else JEFI_ERR_TIME_RANGE. */
jefi_status jefi_fields_at_time(jefi_ctx* ctx, double t, int64_t obs_begin, int64_t obs_count,
                                void* E_out_dev, void* B_out_dev, jefi_stream stream);

/* Same as jefi_fields, results copied to HOST buffers [3][obs_count] on `stream` (the paper
 * copies E, B to the host every step).  Returns after enqueueing; synchronise the
 * stream before reading. */
jefi_status jefi_fields_host(jefi_ctx* ctx, int32_t step, int64_t obs_begin, int64_t obs_count,
                             void* E_out_host, void* B_out_host, jefi_stream stream);

/* Kernel selection: 0 = automatic (tiled kernels for regular observation grids -- one-step for
 * jefi_fields, time-blocked for jefi_fields_series -- per-point kernel otherwise), 1 = always the
 * per-point kernel (one thread per observation point, the paper's shape PAPER.md:93), 2 = the
 * one-step tiled kernel or JEFI_ERR_UNSUPPORTED (jefi_fields_series then loops over it),
 * 3 = like 0, but jefi_fields_series of at least half a block of steps must run the
 * time-blocked kernel or fails with JEFI_ERR_UNSUPPORTED. */
jefi_status jefi_set_kernel(jefi_ctx* ctx, int32_t which);

/* Bytes of device memory owned by the context. */
int64_t     jefi_device_bytes(const jefi_ctx* ctx);

/* Waits for all work of the context's device; frees everything it owns. */
jefi_status jefi_destroy(jefi_ctx* ctx);

const char* jefi_status_string(jefi_status s);
/* Text of the last error of this context ("" if none); valid until the next call on it. */
const char* jefi_last_error(const jefi_ctx* ctx);
/* The fixed nominal operation count per (observation point, source cell) interaction: 52,
 * the flop count of the oracle's loop body. */
int         jefi_flops_per_pair(void);

/* Host-only helper for one-process-per-GPU runs (the paper's one source-observation pair per
 * GPU card): the contiguous slice [*begin, *begin + *count) of the observation
 * set that rank `rank` of `world` evaluates when one history is replicated and the observation
 * points are partitioned.  Slices are disjoint, cover the set in rank order, and are made of
 * whole z-layers of a regular grid when there are at least `world` layers (else whole x-rows,
 * else single points); sizes differ by at most one such granule.  Touches no device.
 * JEFI_ERR_INVALID_ARG on null pointers, world <= 0 or rank outside [0, world). */
jefi_status jefi_shard_obs(const jefi_obs_desc* obs, int32_t rank, int32_t world,
                           int64_t* begin, int64_t* count);

/* The other decomposition of the paper's Fig. 2: the SOURCE region is cut
 * and every rank evaluates the fields of its own sources at every observation point; the fields
 * are linear in rho and J (Eq. (4)-(5)), so one sum over the ranks (an all-reduce of the 6 N_o
 * values) gives the total.  Host-only helper: rank `rank` of `world` owns a contiguous run of
 * whole z-layers of `src` (sizes differ by at most one layer); *slab is the grid descriptor of
 * that run -- the same x, y extent and spacing, n[2] = its layers, origin[2] moved to its first
 * layer -- to be given to jefi_create as the source grid, and *cell_begin the linear index of its
 * first cell in the full grid: the rank's history is rows [cell_begin, cell_begin + slab cells) of
 * every rho[m][.] and J[m][comp][.].  A rank beyond the number of layers gets n[2] = 0 (nothing
 * to do; not a grid jefi_create accepts).  JEFI_ERR_INVALID_ARG on null pointers, a bad grid,
 * world <= 0 or rank outside [0, world).  Touches no device. */
jefi_status jefi_shard_src(const jefi_grid_desc* src, int32_t rank, int32_t world,
                           jefi_grid_desc* slab, int64_t* cell_begin);

/* Steps a2-a6 for callers that cannot allocate device memory.
 *
 * Every other entry point needs a jefi_ctx, and jefi_create cudaMallocs the packed history, the
 * partial-sum scratch and the staging buffers.  That rules the library out for two kinds of host:
 * a solver embedded in an application whose own memory pool has already taken all free device
 * memory (cudaMalloc just fails there), and a stepping loop that must never stall (cudaMalloc and
 * cudaFree synchronise the whole device).  jefi_fields_noalloc is for them: no context, and no
 * cudaMalloc, cudaFree or allocating library routine on any path through it.
 *
 * Same definition and same descriptors as jefi_create + jefi_upload_history + jefi_fields (Eq.
 * (4)-(6); screening PAPER.md:75; deriv_mode, rounding of the retarded step and
 * powers of c as stated at the top of this file), same tolerances against it, not the same bits.
 * The caller passes its own buffers: the raw history rho_dev[nsteps][N_s], J_dev[nsteps][3][N_s]
 * (device, `dtype`, read only, x fastest) and the outputs E_out_dev, B_out_dev [3][obs_count]
 * (device, `dtype`, fully overwritten); obs / obs_begin / obs_count / step as in jefi_fields;
 * time->t0 is not used.  A per-point kernel reads the raw snapshots and differences them in
 * time on the fly (no packed history), so it is far slower than the tiled kernels behind
 * jefi_fields -- it is meant for modest problems, not for the benchmark configurations.
 *
 * Scratch: the partial sums of the source chunks go to ONE fixed array of
 * JEFI_NOALLOC_SCRATCH_BYTES that is part of the library image; each GPU that loads libjefi.so
 * holds it until the process exits, used or not.  Hence the limit: obs_count larger than
 * JEFI_NOALLOC_MAX_OBS is refused with JEFI_ERR_UNSUPPORTED and a message saying so (split the
 * request into several calls, or use a context); N_s and nsteps are not limited.  All calls on
 * a device share that array: calls whose kernels may overlap on the GPU (two streams, no
 * ordering between them) race on it and give wrong fields; issue them on one stream or order
 * them with events.  A call never depends on what an earlier call left there.
 *
 * Works on the CURRENT device (cudaSetDevice is the caller's business; all pointers must belong
 * to it) and enqueues two kernels on `stream` without waiting for them.  The first call on each
 * device also does a one-time set-up (it asks the runtime where that device keeps the scratch
 * array); make that first call outside any stream capture.  Thread-safe as far as that set-up
 * goes.  `err` (host, may be NULL) receives a NUL-terminated message of at most err_len bytes on
 * failure and "" on success.  Arguments are checked before any CUDA call. */
#define JEFI_NOALLOC_SCRATCH_BYTES (8 * 1024 * 1024)
#define JEFI_NOALLOC_MAX_OBS       131072
jefi_status jefi_fields_noalloc(const jefi_grid_desc* src, const jefi_obs_desc* obs,
                                const jefi_time_desc* time, jefi_dtype dtype, int32_t step,
                                const void* rho_dev, const void* J_dev,
                                int64_t obs_begin, int64_t obs_count,
                                void* E_out_dev, void* B_out_dev, jefi_stream stream,
                                char* err, int32_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* JEFI_H */
