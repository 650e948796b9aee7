// jefi_internal.h -- context and kernel-launcher declarations shared by the .cu files of
// libjefi.so.  Not part of the ABI (include/jefi.h is).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "jefi.h"

namespace jefi {

// Geometry and time parameters every kernel needs, passed by value (host fp64; kernels
// convert to their own precision).
struct Params {
    int     ns[3];          // source cells per axis
    double  so[3];          // centre of source cell (0,0,0)
    double  sh[3];          // source spacing
    int     no[3];          // observation grid points per axis (kind 0)
    double  oo[3];          // centre of obs point (0,0,0)
    double  oh[3];          // obs spacing
    int     obs_kind;       // 0 grid, 1 explicit points
    long long n_obs;        // total observation points
    const void* obs_points; // kind 1: [n_obs][3] device, ctx dtype
    long long Ns;           // source cells
    int     T;              // stored steps
    int     Tp;             // T + 1: packed steps p = m + 1, p = 0 is the all-zero record
    int     origin;         // ring origin of the packed history (tiled_common.cuh ring_slot)
    double  dt, c;
    int     deriv_mode;
};

// Packed history layout: 16-byte units, U per record (fp32: 2
// float4, fp64: 4 double2); for cell j, unit u, packed step p in [0, Tp): unit index (j*U + u)*Tp + p.
// The 8 values of a record in unit order:
//   { rho, rho_dot/c, Jx/c, Jy/c | Jz/c, Jx_dot/c^2, Jy_dot/c^2, Jz_dot/c^2 }
// so that a retarded-time window of one cell is one contiguous run of 16-byte elements per unit.

struct FieldsLaunch {
    int       step;        // evaluation step n
    long long obs_begin, obs_count;
    void*     E_out;       // [3][obs_count]
    void*     B_out;
    void*     scratch;     // partial sums [S][6][obs_count]
    long long scratch_elems;
    long long chunk_bytes;  // a source chunk's packed history stays below this (L2 sharing)
    int       sm_count;
    cudaStream_t stream;
};

// Explicit point lists on the tiled path (pairwise_list.cu): jefi_create sorts the points into
// spatially compact tiles -- perm[s] = original index of entry s of the sorted order,
// boxes[tile][6] = min xyz, max xyz of the tile relative to source cell (0,0,0)
struct PointTiles {
    int*      perm;
    double*   boxes;
    long long ntiles;
    int       tile_points;
    double    max_diam;     // longest tile-box diagonal
    double    far;          // bound on the distance between any point and any source cell
};
int list_tile_points(jefi_dtype dt);
// synchronous; returns kernels launched, -1 on a CUDA error, -2 on non-finite positions
int build_point_tiles(const Params& P, jefi_dtype dt, PointTiles& pt);
// whole-list requests only; returns 0 if it does not support the request
struct FieldsLaunch;
int launch_fields_list(const Params& P, jefi_dtype dt, const void* hist, const FieldsLaunch& L, const PointTiles& pt);

// each returns the number of kernels it launched (>0) or a negative value on a launch error,
// leaving the CUDA error in cudaGetLastError()/cudaPeekAtLastError()
int launch_prepass(const Params& P, jefi_dtype dt, const void* rho, const void* J, void* hist,
                   cudaStream_t stream);
// sliding window: drop the oldest step, append (rho_new[N_s], J_new[3][N_s]); `last` = raw values
// of the two newest steps, [2][4][N_s]
int launch_append(const Params& P, jefi_dtype dt, const void* rho_new, const void* J_new, void* last,
                  void* hist, cudaStream_t stream);
int launch_fields_point(const Params& P, jefi_dtype dt, const void* hist, const FieldsLaunch& L);
// tiled kernel: regular observation grids only; returns 0 if it does not support the request
int launch_fields_tiled(const Params& P, jefi_dtype dt, const void* hist, const FieldsLaunch& L);
int launch_reduce_scale(const Params& P, jefi_dtype dt, const FieldsLaunch& L, int S);
// time-blocked kernel (pairwise_series.cu): the series layout (raw 16-byte
// records [cell][unit][T+3]) is built from the packed history; launch_fields_series evaluates
// step_count consecutive steps into E_out/B_out [step][3][obs_count]; returns 0 if unsupported
int launch_series_layout(const Params& P, jefi_dtype dt, const void* packed, void* series, cudaStream_t stream);
int launch_fields_series(const Params& P, jefi_dtype dt, const void* series, const FieldsLaunch& L, int step_begin,
                         int step_count);
int series_block_steps(jefi_dtype dt);

}  // namespace jefi

// the context behind the opaque handle of include/jefi.h (defined here so that the instrumentation
// entry points of include/jefi_instrument.h, in instrument.cu, can read it)
struct jefi_ctx {
    jefi::Params P;
    jefi_dtype   dtype;
    int          device;
    double       t0;
    int          sm_count;
    size_t       elem;             // sizeof(float|double)
    void*        hist;             // packed history, [N_s][units][Tp], 16-byte units
    size_t       hist_bytes;
    void*        scratch;          // partial sums (double)
    long long    scratch_elems;    // what the launchers may use (= allocated, unless a test caps it)
    long long    scratch_alloc_elems;
    long long    chunk_bytes;      // packed-history bytes per source chunk (L2 sharing, pairwise_tiled.cu)
    void*        stage_E;          // device staging for jefi_fields_host, [3][N_o]
    void*        stage_B;
    void*        stage_series;     // device staging for jefi_fields_series_host (lazy, grows), E then B
    size_t       stage_series_bytes;
    jefi::PointTiles tiles;        // kind 1 observation sets: the tiling built by jefi_create
    void*        series;           // series layout of the history (lazy: first jefi_fields_series), [N_s][units][T+3]
    bool         series_valid;     // matches the packed history
    void*        last;             // raw values of the two newest stored steps, [2][4][N_s]
    void*        new_stage;        // device staging for jefi_append_step_host, [4][N_s] (lazy)
    void*        raw_rho;          // device staging for jefi_upload_history_host (lazy)
    void*        raw_J;
    cudaStream_t copy_stream;      // H2D of the raw history runs here, beside the caller's stream
    cudaEvent_t  ev_copied;        // copy_stream: raw staging filled
    cudaEvent_t  ev_raw_free;      // caller's stream: the pre-pass has consumed the raw staging
    bool         raw_in_use;
    bool         has_history;
    int          kernel_choice;
    long long    launches;
    long long    dev_bytes;
    char         err[512];
};

