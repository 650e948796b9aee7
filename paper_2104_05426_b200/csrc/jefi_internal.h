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
    double  dt, c;
    int     deriv_mode;
};

// Packed history layout: for cell j, half h in {0,1},
// packed step p in [0, Tp):  vec4 at index (j*2 + h)*Tp + p
//   half 0 = { rho, rho_dot/c, Jx/c, Jy/c },  half 1 = { Jz/c, Jx_dot/c^2, Jy_dot/c^2, Jz_dot/c^2 }
// so that a retarded-time window of one cell is one contiguous run of 16-byte (fp32) or
// 32-byte (fp64) elements.

struct FieldsLaunch {
    int       step;        // evaluation step n
    long long obs_begin, obs_count;
    void*     E_out;       // [3][obs_count]
    void*     B_out;
    void*     scratch;     // partial sums [S][6][obs_count]
    long long scratch_elems;
    int       sm_count;
    cudaStream_t stream;
};

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

double measure_alu_peak(jefi_dtype dt, int sm_count, int clock_khz);

}  // namespace jefi
