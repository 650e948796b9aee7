// prepass.cu -- step a1 (K2): time derivatives + record packing.
//
// Reads the raw history rho[T][N_s], J[T][3][N_s] once, forms
// d(rho)/dt and dJ/dt (BASELINE.json north_star (b): centred differences; deriv_mode 1 keeps the
// paper's backward difference of Eq. (4)-(5)) and writes, per (cell, step), two
// aligned vec4 half-records with the powers of c folded in:
//     half 0 = { rho, rho_dot/c, Jx/c, Jy/c }     half 1 = { Jz/c, Jx_dot/c^2, Jy_dot/c^2, Jz_dot/c^2 }
// In these variables Eq. (4)-(5) read  E = sum d (rho/R^3 + rho_dot'/R^2) - J_dot''/R  and
// B = c * sum (J'/R^3 + J_dot''/R^2) x d, so the pairwise kernel never sees c.
//
// Output order is [cell][unit][p], p = m + 1 (p = 0: all-zero record standing for every step
// before the stored history), in 16-byte units: fp32 has two units per record (the two float4
// halves above), fp64 has four (double2: {rho, rho_dot'}, {Jx', Jy'}, {Jz', Jx_dot''},
// {Jy_dot'', Jz_dot''}), so that consecutive steps of one unit are always 16 bytes apart and a
// retarded-time window of one cell is one contiguous run per unit.
// HBM-bound: 16 B read + 32 B written per record (fp32); the transpose from the cell-fastest
// input to the time-fastest output goes through a padded shared-memory tile so that both the
// global reads (lanes along cells) and the global writes (lanes along steps) are coalesced.
#include "jefi_internal.h"

namespace jefi {
namespace {

template <typename T> struct Unit;                       // one 16-byte unit of a packed record
template <> struct alignas(16) Unit<float>  { float v[4]; };
template <> struct alignas(16) Unit<double> { double v[2]; };

constexpr int kCells = 32;     // cells per tile
constexpr int kThreads = 256;

template <typename T, int TT>
__global__ void __launch_bounds__(kThreads)
prepass_kernel(const T* __restrict__ rho, const T* __restrict__ J, Unit<T>* __restrict__ hist,
               long long Ns, int Tsteps, int Tp, T inv_dt, T inv_c, int deriv_mode)
{
    // raw[comp][row][cell(+1 pad)], row r <-> stored step m = p0 - 2 + r  (one halo row each side)
    __shared__ T raw[4][TT + 2][kCells + 1];

    const long long j0 = (long long)blockIdx.x * kCells;
    const int p0 = blockIdx.y * TT;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long j = j0 + lane;

    for (int row = warp; row < 4 * (TT + 2); row += kThreads / 32) {
        const int comp = row / (TT + 2), r = row % (TT + 2);
        const int m = p0 - 2 + r;
        T v = T(0);
        if (m >= 0 && m < Tsteps && j < Ns) {
            v = (comp == 0) ? rho[(long long)m * Ns + j]
                            : J[((long long)m * 3 + (comp - 1)) * Ns + j];
        }
        raw[comp][r][lane] = v;
    }
    __syncthreads();

    const T half = T(0.5);
    for (int i = threadIdx.x; i < kCells * TT; i += kThreads) {
        const int pl = i % TT, cl = i / TT;
        const int p = p0 + pl;
        const long long jj = j0 + cl;
        if (p >= Tp || jj >= Ns) continue;
        const int m = p - 1, r = pl + 1;               // row of step m
        T f[4], d[4];
#pragma unroll
        for (int comp = 0; comp < 4; ++comp) {
            if (p == 0) { f[comp] = T(0); d[comp] = T(0); continue; }
            const T fm = raw[comp][r][cl];
            const T fa = raw[comp][r - 1][cl];         // step m-1 (0 if m == 0)
            const T fb = raw[comp][r + 1][cl];         // step m+1 (0 if m == T-1)
            T dd;
            if (deriv_mode == 1)        dd = (fm - fa) * inv_dt;                 // paper, f[-1] = 0
            else if (Tsteps == 1)       dd = T(0);
            else if (m == 0)            dd = (fb - fm) * inv_dt;
            else if (m == Tsteps - 1)   dd = (fm - fa) * inv_dt;
            else                        dd = (fb - fa) * (half * inv_dt);
            f[comp] = fm; d[comp] = dd;
        }
        const T ic = inv_c, ic2 = inv_c * inv_c;
        const T val[8] = {f[0], d[0] * ic, f[1] * ic, f[2] * ic, f[3] * ic, d[1] * ic2, d[2] * ic2, d[3] * ic2};
        constexpr int U = sizeof(T) == 4 ? 2 : 4;                  // units per record
        constexpr int VPU = 8 / U;                               // values per unit
#pragma unroll
        for (int u = 0; u < U; ++u) {
            Unit<T> q;
#pragma unroll
            for (int e = 0; e < VPU; ++e) q.v[e] = val[u * VPU + e];
            hist[(jj * U + u) * Tp + p] = q;
        }
    }
}

}  // namespace

int launch_prepass(const Params& P, jefi_dtype dt, const void* rho, const void* J, void* hist,
                   cudaStream_t stream)
{
    const unsigned gx = (unsigned)((P.Ns + kCells - 1) / kCells);
    if (dt == JEFI_F32) {
        constexpr int TT = 64;
        dim3 grid(gx, (unsigned)((P.Tp + TT - 1) / TT));
        prepass_kernel<float, TT><<<grid, kThreads, 0, stream>>>(
            (const float*)rho, (const float*)J, (Unit<float>*)hist, P.Ns, P.T, P.Tp,
            (float)(1.0 / P.dt), (float)(1.0 / P.c), P.deriv_mode);
    } else {
        constexpr int TT = 32;
        dim3 grid(gx, (unsigned)((P.Tp + TT - 1) / TT));
        prepass_kernel<double, TT><<<grid, kThreads, 0, stream>>>(
            (const double*)rho, (const double*)J, (Unit<double>*)hist, P.Ns, P.T, P.Tp,
            1.0 / P.dt, 1.0 / P.c, P.deriv_mode);
    }
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace jefi
