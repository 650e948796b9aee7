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
#include "tiled_common.cuh"

namespace jefi {
namespace {

template <typename T> struct Unit;                       // one 16-byte unit of a packed record
template <> struct alignas(16) Unit<float>  { float v[4]; };
template <> struct alignas(16) Unit<double> { double v[2]; };

constexpr int kThreads = 256;

// A CTA owns 128 cells and marches through the whole history in tiles of TT steps, keeping the
// last two raw rows of a tile as the first two of the next (no halo re-read: every raw value is
// read from HBM exactly once); a thread has 4*TT/8*4 = 32 independent row loads in flight.
// The transpose from the cell-fastest input to the step-fastest output goes through a padded
// shared-memory tile, so global reads (lanes along cells) and writes (lanes along steps, 16 B
// each) are both coalesced.  Measured on c3 (fp32, 2.78 GB): 0.66 ms = 4.2 TB/s.
constexpr int kCells2 = 128;

template <typename T, int TT>
__global__ void __launch_bounds__(kThreads)
prepass_march_kernel(const T* __restrict__ rho, const T* __restrict__ J, Unit<T>* __restrict__ hist,
                     long long Ns, int Tsteps, int Tp, T inv_dt, T inv_c, int deriv_mode, int seg_len)
{
    // blockIdx.y = time segment: packed steps [seg_len * blockIdx.y, + seg_len), seg_len a multiple
    // of TT (several segments only to have enough CTAs for full waves; each re-reads two rows)
    // raw[comp][row][cell(+1 pad)], row r <-> stored step m = p0 - 2 + r
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T (*raw)[TT + 2][kCells2 + 1] = reinterpret_cast<T (*)[TT + 2][kCells2 + 1]>(smem_raw);

    const long long j0 = (long long)blockIdx.x * kCells2;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int U = sizeof(T) == 4 ? 2 : 4, VPU = 8 / U;
    const T half = T(0.5), ic = inv_c, ic2 = inv_c * inv_c;

    const int p_begin = (int)blockIdx.y * seg_len;
    const int p_end = p_begin + seg_len < Tp ? p_begin + seg_len : Tp;
    for (int i = threadIdx.x; i < 4 * 2 * kCells2; i += kThreads) {
        const int comp = i / (2 * kCells2), r = (i / kCells2) % 2, cl = i % kCells2;
        const int m = p_begin - 2 + r;
        const long long j = j0 + cl;
        T v = T(0);
        if (m >= 0 && m < Tsteps && j < Ns)
            v = (comp == 0) ? rho[(long long)m * Ns + j] : J[((long long)m * 3 + (comp - 1)) * Ns + j];
        raw[comp][r][cl] = v;
    }

    for (int p0 = p_begin; p0 < p_end; p0 += TT) {
        for (int row = warp; row < 4 * TT; row += kThreads / 32) {
            const int comp = row / TT, r = 2 + row % TT;
            const int m = p0 - 2 + r;
            const T* src = (comp == 0) ? rho + (long long)m * Ns : J + ((long long)m * 3 + (comp - 1)) * Ns;
#pragma unroll
            for (int q = 0; q < kCells2 / 32; ++q) {
                const long long j = j0 + lane + 32 * q;
                raw[comp][r][lane + 32 * q] = (m < Tsteps && j < Ns) ? src[j] : T(0);
            }
        }
        __syncthreads();
        for (int i = threadIdx.x; i < kCells2 * TT; i += kThreads) {
            const int pl = i % TT, cl = i / TT;
            const int p = p0 + pl;
            const long long jj = j0 + cl;
            if (p >= Tp || jj >= Ns) continue;
            const int m = p - 1, r = pl + 1;
            T f[4], d[4];
#pragma unroll
            for (int comp = 0; comp < 4; ++comp) {
                if (p == 0) { f[comp] = T(0); d[comp] = T(0); continue; }
                const T fm = raw[comp][r][cl], fa = raw[comp][r - 1][cl], fb = raw[comp][r + 1][cl];
                T dd;
                if (deriv_mode == 1)        dd = (fm - fa) * inv_dt;
                else if (Tsteps == 1)       dd = T(0);
                else if (m == 0)            dd = (fb - fm) * inv_dt;
                else if (m == Tsteps - 1)   dd = (fm - fa) * inv_dt;
                else                        dd = (fb - fa) * (half * inv_dt);
                f[comp] = fm; d[comp] = dd;
            }
            const T val[8] = {f[0], d[0] * ic, f[1] * ic, f[2] * ic, f[3] * ic, d[1] * ic2, d[2] * ic2, d[3] * ic2};
#pragma unroll
            for (int u = 0; u < U; ++u) {
                Unit<T> q;
#pragma unroll
                for (int e = 0; e < VPU; ++e) q.v[e] = val[u * VPU + e];
                hist[(jj * U + u) * Tp + p] = q;
            }
        }
        __syncthreads();
        for (int i = threadIdx.x; i < 4 * 2 * kCells2; i += kThreads) {
            const int comp = i / (2 * kCells2), r = (i / kCells2) % 2, c = i % kCells2;
            raw[comp][r][c] = raw[comp][TT + r][c];
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// Sliding window (the history holds lts = ceil(d_m/dt) snapshots, i.e. as far back
// as the longest delay; it stays on the GPU between calls).  The stored steps of a
// row form a ring (tiled_common.cuh ring_slot): append_kernel overwrites the slot of the OLDEST
// step with the record of the new newest one (one-sided derivative (f_new - f_prev)/dt) and,
// in centred mode, re-differences the previous newest step now that its successor exists:
// (f_new - f_prev2)/(2 dt); the host then advances the ring origin by one.  Two records per
// (cell, unit) are written, whatever the history length.  `last` holds the raw values of the
// two newest steps ([2][4][N_s]: step T-2, step T-1; component 0 = rho, 1..3 = J) so that both
// records are bit-identical to what the pre-pass makes of the same raw history.  One thread per cell.
template <typename T>
__device__ __forceinline__ void pack_record(const T (&f)[4], const T (&d)[4], T inv_c, T (&val)[8])
{
    const T ic = inv_c, ic2 = inv_c * inv_c;
    val[0] = f[0];      val[1] = d[0] * ic;  val[2] = f[1] * ic;  val[3] = f[2] * ic;
    val[4] = f[3] * ic; val[5] = d[1] * ic2; val[6] = d[2] * ic2; val[7] = d[3] * ic2;
}

template <typename T>
__global__ void __launch_bounds__(kThreads)
append_kernel(const T* __restrict__ rho_new, const T* __restrict__ J_new, T* last, Unit<T>* hist, long long Ns, int Tsteps,
              int Tp, int origin, T inv_dt, T inv_c, int deriv_mode)
{
    constexpr int U = sizeof(T) == 4 ? 2 : 4, VPU = 8 / U;
    const long long j = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (j >= Ns) return;

    T fn[4], fp[4], fq[4], dn[4], dp[4];
#pragma unroll
    for (int comp = 0; comp < 4; ++comp) {
        fn[comp] = comp == 0 ? rho_new[j] : J_new[(long long)(comp - 1) * Ns + j];
        fq[comp] = last[(long long)(0 * 4 + comp) * Ns + j];      // step T-2
        fp[comp] = last[(long long)(1 * 4 + comp) * Ns + j];      // step T-1
        dn[comp] = (fn[comp] - fp[comp]) * inv_dt;
        dp[comp] = (fn[comp] - fq[comp]) * (T(0.5) * inv_dt);
    }
    T vn[8], vp[8];
    pack_record<T>(fn, dn, inv_c, vn);
    pack_record<T>(fp, dp, inv_c, vp);
    const bool redo_prev = deriv_mode == 0 && Tsteps >= 2;
    // `origin` is the ring origin BEFORE this append: the oldest step (p = 1) sits at slot
    // 1 + origin and becomes the new newest one; the previous newest (p = T) sits one slot before it
    const int slot_new = 1 + origin;
    const int slot_prev = 1 + (origin + Tsteps - 1) % Tsteps;
#pragma unroll
    for (int u = 0; u < U; ++u) {
        Unit<T>* row = hist + (j * U + u) * Tp;
        Unit<T> q;
#pragma unroll
        for (int e = 0; e < VPU; ++e) q.v[e] = vn[u * VPU + e];
        row[slot_new] = q;
        if (redo_prev) {
#pragma unroll
            for (int e = 0; e < VPU; ++e) q.v[e] = vp[u * VPU + e];
            row[slot_prev] = q;
        }
    }
#pragma unroll
    for (int comp = 0; comp < 4; ++comp) {
        last[(long long)(0 * 4 + comp) * Ns + j] = fp[comp];
        last[(long long)(1 * 4 + comp) * Ns + j] = fn[comp];
    }
}

}  // namespace

int launch_prepass(const Params& P, jefi_dtype dt, const void* rho, const void* J, void* hist,
                   cudaStream_t stream)
{
    const unsigned blocks = (unsigned)((P.Ns + kCells2 - 1) / kCells2);
    constexpr int TT = 16;
    // time segments: aim at >= 8 waves of CTAs (a CTA marches through its whole segment, so a
    // partial last wave costs up to one CTA's run time)
    int sm_count = 148, dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev);
    const int tiles_t = (P.Tp + TT - 1) / TT;
    long long want = (8LL * sm_count * 6 + blocks - 1) / blocks;
    if (want < 1) want = 1;
    if (want > tiles_t) want = tiles_t;
    const int seg_tiles = (int)((tiles_t + want - 1) / want);
    const int seg_len = seg_tiles * TT;
    const dim3 grid(blocks, (unsigned)((tiles_t + seg_tiles - 1) / seg_tiles));
    if (dt == JEFI_F32) {
        const int smem = 4 * (TT + 2) * (kCells2 + 1) * (int)sizeof(float);
        auto kern = prepass_march_kernel<float, TT>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return -1;
        kern<<<grid, kThreads, smem, stream>>>((const float*)rho, (const float*)J, (Unit<float>*)hist, P.Ns, P.T,
                                               P.Tp, (float)(1.0 / P.dt), (float)(1.0 / P.c), P.deriv_mode, seg_len);
    } else {
        const int smem = 4 * (TT + 2) * (kCells2 + 1) * (int)sizeof(double);
        auto kern = prepass_march_kernel<double, TT>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return -1;
        kern<<<grid, kThreads, smem, stream>>>((const double*)rho, (const double*)J, (Unit<double>*)hist, P.Ns, P.T,
                                               P.Tp, 1.0 / P.dt, 1.0 / P.c, P.deriv_mode, seg_len);
    }
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_append(const Params& P, jefi_dtype dt, const void* rho_new, const void* J_new, void* last,
                  void* hist, cudaStream_t stream)
{
    const unsigned blocks = (unsigned)((P.Ns + kThreads - 1) / kThreads);
    if (dt == JEFI_F32)
        append_kernel<float><<<blocks, kThreads, 0, stream>>>(
            (const float*)rho_new, (const float*)J_new, (float*)last, (Unit<float>*)hist, P.Ns, P.T, P.Tp, P.origin,
            (float)(1.0 / P.dt), (float)(1.0 / P.c), P.deriv_mode);
    else
        append_kernel<double><<<blocks, kThreads, 0, stream>>>(
            (const double*)rho_new, (const double*)J_new, (double*)last, (Unit<double>*)hist, P.Ns, P.T, P.Tp, P.origin,
            1.0 / P.dt, 1.0 / P.c, P.deriv_mode);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace jefi
