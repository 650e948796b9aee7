// instrument.cu -- the entry points of include/jefi_instrument.h: launch counter, the register-only
// FFMA / DFMA chains the bench states beside its ALU peak, and the retarded-lag dump of the
// parity report.  Measurement and test instrumentation, not product path:
// nothing in jefi.h's entry points calls into this file.
#include "tiled_common.cuh"
#include "jefi_instrument.h"

namespace jefi {
namespace {

// ------------------------------------------------------------------ ALU peak chains
template <typename T>
__global__ void __launch_bounds__(256)
fma_chain_kernel(T* out, T a, T b, int iters)
{
    T x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = x0 * a + b; x1 = x1 * a + b; x2 = x2 * a + b; x3 = x3 * a + b;
            x4 = x4 * a + b; x5 = x5 * a + b; x6 = x6 * a + b; x7 = x7 * a + b;
        }
    }
    const T s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == T(-12345.678)) out[0] = s;       // never true; keeps the chains alive
}

template <typename T>
double run_chain(int sm_count)
{
    T* out = nullptr;
    if (cudaMalloc(&out, 64) != cudaSuccess) return -1.0;
    const int iters = sizeof(T) == 4 ? 4096 : 2048;
    const int blocks = sm_count * 8;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = -1.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0);
        fma_chain_kernel<T><<<blocks, 256>>>(out, T(0.999), T(0.001), iters);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 64.0 * (double)iters * 256.0 * (double)blocks;
        const double tf = flops / (ms * 1e-3) * 1e-12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    return best;
}

// FP32 FFMA rate as a function of where the operands come from (what bounds
// the time-blocked kernel once the shared-memory gather is relieved).  MODE 0: 64 accumulators,
// acc += v[j % 8] * w -- two fresh register reads (accumulator, value) and one the operand-reuse
// cache serves (w); MODE 1: acc += v[a] * u[b] with all three registers fresh.
template <int MODE>
__global__ void __launch_bounds__(256)
ffma_operand_kernel(float* out, const float* in, int iters)
{
    float acc[64], v[32], u[32];
    for (int i = 0; i < 64; ++i) acc[i] = threadIdx.x + i;
    for (int i = 0; i < 32; ++i) { v[i] = in[i + threadIdx.x]; u[i] = in[i + 64 + threadIdx.x]; }
    float w = in[100 + threadIdx.x];
    for (int it = 0; it < iters; ++it) {
        if (MODE == 0) {
#pragma unroll
            for (int j = 0; j < 64; ++j) acc[j] = fmaf(v[j % 8], w, acc[j]);
            w += 1e-9f;
        } else {
#pragma unroll
            for (int j = 0; j < 64; ++j) acc[j] = fmaf(v[j % 32], u[(j * 7 + 3) % 32], acc[j]);
        }
    }
    float s = 0;
    for (int i = 0; i < 64; ++i) s += acc[i];
    if (s == -12345.678f) out[0] = s;
}

template <int MODE>
double run_operand(int sm_count)
{
    float *out = nullptr, *in = nullptr;
    if (cudaMalloc(&out, 64) != cudaSuccess || cudaMalloc(&in, 4096) != cudaSuccess) return -1.0;
    cudaMemset(in, 0, 4096);
    const int iters = 2048, blocks = sm_count * 8;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = -1.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0);
        ffma_operand_kernel<MODE><<<blocks, 256>>>(out, in, iters);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        const double tf = 2.0 * 64.0 * iters * 256.0 * blocks / (ms * 1e-3) * 1e-12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out); cudaFree(in);
    return best;
}

// ------------------------------------------------------------------ lag dump
struct LagArgs {
    int nsx, nsy, nsz, nox, noy;
    float tie_lim_list;         // the list kernel's near-tie threshold (pairwise_list.cu), 0 = no list tiling
    double shx, shy, shz, ohx, ohy, ohz, d0x, d0y, d0z, sox, soy, soz;
    double rcut2, inv_cdt;
    int obs_kind, which;
    const void* points;
};

// One thread per requested pair; positions and lag formed by the SAME inlined helpers the
// pairwise kernels call (tiled_common.cuh: obs_coord, src_coord, row_ryz, pair_geo / point_geo).
template <typename T>
__global__ void __launch_bounds__(256)
lag_dump_kernel(const long long* __restrict__ obs_idx, const long long* __restrict__ cell_idx, int* __restrict__ out,
                long long n, LagArgs a)
{
    const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
    if (t >= n) return;
    const long long gi = obs_idx[t], j = cell_idx[t];
    const int jx = (int)(j % a.nsx), jy = (int)((j / a.nsx) % a.nsy), jz = (int)(j / ((long long)a.nsx * a.nsy));
    T ox, oy, oz;
    double pdx = 0, pdy = 0, pdz = 0;
    if (a.obs_kind == 0) {
        const int ix = (int)(gi % a.nox), iy = (int)((gi / a.nox) % a.noy);
        const int iz = (int)(gi / ((long long)a.nox * a.noy));
        ox = obs_coord<T>(a.d0x, ix, a.ohx); oy = obs_coord<T>(a.d0y, iy, a.ohy); oz = obs_coord<T>(a.d0z, iz, a.ohz);
    } else {
        const T* p = (const T*)a.points + 3 * gi;
        pdx = (double)p[0] - a.sox; pdy = (double)p[1] - a.soy; pdz = (double)p[2] - a.soz;
        ox = (T)pdx; oy = (T)pdy; oz = (T)pdz;
    }
    // fp32 on a point list: the kernels redo near-tie lags in fp64 (tiled_common.cuh tie_delta,
    // near_tie_lag); the same test with the same threshold each of them uses
    const bool fix_ties = sizeof(T) == 4 && a.obs_kind == 1;
    T dy, dz, dx, w;
    const T ryz = row_ryz<T>(oy, oz, jy, jz, (T)a.shy, (T)a.shz, dy, dz);
    int k;
    if (a.which == 1) {
        point_geo<T>(ox, jx, (T)a.shx, ryz, (T)a.rcut2, -tie_biased_neg_inv_cdt<T>(a.inv_cdt), dx, w, k);
        if (fix_ties) {
            const double fx = fmax(fabs(pdx), fabs(pdx - (a.nsx - 1) * a.shx));
            const double fy = fmax(fabs(pdy), fabs(pdy - (a.nsy - 1) * a.shy));
            const double fz = fmax(fabs(pdz), fabs(pdz - (a.nsz - 1) * a.shz));
            const T tie_lim = (T)(0.5f - tie_delta(sqrt(fx * fx + fy * fy + fz * fz) * a.inv_cdt));
            const T e = (dx * dx + ryz) * w * (T)a.inv_cdt - (T)k;
            if ((e < T(0) ? -e : e) >= tie_lim && w != T(0))
                k = near_tie_lag(pdx, pdy, pdz, jx, jy, jz, a.shx, a.shy, a.shz, a.inv_cdt);
        }
    } else {
        unsigned bits;
        T R;
        // (the SLOW variant: the one the kernels run wherever a pair can be as close as R = 0, and
        // identical to the fast one for every R2 >= 1e-30)
        pair_geo_r<T, true>(ox, src_coord<T>(jx, a.shx), ryz, tie_biased_neg_inv_cdt<T>(a.inv_cdt), (T)a.rcut2, dx, w, bits, R);
        k = lag_of_bits(bits, Prec<T>::kMagicLo);
        if (fix_ties) {
            const float e = fmaf((float)R, (float)(-a.inv_cdt), (float)k);
            if (fabsf(e) >= a.tie_lim_list) k = near_tie_lag(pdx, pdy, pdz, jx, jy, jz, a.shx, a.shy, a.shz, a.inv_cdt);
        }
    }
    out[t] = k;
}

}  // namespace
}  // namespace jefi

extern "C" {

int64_t jefi_launch_count(const jefi_ctx* ctx) { return ctx ? ctx->launches : 0; }

jefi_status jefi_measure_alu_peak(int device, jefi_dtype dtype, double* tflops)
{
    if (!tflops || device < 0 || (dtype != JEFI_F32 && dtype != JEFI_F64)) return JEFI_ERR_INVALID_ARG;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return JEFI_ERR_CUDA; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaGetLastError(); return JEFI_ERR_CUDA; }
    const double v = dtype == JEFI_F32 ? jefi::run_chain<float>(prop.multiProcessorCount)
                                       : jefi::run_chain<double>(prop.multiProcessorCount);
    if (v < 0) { cudaGetLastError(); return JEFI_ERR_CUDA; }
    *tflops = v;
    return JEFI_OK;
}

jefi_status jefi_measure_ffma_operand_rates(int device, double* two_fresh_tflops, double* three_fresh_tflops)
{
    if (!two_fresh_tflops || !three_fresh_tflops || device < 0) return JEFI_ERR_INVALID_ARG;
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return JEFI_ERR_CUDA; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaGetLastError(); return JEFI_ERR_CUDA; }
    const double a = jefi::run_operand<0>(prop.multiProcessorCount), b = jefi::run_operand<1>(prop.multiProcessorCount);
    if (a < 0 || b < 0) { cudaGetLastError(); return JEFI_ERR_CUDA; }
    *two_fresh_tflops = a; *three_fresh_tflops = b;
    return JEFI_OK;
}

jefi_status jefi_debug_pair_lags(jefi_ctx* ctx, int32_t which, int64_t n_pairs, const int64_t* obs_index_dev,
                                 const int64_t* cell_index_dev, int32_t* lag_out_dev, jefi_stream stream)
{
    if (!ctx || (which != 1 && which != 2) || n_pairs < 0) return JEFI_ERR_INVALID_ARG;
    if (n_pairs == 0) return JEFI_OK;
    if (!obs_index_dev || !cell_index_dev || !lag_out_dev) return JEFI_ERR_INVALID_ARG;
    const jefi::Params& P = ctx->P;
    if (which == 2 && P.obs_kind != 0 && !ctx->tiles.perm) return JEFI_ERR_UNSUPPORTED;
    if (cudaSetDevice(ctx->device) != cudaSuccess) { cudaGetLastError(); return JEFI_ERR_CUDA; }
    jefi::LagArgs a;
    a.nsx = P.ns[0]; a.nsy = P.ns[1]; a.nsz = P.ns[2]; a.nox = P.no[0]; a.noy = P.no[1];
    a.tie_lim_list = P.obs_kind != 0 && ctx->tiles.perm ? 0.5f - jefi::tie_delta(ctx->tiles.far / (P.c * P.dt)) : 0.f;
    a.shx = P.sh[0]; a.shy = P.sh[1]; a.shz = P.sh[2];
    a.ohx = P.oh[0]; a.ohy = P.oh[1]; a.ohz = P.oh[2];
    a.d0x = P.oo[0] - P.so[0]; a.d0y = P.oo[1] - P.so[1]; a.d0z = P.oo[2] - P.so[2];
    a.sox = P.so[0]; a.soy = P.so[1]; a.soz = P.so[2];
    double hmin = P.sh[0] < P.sh[1] ? P.sh[0] : P.sh[1];
    hmin = hmin < P.sh[2] ? hmin : P.sh[2];
    a.rcut2 = 0.25 * hmin * hmin;
    a.inv_cdt = 1.0 / (P.c * P.dt);
    a.obs_kind = P.obs_kind; a.which = which; a.points = P.obs_points;
    const unsigned blocks = (unsigned)((n_pairs + 255) / 256);
    if (ctx->dtype == JEFI_F32)
        jefi::lag_dump_kernel<float><<<blocks, 256, 0, (cudaStream_t)stream>>>(
            (const long long*)obs_index_dev, (const long long*)cell_index_dev, lag_out_dev, n_pairs, a);
    else
        jefi::lag_dump_kernel<double><<<blocks, 256, 0, (cudaStream_t)stream>>>(
            (const long long*)obs_index_dev, (const long long*)cell_index_dev, lag_out_dev, n_pairs, a);
    if (cudaPeekAtLastError() != cudaSuccess) { cudaGetLastError(); return JEFI_ERR_CUDA; }
    ctx->launches += 1;
    return JEFI_OK;
}

jefi_status jefi_debug_launch_limits(jefi_ctx* ctx, int64_t scratch_elems, int64_t chunk_bytes)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    if (scratch_elems > 0) {
        long long e = scratch_elems < 6 * ctx->P.n_obs ? 6 * ctx->P.n_obs : scratch_elems;
        if (e > ctx->scratch_alloc_elems) e = ctx->scratch_alloc_elems;
        ctx->scratch_elems = e;
    }
    if (chunk_bytes > 0) ctx->chunk_bytes = chunk_bytes;
    return JEFI_OK;
}

}  // extern "C"
