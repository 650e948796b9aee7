// alu_peak.cu -- register-only FFMA / DFMA chains: the ALU peak the bench divides by
// (MEASURED_PEAKS.json carries no FP32/FP64 figure).
#include "jefi_internal.h"

namespace jefi {
namespace {

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
double run(int sm_count)
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

}  // namespace

double measure_alu_peak(jefi_dtype dt, int sm_count, int)
{
    return dt == JEFI_F32 ? run<float>(sm_count) : run<double>(sm_count);
}

}  // namespace jefi
