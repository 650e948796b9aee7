/*
 * jefi_instrument.h -- measurement and test instrumentation of libjefi.so.
 *
 * NOT part of the product ABI (that is include/jefi.h): nothing here is needed to compute
 * fields.  bench.py uses the launch counter and the ALU-peak chain for its report; the -m gpu
 * tests use the lag dump for the parity report SURVEY.md 8(d) asks for (retarded-index
 * mismatches between the kernels and the fp64 oracle).  All of it lives in one translation
 * unit, csrc/instrument.cu.
 */
#ifndef JEFI_INSTRUMENT_H
#define JEFI_INSTRUMENT_H

#include "jefi.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Number of kernels launched by this context so far (bench.py: "gpu_launches"). */
int64_t     jefi_launch_count(const jefi_ctx* ctx);

/* Register-only FFMA (dtype F32) or DFMA (dtype F64) chain on `device`: the measured TFLOP/s
 * in *tflops (synchronous).  bench.py prints it beside the nominal ALU peak it divides by
 * (MEASURED_PEAKS.json carries no FP32/FP64 figure). */
jefi_status jefi_measure_alu_peak(int device, jefi_dtype dtype, double* tflops);

/* FP32 FFMA throughput by operand source on `device` (TFLOP/s, synchronous): accumulate
 * instructions acc += v * w that read two fresh registers and one the operand-reuse cache serves,
 * and ones that read three fresh registers.  jefi_measure_alu_peak's chain takes its other two
 * operands from the constant bank.  bench.py prints all three beside the series workloads: the
 * register file, not the FMA pipe, bounds the time-blocked kernel. */
jefi_status jefi_measure_ffma_operand_rates(int device, double* two_fresh_tflops, double* three_fresh_tflops);

/* Retarded lag k (Eq. (6): the stored step is m = step - k) that kernel `which`
 * computes for n_pairs explicit (observation point, source cell) pairs:
 * obs_index_dev[i] = linear index into the observation set, cell_index_dev[i] = linear source
 * cell index (both int64, device), lag_out_dev[i] = k (int32, device).  which = 1: the
 * per-point kernel's arithmetic (floor(R/(c dt) + 1/2) in the context dtype); which = 2: the
 * tiled kernels' (rsqrt.approx + magic-constant FMA, the same inlined device function
 * pair_geo() that the pairwise kernels call, so the dump IS their decision).  The history is
 * not read; no upload is needed.  which = 2 needs a regular observation grid
 * (JEFI_ERR_UNSUPPORTED otherwise).  One kernel on `stream`. */
jefi_status jefi_debug_pair_lags(jefi_ctx* ctx, int32_t which, int64_t n_pairs,
                                 const int64_t* obs_index_dev, const int64_t* cell_index_dev,
                                 int32_t* lag_out_dev, jefi_stream stream);

/* Test hook for the launchers' multi-launch path: caps the partial-sum scratch the launchers may
 * use at `scratch_elems` doubles (clamped to [6 * N_o, the allocated size]; <= 0: leave) and the
 * packed-history bytes one source chunk may span at `chunk_bytes` (default 384 MB; <= 0: leave),
 * so that a small problem needs more source chunks than one launch holds and goes through the
 * accumulating launches that otherwise only very large histories reach
 * (> 384 MB x scratch / (48 B x N_o), e.g. the paper's 160^3 x 500-step case). */
jefi_status jefi_debug_launch_limits(jefi_ctx* ctx, int64_t scratch_elems, int64_t chunk_bytes);

#ifdef __cplusplus
}
#endif
#endif /* JEFI_INSTRUMENT_H */
