// jefi_api.cu -- the C ABI of include/jefi.h: context, validation, error reporting, launches.
// No arithmetic of the method lives here; every step of the path is a kernel in prepass.cu,
// pairwise_tiled.cu and pairwise_point.cu.  There is no CPU fallback.
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <new>
#include "jefi_internal.h"
#include "jefi_instrument.h"

namespace {

void set_err(jefi_ctx* c, const char* what, cudaError_t e)
{
    if (!c) return;
    if (e != cudaSuccess) snprintf(c->err, sizeof(c->err), "%s: %s", what, cudaGetErrorString(e));
    else snprintf(c->err, sizeof(c->err), "%s", what);
}

jefi_status cuda_fail(jefi_ctx* c, const char* what, cudaError_t e)
{
    set_err(c, what, e);
    cudaGetLastError();            // clear the sticky-less error state
    return e == cudaErrorMemoryAllocation ? JEFI_ERR_OOM : JEFI_ERR_CUDA;
}

bool grid_ok(const jefi_grid_desc& g)
{
    for (int a = 0; a < 3; ++a) {
        if (g.n[a] <= 0) return false;
        if (!(g.spacing[a] > 0.0) || !isfinite(g.spacing[a]) || !isfinite(g.origin[a])) return false;
    }
    return true;
}

jefi_status dev_alloc(jefi_ctx* c, void** p, size_t bytes, const char* what)
{
    if (bytes == 0) bytes = 16;
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) { *p = nullptr; return cuda_fail(c, what, e); }
    c->dev_bytes += (long long)bytes;
    return JEFI_OK;
}

void free_all(jefi_ctx* c)
{
    cudaFree(c->hist); cudaFree(c->scratch); cudaFree(c->stage_E); cudaFree(c->stage_B);
    cudaFree(c->tiles.perm); cudaFree(c->tiles.boxes);
    cudaFree(c->series); cudaFree(c->stage_series); cudaFree(c->raw_rho); cudaFree(c->raw_J); cudaFree(c->last); cudaFree(c->new_stage);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->ev_copied) cudaEventDestroy(c->ev_copied);
    if (c->ev_raw_free) cudaEventDestroy(c->ev_raw_free);
}

jefi_status check_fields_args(jefi_ctx* ctx, int32_t step, int64_t obs_begin, int64_t obs_count,
                              const void* E, const void* B)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    ctx->err[0] = 0;
    if (obs_begin < 0 || obs_count < 0 || obs_begin > ctx->P.n_obs || obs_count > ctx->P.n_obs - obs_begin) {
        set_err(ctx, "observation range outside the observation set", cudaSuccess);
        return JEFI_ERR_INVALID_ARG;
    }
    if (obs_count > 0 && (!E || !B)) {
        set_err(ctx, "null output pointer", cudaSuccess);
        return JEFI_ERR_INVALID_ARG;
    }
    if (step < 0 || step >= ctx->P.T) {
        set_err(ctx, "step outside the stored history", cudaSuccess);
        return JEFI_ERR_TIME_RANGE;
    }
    if (!ctx->has_history) {
        set_err(ctx, "jefi_fields before jefi_upload_history", cudaSuccess);
        return JEFI_ERR_NO_HISTORY;
    }
    return JEFI_OK;
}

jefi_status run_fields(jefi_ctx* ctx, int32_t step, int64_t obs_begin, int64_t obs_count,
                       void* E, void* B, cudaStream_t stream)
{
    if (obs_count == 0) return JEFI_OK;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return cuda_fail(ctx, "cudaSetDevice", e);
    jefi::FieldsLaunch L;
    L.step = step; L.obs_begin = obs_begin; L.obs_count = obs_count;
    L.E_out = E; L.B_out = B;
    L.scratch = ctx->scratch; L.scratch_elems = ctx->scratch_elems; L.chunk_bytes = ctx->chunk_bytes;
    L.sm_count = ctx->sm_count; L.stream = stream;
    int n = 0;
    if (ctx->kernel_choice != 1) {
        n = jefi::launch_fields_tiled(ctx->P, ctx->dtype, ctx->hist, L);
        if (n == 0) n = jefi::launch_fields_list(ctx->P, ctx->dtype, ctx->hist, L, ctx->tiles);
        if (n == 0 && ctx->kernel_choice == 2) {
            set_err(ctx, "tiled kernel does not support this request", cudaSuccess);
            return JEFI_ERR_UNSUPPORTED;
        }
    }
    if (n == 0) n = jefi::launch_fields_point(ctx->P, ctx->dtype, ctx->hist, L);
    if (n < 0) return cuda_fail(ctx, "fields kernel launch", cudaGetLastError());
    ctx->launches += n;
    return JEFI_OK;
}

// The partial sums of a series are [chunks][steps][6][points]: when the scratch sized by
// jefi_create for one-step calls cannot hold the whole series twice over, it is regrown (up to
// 1 GiB) so that the series goes in one batch of step blocks instead of several.  Blocks the
// device when it grows; never shrinks; keeps the old scratch if there is no room.
void grow_series_scratch(jefi_ctx* ctx, long long step_count, long long obs_count)
{
    const int nsb = jefi::series_block_steps(ctx->dtype);
    long long want = 2LL * 6 * obs_count * ((step_count + nsb - 1) / nsb * nsb);
    if (want > (1LL << 27)) want = 1LL << 27;
    if (want <= ctx->scratch_alloc_elems || ctx->scratch_elems != ctx->scratch_alloc_elems) return;
    void* bigger = nullptr;
    if (cudaMalloc(&bigger, (size_t)want * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return; }
    cudaDeviceSynchronize();                   // earlier launches may still use the old one
    cudaFree(ctx->scratch);
    ctx->dev_bytes += (want - ctx->scratch_alloc_elems) * (long long)sizeof(double);
    ctx->scratch = bigger;
    ctx->scratch_elems = ctx->scratch_alloc_elems = want;
}

// device staging of jefi_fields_series_host (E then B); growing frees the old one, so it waits
// for the copies still reading it
jefi_status grow_series_staging(jefi_ctx* ctx, size_t bytes)
{
    if (ctx->stage_series_bytes >= bytes) return JEFI_OK;
    if (ctx->stage_series) { cudaDeviceSynchronize(); cudaFree(ctx->stage_series); ctx->dev_bytes -= (long long)ctx->stage_series_bytes; }
    ctx->stage_series = nullptr; ctx->stage_series_bytes = 0;
    jefi_status s = dev_alloc(ctx, &ctx->stage_series, bytes, "cudaMalloc(series staging)");
    if (s == JEFI_OK) ctx->stage_series_bytes = bytes;
    return s;
}

jefi_status alloc_series_layout(jefi_ctx* ctx)
{
    if (ctx->series) return JEFI_OK;
    const size_t bytes = (size_t)ctx->P.Ns * (size_t)(ctx->P.T + 3) * 4 * ctx->elem;
    ctx->series_valid = false;
    return dev_alloc(ctx, &ctx->series, bytes, "cudaMalloc(series layout)");
}

}  // namespace

extern "C" {

jefi_status jefi_reserve_series(jefi_ctx* ctx, int32_t max_steps, int64_t max_obs, int32_t host_staging)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    ctx->err[0] = 0;
    if (max_steps <= 0 || max_steps > ctx->P.T || max_obs <= 0 || max_obs > ctx->P.n_obs) {
        set_err(ctx, "jefi_reserve_series: max_steps must be in [1, nsteps], max_obs in [1, N_o]", cudaSuccess);
        return JEFI_ERR_INVALID_ARG;
    }
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return cuda_fail(ctx, "cudaSetDevice", e);
    jefi_status s = alloc_series_layout(ctx);
    if (s != JEFI_OK) return s;
    grow_series_scratch(ctx, max_steps, max_obs);
    if (host_staging) {
        s = grow_series_staging(ctx, 2 * (size_t)max_steps * 3 * (size_t)max_obs * ctx->elem);
        if (s != JEFI_OK) return s;
    }
    return JEFI_OK;
}

jefi_status jefi_create(const jefi_grid_desc* src, const jefi_obs_desc* obs,
                        const jefi_time_desc* time, jefi_dtype dtype, int device, jefi_ctx** out)
{
    if (!src || !obs || !time || !out) return JEFI_ERR_INVALID_ARG;
    if (dtype != JEFI_F32 && dtype != JEFI_F64) return JEFI_ERR_INVALID_ARG;
    if (!grid_ok(*src)) return JEFI_ERR_INVALID_ARG;
    if (obs->kind != 0 && obs->kind != 1) return JEFI_ERR_INVALID_ARG;
    if (obs->kind == 0 && !grid_ok(obs->grid)) return JEFI_ERR_INVALID_ARG;
    if (obs->kind == 1 && (obs->npoints < 0 || (obs->npoints > 0 && !obs->points_dev)))
        return JEFI_ERR_INVALID_ARG;
    if (!(time->dt > 0.0) || !(time->c > 0.0) || !isfinite(time->dt) || !isfinite(time->c) ||
        !isfinite(time->t0) || time->nsteps <= 0)
        return JEFI_ERR_INVALID_ARG;
    if (time->deriv_mode != 0 && time->deriv_mode != 1) return JEFI_ERR_INVALID_ARG;
    if (time->past_mode != 0) return JEFI_ERR_UNSUPPORTED;
    if (device < 0) return JEFI_ERR_INVALID_ARG;

    jefi_ctx* c = new (std::nothrow) jefi_ctx;
    if (!c) return JEFI_ERR_OOM;
    memset(c, 0, sizeof(*c));
    jefi::Params& P = c->P;
    P.Ns = 1; P.n_obs = 1;
    for (int a = 0; a < 3; ++a) {
        P.ns[a] = src->n[a]; P.so[a] = src->origin[a]; P.sh[a] = src->spacing[a];
        P.Ns *= src->n[a];
        if (obs->kind == 0) {
            P.no[a] = obs->grid.n[a]; P.oo[a] = obs->grid.origin[a]; P.oh[a] = obs->grid.spacing[a];
            P.n_obs *= obs->grid.n[a];
        } else {
            P.no[a] = 1; P.oo[a] = 0; P.oh[a] = 1;
        }
    }
    if (obs->kind == 1) { P.n_obs = obs->npoints; P.no[0] = (int)(obs->npoints > 0x7fffffff ? 0x7fffffff : obs->npoints); }
    P.obs_kind = obs->kind; P.obs_points = obs->points_dev;
    P.T = time->nsteps; P.Tp = time->nsteps + 1;
    P.dt = time->dt; P.c = time->c; P.deriv_mode = time->deriv_mode;
    c->dtype = dtype; c->device = device; c->t0 = time->t0;
    c->elem = dtype == JEFI_F32 ? sizeof(float) : sizeof(double);
    if (P.Ns > (1LL << 31) - 64 || P.n_obs >= (1LL << 40)) { delete c; return JEFI_ERR_UNSUPPORTED; }

    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) { cudaGetLastError(); delete c; return JEFI_ERR_CUDA; }
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) { cudaGetLastError(); delete c; return JEFI_ERR_CUDA; }
    c->sm_count = prop.multiProcessorCount;

    // scratch: partial sums [S chunks][6 components][points] in double.  Room for 64 chunks of the
    // whole observation set (capped at 1 GiB, never below one chunk), so that the launchers can
    // pick a chunk count that fills the last wave of CTAs; more chunks than fit go to further,
    // accumulating launches.
    long long pts = P.n_obs < 8192 ? 8192 : P.n_obs;
    long long elems = 6 * 64 * pts;
    if (elems > (1LL << 27)) elems = (1LL << 27);
    if (elems < 6 * P.n_obs) elems = 6 * P.n_obs;
    c->scratch_elems = c->scratch_alloc_elems = elems;
    c->chunk_bytes = 384LL * 1024 * 1024;

    c->hist_bytes = (size_t)P.Ns * 2 * (size_t)P.Tp * 4 * c->elem;
    jefi_status s;
    if ((s = dev_alloc(c, &c->hist, c->hist_bytes, "cudaMalloc(packed history)")) != JEFI_OK ||
        (s = dev_alloc(c, &c->scratch, (size_t)c->scratch_elems * sizeof(double), "cudaMalloc(scratch)")) != JEFI_OK ||
        (s = dev_alloc(c, &c->last, (size_t)P.Ns * 8 * c->elem, "cudaMalloc(newest raw steps)")) != JEFI_OK ||
        (s = dev_alloc(c, &c->stage_E, (size_t)P.n_obs * 3 * c->elem, "cudaMalloc(E staging)")) != JEFI_OK ||
        (s = dev_alloc(c, &c->stage_B, (size_t)P.n_obs * 3 * c->elem, "cudaMalloc(B staging)")) != JEFI_OK) {
        free_all(c); delete c; return s;
    }
    if (obs->kind == 1 && P.n_obs > 0 && P.n_obs < (1LL << 31)) {
        // explicit points: sort them into spatially compact tiles for the tiled kernel (pairwise_list.cu)
        jefi::PointTiles& t = c->tiles;
        t.tile_points = jefi::list_tile_points(dtype);
        t.ntiles = (P.n_obs + t.tile_points - 1) / t.tile_points;
        if ((s = dev_alloc(c, (void**)&t.perm, (size_t)P.n_obs * sizeof(int), "cudaMalloc(point permutation)")) != JEFI_OK ||
            (s = dev_alloc(c, (void**)&t.boxes, (size_t)t.ntiles * 6 * sizeof(double), "cudaMalloc(tile boxes)")) != JEFI_OK) {
            free_all(c); delete c; return s;
        }
        const int n = jefi::build_point_tiles(P, dtype, t);
        if (n < 0) {
            cudaGetLastError();
            free_all(c); delete c;
            return n == -2 ? JEFI_ERR_INVALID_ARG : JEFI_ERR_CUDA;
        }
        c->launches += n;
    }
    *out = c;
    return JEFI_OK;
}

jefi_status jefi_upload_history(jefi_ctx* ctx, const void* rho_dev, const void* J_dev,
                                jefi_stream stream)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    ctx->err[0] = 0;
    if (!rho_dev || !J_dev) { set_err(ctx, "null history pointer", cudaSuccess); return JEFI_ERR_INVALID_ARG; }
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return cuda_fail(ctx, "cudaSetDevice", e);
    ctx->P.origin = 0;                     // the pre-pass writes packed step p at slot p
    int n = jefi::launch_prepass(ctx->P, ctx->dtype, rho_dev, J_dev, ctx->hist, (cudaStream_t)stream);
    if (n < 0) return cuda_fail(ctx, "pre-pass launch", cudaGetLastError());
    ctx->launches += n;
    // keep the raw values of the two newest steps for jefi_append_step (copies, no arithmetic)
    {
        const size_t plane = (size_t)ctx->P.Ns * ctx->elem;
        const int T = ctx->P.T;
        char* last = (char*)ctx->last;
        const char* r = (const char*)rho_dev;
        const char* Jp = (const char*)J_dev;
        cudaStream_t st = (cudaStream_t)stream;
        for (int s = 0; s < 2 && e == cudaSuccess; ++s) {
            const int m = T - 2 + s;
            if (m < 0) { e = cudaMemsetAsync(last + (size_t)s * 4 * plane, 0, 4 * plane, st); continue; }
            e = cudaMemcpyAsync(last + (size_t)s * 4 * plane, r + (size_t)m * plane, plane,
                                cudaMemcpyDeviceToDevice, st);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(last + ((size_t)s * 4 + 1) * plane, Jp + (size_t)m * 3 * plane, 3 * plane,
                                    cudaMemcpyDeviceToDevice, st);
        }
        if (e != cudaSuccess) return cuda_fail(ctx, "copy of the newest raw steps", e);
    }
    ctx->has_history = true;
    ctx->series_valid = false;
    return JEFI_OK;
}

jefi_status jefi_append_step(jefi_ctx* ctx, const void* rho_new_dev, const void* J_new_dev, jefi_stream stream)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    ctx->err[0] = 0;
    if (!rho_new_dev || !J_new_dev) { set_err(ctx, "null step pointer", cudaSuccess); return JEFI_ERR_INVALID_ARG; }
    if (!ctx->has_history) {
        set_err(ctx, "jefi_append_step before jefi_upload_history", cudaSuccess);
        return JEFI_ERR_NO_HISTORY;
    }
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return cuda_fail(ctx, "cudaSetDevice", e);
    int n = jefi::launch_append(ctx->P, ctx->dtype, rho_new_dev, J_new_dev, ctx->last, ctx->hist,
                                (cudaStream_t)stream);
    if (n < 0) return cuda_fail(ctx, "append launch", cudaGetLastError());
    ctx->launches += n;
    ctx->P.origin = (ctx->P.origin + 1) % ctx->P.T;      // the ring advances: packed step p now sits one slot on
    ctx->series_valid = false;
    ctx->t0 += ctx->P.dt;
    return JEFI_OK;
}

jefi_status jefi_append_step_host(jefi_ctx* ctx, const void* rho_new_host, const void* J_new_host,
                                  jefi_stream stream)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    ctx->err[0] = 0;
    if (!rho_new_host || !J_new_host) { set_err(ctx, "null step pointer", cudaSuccess); return JEFI_ERR_INVALID_ARG; }
    if (!ctx->has_history) {
        set_err(ctx, "jefi_append_step before jefi_upload_history", cudaSuccess);
        return JEFI_ERR_NO_HISTORY;
    }
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return cuda_fail(ctx, "cudaSetDevice", e);
    const size_t plane = (size_t)ctx->P.Ns * ctx->elem;
    if (!ctx->new_stage) {
        jefi_status s = dev_alloc(ctx, &ctx->new_stage, 4 * plane, "cudaMalloc(new step staging)");
        if (s != JEFI_OK) return s;
    }
    cudaStream_t st = (cudaStream_t)stream;
    char* stage = (char*)ctx->new_stage;
    if ((e = cudaMemcpyAsync(stage, rho_new_host, plane, cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(stage + plane, J_new_host, 3 * plane, cudaMemcpyHostToDevice, st)) != cudaSuccess)
        return cuda_fail(ctx, "cudaMemcpyAsync(new step)", e);
    return jefi_append_step(ctx, stage, stage + plane, stream);
}

jefi_status jefi_upload_history_host(jefi_ctx* ctx, const void* rho_host, const void* J_host,
                                     jefi_stream stream)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    ctx->err[0] = 0;
    if (!rho_host || !J_host) { set_err(ctx, "null history pointer", cudaSuccess); return JEFI_ERR_INVALID_ARG; }
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return cuda_fail(ctx, "cudaSetDevice", e);
    const size_t rho_bytes = (size_t)ctx->P.T * (size_t)ctx->P.Ns * ctx->elem;
    // (each staging buffer is guarded on its own: a failed second allocation is retried by the
    // next call instead of leaving a null raw_J behind a non-null raw_rho)
    {
        jefi_status s;
        if (!ctx->raw_rho && (s = dev_alloc(ctx, &ctx->raw_rho, rho_bytes, "cudaMalloc(raw rho)")) != JEFI_OK) return s;
        if (!ctx->raw_J && (s = dev_alloc(ctx, &ctx->raw_J, 3 * rho_bytes, "cudaMalloc(raw J)")) != JEFI_OK) return s;
    }
    // The copy goes on the context's own stream so that, in a stepping loop, the H2D of the next
    // history overlaps the pairwise kernel of the current step still running on `stream`:
    //   copy_stream: wait(raw staging free) -> H2D rho, J -> record(copied)
    //   stream:      wait(copied) -> pre-pass -> record(raw staging free)
    if (!ctx->copy_stream) {
        if ((e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking)) != cudaSuccess ||
            (e = cudaEventCreateWithFlags(&ctx->ev_copied, cudaEventDisableTiming)) != cudaSuccess ||
            (e = cudaEventCreateWithFlags(&ctx->ev_raw_free, cudaEventDisableTiming)) != cudaSuccess)
            return cuda_fail(ctx, "copy stream/event creation", e);
    }
    cudaStream_t st = (cudaStream_t)stream, cs = ctx->copy_stream;
    if (ctx->raw_in_use && (e = cudaStreamWaitEvent(cs, ctx->ev_raw_free, 0)) != cudaSuccess)
        return cuda_fail(ctx, "cudaStreamWaitEvent(raw free)", e);
    if ((e = cudaMemcpyAsync(ctx->raw_rho, rho_host, rho_bytes, cudaMemcpyHostToDevice, cs)) != cudaSuccess)
        return cuda_fail(ctx, "cudaMemcpyAsync(rho)", e);
    if ((e = cudaMemcpyAsync(ctx->raw_J, J_host, 3 * rho_bytes, cudaMemcpyHostToDevice, cs)) != cudaSuccess)
        return cuda_fail(ctx, "cudaMemcpyAsync(J)", e);
    if ((e = cudaEventRecord(ctx->ev_copied, cs)) != cudaSuccess ||
        (e = cudaStreamWaitEvent(st, ctx->ev_copied, 0)) != cudaSuccess)
        return cuda_fail(ctx, "cudaEventRecord/WaitEvent(copied)", e);
    jefi_status s = jefi_upload_history(ctx, ctx->raw_rho, ctx->raw_J, stream);
    if (s != JEFI_OK) return s;
    if ((e = cudaEventRecord(ctx->ev_raw_free, st)) != cudaSuccess)
        return cuda_fail(ctx, "cudaEventRecord(raw free)", e);
    ctx->raw_in_use = true;
    return JEFI_OK;
}

jefi_status jefi_fields(jefi_ctx* ctx, int32_t step, int64_t obs_begin, int64_t obs_count,
                        void* E_out_dev, void* B_out_dev, jefi_stream stream)
{
    jefi_status s = check_fields_args(ctx, step, obs_begin, obs_count, E_out_dev, B_out_dev);
    if (s != JEFI_OK) return s;
    return run_fields(ctx, step, obs_begin, obs_count, E_out_dev, B_out_dev, (cudaStream_t)stream);
}

jefi_status jefi_fields_series(jefi_ctx* ctx, int32_t step_begin, int32_t step_count,
                               int64_t obs_begin, int64_t obs_count,
                               void* E_out_dev, void* B_out_dev, jefi_stream stream)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    if (step_count < 0) { set_err(ctx, "negative step count", cudaSuccess); return JEFI_ERR_INVALID_ARG; }
    if (step_count == 0) return JEFI_OK;
    // every argument is checked before the first launch
    jefi_status s = check_fields_args(ctx, step_begin, obs_begin, obs_count, E_out_dev, B_out_dev);
    if (s != JEFI_OK) return s;
    if (step_count > ctx->P.T - step_begin) {          // (overflow-safe form of begin + count - 1 < T)
        set_err(ctx, "step outside the stored history", cudaSuccess);
        return JEFI_ERR_TIME_RANGE;
    }
    if (obs_count == 0) return JEFI_OK;
    // Regular observation grids and enough steps to fill a block: the time-blocked kernel
    // (pairwise_series.cu), which evaluates NS consecutive steps per (point, cell) pair.
    if ((ctx->kernel_choice == 0 || ctx->kernel_choice == 3) && ctx->P.obs_kind == 0 && 2 * step_count >= jefi::series_block_steps(ctx->dtype)) {
        cudaError_t e = cudaSetDevice(ctx->device);
        if (e != cudaSuccess) return cuda_fail(ctx, "cudaSetDevice", e);
        if ((s = alloc_series_layout(ctx)) != JEFI_OK) return s;
        if (!ctx->series_valid) {
            int n = jefi::launch_series_layout(ctx->P, ctx->dtype, ctx->hist, ctx->series, (cudaStream_t)stream);
            if (n < 0) return cuda_fail(ctx, "series layout launch", cudaGetLastError());
            ctx->launches += n;
            ctx->series_valid = true;
        }
        // The partial sums of a series are [chunks][steps][6][points]: when the scratch sized by
        // jefi_create for one-step calls cannot hold the whole series twice over, it is regrown
        // once (up to 1 GiB) so that the series goes in one batch of step blocks instead of several
        // (X1: 411 steps x 3375 points in 3 batches of ~2 waves -> 1 batch of 5 waves).
        grow_series_scratch(ctx, step_count, obs_count);
        jefi::FieldsLaunch L;
        L.step = step_begin; L.obs_begin = obs_begin; L.obs_count = obs_count;
        L.E_out = E_out_dev; L.B_out = B_out_dev;
        L.scratch = ctx->scratch; L.scratch_elems = ctx->scratch_elems; L.chunk_bytes = ctx->chunk_bytes;
        L.sm_count = ctx->sm_count; L.stream = (cudaStream_t)stream;
        int n = jefi::launch_fields_series(ctx->P, ctx->dtype, ctx->series, L, step_begin, step_count);
        if (n < 0) return cuda_fail(ctx, "series kernel launch", cudaGetLastError());
        if (n > 0) { ctx->launches += n; return JEFI_OK; }
        if (ctx->kernel_choice == 3) {
            set_err(ctx, "time-blocked kernel does not support this request", cudaSuccess);
            return JEFI_ERR_UNSUPPORTED;
        }
    }
    const size_t stride = (size_t)obs_count * 3 * ctx->elem;
    for (int32_t k = 0; k < step_count; ++k) {
        s = run_fields(ctx, step_begin + k, obs_begin, obs_count, (char*)E_out_dev + (size_t)k * stride,
                       (char*)B_out_dev + (size_t)k * stride, (cudaStream_t)stream);
        if (s != JEFI_OK) return s;
    }
    return JEFI_OK;
}

jefi_status jefi_fields_at_time(jefi_ctx* ctx, double t, int64_t obs_begin, int64_t obs_count,
                                void* E_out_dev, void* B_out_dev, jefi_stream stream)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    ctx->err[0] = 0;
    const double x = (t - ctx->t0) / ctx->P.dt;
    const double n = floor(x + 0.5);
    if (!isfinite(x) || fabs(x - n) > 1e-6 || n < 0.0 || n > (double)(ctx->P.T - 1)) {
        set_err(ctx, "t is not on the stored step grid", cudaSuccess);
        return JEFI_ERR_TIME_RANGE;
    }
    return jefi_fields(ctx, (int32_t)n, obs_begin, obs_count, E_out_dev, B_out_dev, stream);
}

jefi_status jefi_fields_host(jefi_ctx* ctx, int32_t step, int64_t obs_begin, int64_t obs_count,
                             void* E_out_host, void* B_out_host, jefi_stream stream)
{
    jefi_status s = check_fields_args(ctx, step, obs_begin, obs_count, E_out_host, B_out_host);
    if (s != JEFI_OK) return s;
    if (obs_count == 0) return JEFI_OK;
    cudaStream_t st = (cudaStream_t)stream;
    s = run_fields(ctx, step, obs_begin, obs_count, ctx->stage_E, ctx->stage_B, st);
    if (s != JEFI_OK) return s;
    const size_t bytes = (size_t)obs_count * 3 * ctx->elem;
    cudaError_t e;
    if ((e = cudaMemcpyAsync(E_out_host, ctx->stage_E, bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return cuda_fail(ctx, "cudaMemcpyAsync(E)", e);
    if ((e = cudaMemcpyAsync(B_out_host, ctx->stage_B, bytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return cuda_fail(ctx, "cudaMemcpyAsync(B)", e);
    return JEFI_OK;
}

jefi_status jefi_fields_series_host(jefi_ctx* ctx, int32_t step_begin, int32_t step_count, int64_t obs_begin,
                                    int64_t obs_count, void* E_out_host, void* B_out_host, jefi_stream stream)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    if (step_count < 0) { set_err(ctx, "negative step count", cudaSuccess); return JEFI_ERR_INVALID_ARG; }
    if (step_count == 0) return JEFI_OK;
    jefi_status s = check_fields_args(ctx, step_begin, obs_begin, obs_count, E_out_host, B_out_host);
    if (s != JEFI_OK) return s;
    if (step_count > ctx->P.T - step_begin) {          // before anything is sized from step_count
        set_err(ctx, "step outside the stored history", cudaSuccess);
        return JEFI_ERR_TIME_RANGE;
    }
    if (obs_count == 0) return JEFI_OK;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return cuda_fail(ctx, "cudaSetDevice", e);
    const size_t half = (size_t)step_count * 3 * (size_t)obs_count * ctx->elem;
    if ((s = grow_series_staging(ctx, 2 * half)) != JEFI_OK) return s;
    char* Ed = (char*)ctx->stage_series;
    char* Bd = Ed + half;
    s = jefi_fields_series(ctx, step_begin, step_count, obs_begin, obs_count, Ed, Bd, stream);
    if (s != JEFI_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    if ((e = cudaMemcpyAsync(E_out_host, Ed, half, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return cuda_fail(ctx, "cudaMemcpyAsync(E series)", e);
    if ((e = cudaMemcpyAsync(B_out_host, Bd, half, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return cuda_fail(ctx, "cudaMemcpyAsync(B series)", e);
    return JEFI_OK;
}

jefi_status jefi_set_kernel(jefi_ctx* ctx, int32_t which)
{
    if (!ctx || which < 0 || which > 3) return JEFI_ERR_INVALID_ARG;
    ctx->kernel_choice = which;
    return JEFI_OK;
}

int64_t jefi_device_bytes(const jefi_ctx* ctx) { return ctx ? ctx->dev_bytes : 0; }

jefi_status jefi_destroy(jefi_ctx* ctx)
{
    if (!ctx) return JEFI_ERR_INVALID_ARG;
    jefi_status s = JEFI_OK;
    if (cudaSetDevice(ctx->device) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) {
        cudaGetLastError();
        s = JEFI_ERR_CUDA;
    }
    free_all(ctx);
    delete ctx;
    return s;
}

const char* jefi_status_string(jefi_status s)
{
    switch (s) {
        case JEFI_OK: return "JEFI_OK";
        case JEFI_ERR_INVALID_ARG: return "JEFI_ERR_INVALID_ARG";
        case JEFI_ERR_CUDA: return "JEFI_ERR_CUDA";
        case JEFI_ERR_OOM: return "JEFI_ERR_OOM";
        case JEFI_ERR_NO_HISTORY: return "JEFI_ERR_NO_HISTORY";
        case JEFI_ERR_TIME_RANGE: return "JEFI_ERR_TIME_RANGE";
        case JEFI_ERR_UNSUPPORTED: return "JEFI_ERR_UNSUPPORTED";
    }
    return "JEFI_ERR_?";
}

const char* jefi_last_error(const jefi_ctx* ctx) { return ctx ? ctx->err : ""; }

int jefi_flops_per_pair(void) { return 52; }

jefi_status jefi_shard_obs(const jefi_obs_desc* obs, int32_t rank, int32_t world,
                           int64_t* begin, int64_t* count)
{
    if (!obs || !begin || !count || world <= 0 || rank < 0 || rank >= world) return JEFI_ERR_INVALID_ARG;
    if (obs->kind != 0 && obs->kind != 1) return JEFI_ERR_INVALID_ARG;
    int64_t total, granule = 1;
    if (obs->kind == 0) {
        if (!grid_ok(obs->grid)) return JEFI_ERR_INVALID_ARG;
        const int64_t nx = obs->grid.n[0], ny = obs->grid.n[1], nz = obs->grid.n[2];
        total = nx * ny * nz;
        if (nz >= world) granule = nx * ny;
        else if (ny * nz >= world) granule = nx;
    } else {
        if (obs->npoints < 0) return JEFI_ERR_INVALID_ARG;
        total = obs->npoints;
    }
    const int64_t units = total / granule, base = units / world, rem = units % world;
    *begin = (rank * base + (rank < rem ? rank : rem)) * granule;
    *count = (base + (rank < rem ? 1 : 0)) * granule;
    return JEFI_OK;
}

jefi_status jefi_shard_src(const jefi_grid_desc* src, int32_t rank, int32_t world, jefi_grid_desc* slab,
                           int64_t* cell_begin)
{
    if (!src || !slab || !cell_begin || world <= 0 || rank < 0 || rank >= world) return JEFI_ERR_INVALID_ARG;
    if (!grid_ok(*src)) return JEFI_ERR_INVALID_ARG;
    const int64_t nz = src->n[2], base = nz / world, rem = nz % world;
    const int64_t z0 = rank * base + (rank < rem ? rank : rem), nl = base + (rank < rem ? 1 : 0);
    *slab = *src;
    slab->n[2] = (int32_t)nl;
    slab->origin[2] = src->origin[2] + (double)z0 * src->spacing[2];
    *cell_begin = z0 * (int64_t)src->n[0] * (int64_t)src->n[1];
    return JEFI_OK;
}

}  // extern "C"
