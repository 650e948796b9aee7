// fields_noalloc.cu -- jefi_fields_noalloc (include/jefi.h): E and B of one evaluation step
// without a context and without a single device allocation.
//
// Who needs this.  Everything else in the library works on a jefi_ctx, and jefi_create
// cudaMallocs the packed history, the partial-sum scratch and the staging buffers.  Some hosts
// cannot do that: a field solver that runs as a plug-in of a simulation whose framework has
// already handed every free byte of HBM to its own memory pool (cudaMalloc then simply fails),
// or a time-stepping loop with a latency budget, where cudaMalloc/cudaFree are unwelcome because
// they synchronise the whole device.  Such a caller owns its buffers already -- the raw history
// rho, J and the output planes -- and passes them in; the only memory the method needs beyond
// them is the partial sums of the source chunks (step a6), and those live here in
// a fixed array inside the library image.
//
// What runs: a variant of the per-point kernel of pairwise_point.cu (one thread per observation
// point, the paper's own shape) that reads the RAW history and forms the time
// derivatives in the kernel from neighbouring snapshots, as the paper does,
// in the arithmetic of prepass.cu (same differences, same pre-scaling by 1/c), so no packed
// history is needed; then the fixed-order reduce + scale epilogue.  The geometry, the screening
// rule and the retarded lag come from the helpers of tiled_common.cuh every other kernel uses, so
// each (point, cell) pair takes the same decisions as in jefi_fields.
//
// The scratch array.  g_partial is 8 MiB of .bss-like device memory that EVERY device holds from
// the moment it loads libjefi.so until the process exits, whether or not this entry point is ever
// called -- hence the modest size, and hence the limit JEFI_NOALLOC_MAX_OBS per call.  In host
// code the name g_partial is only a handle for the runtime, not a device address: the address is
// asked for once per device with cudaGetSymbolAddress, with that device current, and that pointer
// is what the kernels get.  All calls on a device share the array and it keeps whatever the last
// call left in it.  Nothing in it has to start at zero: every element the epilogue reads
// ([S][6][obs_count]) is written by the pairwise kernel of the same call first.  Two calls whose
// kernels can overlap on one device (different streams, no dependency) race on it.
#include <math.h>
#include <stdio.h>
#include <mutex>
#include "tiled_common.cuh"

namespace {

constexpr long long kScratchElems = JEFI_NOALLOC_SCRATCH_BYTES / (long long)sizeof(double);
static_assert(6LL * JEFI_NOALLOC_MAX_OBS <= kScratchElems, "one chunk of the largest request must fit");

// partial sums [S][6][obs_count] of the call in flight
static __device__ __align__(256) double g_partial[kScratchElems];

struct RawArgs {
    int nsx, nsy, nsz;
    int nox, noy;
    double shx, shy, shz;       // source spacing
    double ohx, ohy, ohz;       // obs spacing
    double d0x, d0y, d0z;       // obs origin - source origin (host fp64)
    double sox, soy, soz;       // source origin (explicit point lists)
    double rcut2, inv_cdt, inv_dt, inv_c;
    long long Ns, obs_begin, obs_count;
    int T, step, deriv_mode;
    int obs_kind;
    const void* points;
    long long cells_per_chunk;
};

constexpr int kThreads = 128;

// f(m) and df/dt(m) of one raw field (a [T][stride] array, this cell) -- prepass.cu's rule:
// backward mode (f(m) - f(m-1))/dt with f(-1) = 0; centred mode (f(m+1) - f(m-1))/(2 dt) inside
// the history, one-sided at m = 0 and m = T-1, zero for a one-step history
template <typename T>
__device__ __forceinline__ void value_and_ddt(const T* __restrict__ f, long long stride, int m, int Tsteps,
                                              int deriv_mode, T inv_dt, T& fm, T& dd)
{
    fm = f[(long long)m * stride];
    const T fa = m > 0 ? f[(long long)(m - 1) * stride] : T(0);
    if (deriv_mode == 1)        { dd = (fm - fa) * inv_dt; return; }
    if (Tsteps == 1)            { dd = T(0); return; }
    if (m == Tsteps - 1)        { dd = (fm - fa) * inv_dt; return; }
    const T fb = f[(long long)(m + 1) * stride];
    dd = m == 0 ? (fb - fm) * inv_dt : (fb - fa) * (T(0.5) * inv_dt);
}

template <typename T>
__global__ void __launch_bounds__(kThreads)
fields_point_raw_kernel(const T* __restrict__ rho, const T* __restrict__ J, double* __restrict__ partial, RawArgs a)
{
    const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
    if (i >= a.obs_count) return;
    const long long gi = a.obs_begin + i;

    T ox, oy, oz;                                   // relative to the centre of source cell (0,0,0)
    if (a.obs_kind == 0) {
        const int ix = (int)(gi % a.nox), iy = (int)((gi / a.nox) % a.noy);
        const int iz = (int)(gi / ((long long)a.nox * a.noy));
        ox = jefi::obs_coord<T>(a.d0x, ix, a.ohx); oy = jefi::obs_coord<T>(a.d0y, iy, a.ohy);
        oz = jefi::obs_coord<T>(a.d0z, iz, a.ohz);
    } else {
        const T* p = (const T*)a.points + 3 * gi;
        ox = (T)((double)p[0] - a.sox); oy = (T)((double)p[1] - a.soy); oz = (T)((double)p[2] - a.soz);
    }
    const T shx = (T)a.shx, shy = (T)a.shy, shz = (T)a.shz;
    const T rcut2 = (T)a.rcut2, inv_cdt = -jefi::tie_biased_neg_inv_cdt<T>(a.inv_cdt);
    const T inv_dt = (T)a.inv_dt, ic = (T)a.inv_c, ic2 = ic * ic;

    const long long cb = (long long)blockIdx.y * a.cells_per_chunk;
    long long ce = cb + a.cells_per_chunk;
    if (ce > a.Ns) ce = a.Ns;
    int sx = (int)(cb % a.nsx), sy = (int)((cb / a.nsx) % a.nsy);
    int sz = (int)(cb / ((long long)a.nsx * a.nsy));

    double tot[6] = {0, 0, 0, 0, 0, 0};
    long long j = cb;
    while (j < ce) {
        T dy, dz;                                   // one (part of a) source row: y, z fixed
        const T ryz = jefi::row_ryz<T>(oy, oz, sy, sz, shy, shz, dy, dz);
        long long row_end = j + (a.nsx - sx);
        if (row_end > ce) row_end = ce;
        T ex = 0, ey = 0, ez = 0, bx = 0, by = 0, bz = 0;
        for (; j < row_end; ++j, ++sx) {
            T dx, rinv;
            int k;
            jefi::point_geo<T>(ox, sx, shx, ryz, rcut2, inv_cdt, dx, rinv, k);
            const int m = a.step - k;               // retarded stored step, Eq. (6)
            if (m < 0 || k < 0) continue;           // before the history (k < 0: lag beyond int range)
            T r, rd, jx, jxd, jy, jyd, jz, jzd;
            value_and_ddt<T>(rho + j, a.Ns, m, a.T, a.deriv_mode, inv_dt, r, rd);
            value_and_ddt<T>(J + j, 3 * a.Ns, m, a.T, a.deriv_mode, inv_dt, jx, jxd);
            value_and_ddt<T>(J + a.Ns + j, 3 * a.Ns, m, a.T, a.deriv_mode, inv_dt, jy, jyd);
            value_and_ddt<T>(J + 2 * a.Ns + j, 3 * a.Ns, m, a.T, a.deriv_mode, inv_dt, jz, jzd);
            rd *= ic; jx *= ic; jy *= ic; jz *= ic; jxd *= ic2; jyd *= ic2; jzd *= ic2;
            const T r2 = rinv * rinv;
            const T s  = (r * rinv + rd) * r2;
            const T ux = (jx * rinv + jxd) * r2;
            const T uy = (jy * rinv + jyd) * r2;
            const T uz = (jz * rinv + jzd) * r2;
            ex += dx * s - jxd * rinv;
            ey += dy * s - jyd * rinv;
            ez += dz * s - jzd * rinv;
            bx += uy * dz - uz * dy;
            by += uz * dx - ux * dz;
            bz += ux * dy - uy * dx;
        }
        tot[0] += (double)ex; tot[1] += (double)ey; tot[2] += (double)ez;
        tot[3] += (double)bx; tot[4] += (double)by; tot[5] += (double)bz;
        sx = 0;
        if (++sy == a.nsy) { sy = 0; ++sz; }
    }
    double* out = partial + (long long)blockIdx.y * 6 * a.obs_count + i;
#pragma unroll
    for (int c = 0; c < 6; ++c) out[(long long)c * a.obs_count] = tot[c];
}

// step a6: sum the S chunks in a fixed order, x dV/(4 pi) (and c for B), store component planes
template <typename T>
__global__ void __launch_bounds__(256)
reduce_scale_raw_kernel(const double* __restrict__ partial, T* __restrict__ E, T* __restrict__ B, long long count,
                        int S, double scaleE, double scaleB)
{
    const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
    if (t >= 6 * count) return;
    const int c = (int)(t / count);
    const long long i = t - (long long)c * count;
    const double* src = partial + (long long)c * count + i;
    double acc = 0.0;
    for (int s = 0; s < S; ++s) acc += src[(long long)s * 6 * count];
    if (c < 3) E[(long long)c * count + i] = (T)(acc * scaleE);
    else       B[(long long)(c - 3) * count + i] = (T)(acc * scaleB);
}

// per-device set-up, done by the first call on that device
struct DeviceSlot {
    bool    ready;
    double* scratch;            // device address of g_partial on this device
    int     sm_count;
};
constexpr int kMaxDevices = 64;
DeviceSlot g_slot[kMaxDevices];
std::mutex g_slot_mutex;

jefi_status fail(char* err, int32_t err_len, jefi_status s, const char* what, cudaError_t e = cudaSuccess)
{
    if (err && err_len > 0) {
        if (e != cudaSuccess) snprintf(err, (size_t)err_len, "%s: %s", what, cudaGetErrorString(e));
        else snprintf(err, (size_t)err_len, "%s", what);
    }
    if (e != cudaSuccess) cudaGetLastError();
    return s;
}

bool grid_ok(const jefi_grid_desc& g)
{
    for (int a = 0; a < 3; ++a)
        if (g.n[a] <= 0 || !(g.spacing[a] > 0.0) || !isfinite(g.spacing[a]) || !isfinite(g.origin[a])) return false;
    return true;
}

}  // namespace

extern "C" jefi_status jefi_fields_noalloc(const jefi_grid_desc* src, const jefi_obs_desc* obs,
                                           const jefi_time_desc* time, jefi_dtype dtype, int32_t step,
                                           const void* rho_dev, const void* J_dev, int64_t obs_begin,
                                           int64_t obs_count, void* E_out_dev, void* B_out_dev,
                                           jefi_stream stream, char* err, int32_t err_len)
{
    if (err && err_len > 0) err[0] = 0;
    // ---- arguments: everything is checked before the first CUDA call
    if (!src || !obs || !time) return fail(err, err_len, JEFI_ERR_INVALID_ARG, "null descriptor");
    if (dtype != JEFI_F32 && dtype != JEFI_F64) return fail(err, err_len, JEFI_ERR_INVALID_ARG, "bad dtype");
    if (!grid_ok(*src)) return fail(err, err_len, JEFI_ERR_INVALID_ARG, "bad source grid");
    if (obs->kind != 0 && obs->kind != 1) return fail(err, err_len, JEFI_ERR_INVALID_ARG, "bad observation kind");
    if (obs->kind == 0 && !grid_ok(obs->grid)) return fail(err, err_len, JEFI_ERR_INVALID_ARG, "bad observation grid");
    if (obs->kind == 1 && (obs->npoints < 0 || (obs->npoints > 0 && !obs->points_dev)))
        return fail(err, err_len, JEFI_ERR_INVALID_ARG, "point list without positions");
    if (!(time->dt > 0.0) || !(time->c > 0.0) || !isfinite(time->dt) || !isfinite(time->c) || time->nsteps <= 0)
        return fail(err, err_len, JEFI_ERR_INVALID_ARG, "bad time descriptor");
    if (time->deriv_mode != 0 && time->deriv_mode != 1) return fail(err, err_len, JEFI_ERR_INVALID_ARG, "bad deriv_mode");
    if (time->past_mode != 0) return fail(err, err_len, JEFI_ERR_UNSUPPORTED, "past_mode must be 0");

    const long long kIndexMax = 1LL << 40;
    long long Ns = 1, n_obs = 1;
    for (int a = 0; a < 3; ++a) {
        Ns *= src->n[a];
        if (Ns > kIndexMax) return fail(err, err_len, JEFI_ERR_INVALID_ARG, "source grid too large");
        if (obs->kind == 0) {
            n_obs *= obs->grid.n[a];
            if (n_obs > kIndexMax) return fail(err, err_len, JEFI_ERR_INVALID_ARG, "observation grid too large");
        }
    }
    if (obs->kind == 1) n_obs = obs->npoints;
    if (obs_begin < 0 || obs_count < 0 || obs_begin > n_obs || obs_count > n_obs - obs_begin)
        return fail(err, err_len, JEFI_ERR_INVALID_ARG, "observation range outside the observation set");
    if (step < 0 || step >= time->nsteps)
        return fail(err, err_len, JEFI_ERR_TIME_RANGE, "step outside the stored history");
    if (obs_count > JEFI_NOALLOC_MAX_OBS) {
        if (err && err_len > 0)
            snprintf(err, (size_t)err_len,
                     "obs_count %lld exceeds JEFI_NOALLOC_MAX_OBS = %d points per call (the partial sums must fit the "
                     "library's fixed %d-byte scratch array): split the request, or use a jefi_ctx",
                     (long long)obs_count, JEFI_NOALLOC_MAX_OBS, JEFI_NOALLOC_SCRATCH_BYTES);
        return JEFI_ERR_UNSUPPORTED;
    }
    if (obs_count == 0) return JEFI_OK;
    if (!rho_dev || !J_dev || !E_out_dev || !B_out_dev)
        return fail(err, err_len, JEFI_ERR_INVALID_ARG, "null device pointer");

    // ---- set-up, once per device: device address of the scratch array, SM count
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(err, err_len, JEFI_ERR_CUDA, "cudaGetDevice", e);
    if (dev < 0 || dev >= kMaxDevices) return fail(err, err_len, JEFI_ERR_UNSUPPORTED, "device ordinal beyond 63");
    DeviceSlot slot;
    {
        std::lock_guard<std::mutex> lock(g_slot_mutex);
        if (!g_slot[dev].ready) {
            double* p = nullptr;
            e = cudaGetSymbolAddress((void**)&p, g_partial);
            if (e != cudaSuccess || !p)
                return fail(err, err_len, JEFI_ERR_CUDA, "cudaGetSymbolAddress(g_partial)", e);
            int sms = 0;
            e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            if (e != cudaSuccess) return fail(err, err_len, JEFI_ERR_CUDA, "cudaDeviceGetAttribute", e);
            g_slot[dev].scratch = p; g_slot[dev].sm_count = sms > 0 ? sms : 1; g_slot[dev].ready = true;
        }
        slot = g_slot[dev];
    }

    // ---- launch
    RawArgs a;
    a.nsx = src->n[0]; a.nsy = src->n[1]; a.nsz = src->n[2];
    a.shx = src->spacing[0]; a.shy = src->spacing[1]; a.shz = src->spacing[2];
    a.sox = src->origin[0]; a.soy = src->origin[1]; a.soz = src->origin[2];
    if (obs->kind == 0) {
        a.nox = obs->grid.n[0]; a.noy = obs->grid.n[1];
        a.ohx = obs->grid.spacing[0]; a.ohy = obs->grid.spacing[1]; a.ohz = obs->grid.spacing[2];
        a.d0x = obs->grid.origin[0] - a.sox; a.d0y = obs->grid.origin[1] - a.soy; a.d0z = obs->grid.origin[2] - a.soz;
    } else {
        a.nox = a.noy = 1; a.ohx = a.ohy = a.ohz = 1.0; a.d0x = a.d0y = a.d0z = 0.0;
    }
    double hmin = a.shx < a.shy ? a.shx : a.shy;
    hmin = hmin < a.shz ? hmin : a.shz;
    a.rcut2 = 0.25 * hmin * hmin;                       // screening radius 0.5*min(dx,dy,dz)
    a.inv_cdt = 1.0 / (time->c * time->dt); a.inv_dt = 1.0 / time->dt; a.inv_c = 1.0 / time->c;
    a.Ns = Ns; a.obs_begin = obs_begin; a.obs_count = obs_count;
    a.T = time->nsteps; a.step = step; a.deriv_mode = time->deriv_mode;
    a.obs_kind = obs->kind; a.points = obs->points_dev;

    // source chunks: enough CTAs for a few waves, bounded by what the scratch array holds
    const long long blocks = (obs_count + kThreads - 1) / kThreads;
    long long S = (4LL * slot.sm_count + blocks - 1) / blocks;
    if (S > 64) S = 64;
    if (S > Ns / 64) S = Ns / 64;
    if (S * 6 * obs_count > kScratchElems) S = kScratchElems / (6 * obs_count);
    if (S < 1) S = 1;
    a.cells_per_chunk = (Ns + S - 1) / S;
    S = (Ns + a.cells_per_chunk - 1) / a.cells_per_chunk;

    const double pi = 3.14159265358979323846;
    const double scaleE = a.shx * a.shy * a.shz / (4.0 * pi), scaleB = time->c * scaleE;
    const cudaStream_t st = (cudaStream_t)stream;
    const dim3 grid((unsigned)blocks, (unsigned)S);
    const unsigned rgrid = (unsigned)((6 * obs_count + 255) / 256);
    if (dtype == JEFI_F32) {
        fields_point_raw_kernel<float><<<grid, kThreads, 0, st>>>((const float*)rho_dev, (const float*)J_dev, slot.scratch, a);
        reduce_scale_raw_kernel<float><<<rgrid, 256, 0, st>>>(slot.scratch, (float*)E_out_dev, (float*)B_out_dev,
                                                              obs_count, (int)S, scaleE, scaleB);
    } else {
        fields_point_raw_kernel<double><<<grid, kThreads, 0, st>>>((const double*)rho_dev, (const double*)J_dev, slot.scratch, a);
        reduce_scale_raw_kernel<double><<<rgrid, 256, 0, st>>>(slot.scratch, (double*)E_out_dev, (double*)B_out_dev,
                                                               obs_count, (int)S, scaleE, scaleB);
    }
    e = cudaPeekAtLastError();
    if (e != cudaSuccess) return fail(err, err_len, JEFI_ERR_CUDA, "kernel launch", e);
    return JEFI_OK;
}
