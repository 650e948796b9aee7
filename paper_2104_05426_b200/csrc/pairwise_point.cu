// pairwise_point.cu -- steps a2-a5 in the paper's own shape (Fig. 1): one
// thread per observation point, a serial loop over source cells, history gathered straight
// from global memory.  It is the general path (explicit point lists, any grid) and the
// bring-up/cross-check kernel; the tiled kernel (pairwise_tiled.cu) is the fast path.
// Also holds step a6, the deterministic reduce + scale + store epilogue both kernels share.
//
// Per pair (Eq. (4)-(6), in the pre-scaled variables of prepass.cu):
//   d = r - r',  R^2 = d.d,  rinv = rsqrt(R^2) (0 if R^2 < rcut^2: screening)
//   k = floor(R/(c dt) + 0.5),  p = max(n + 1 - k, 0)            (p = 0: the all-zero record)
//   s = (rho*rinv + rho_dot')*rinv^2,   u = (J'*rinv + J_dot'')*rinv^2
//   E += d*s - J_dot''*rinv,            B' += u x d               (B = c * B')
#include "tiled_common.cuh"

namespace jefi {
namespace {

// packed history: [cell][unit][p] in 16-byte units (prepass.cu); a record is 8 values
template <typename T> struct Rec { T v[8]; };
__device__ __forceinline__ Rec<float> load_rec(const float* __restrict__ hist, long long j, int Tp, int p)
{
    const float4* h = reinterpret_cast<const float4*>(hist);
    const float4 a = h[(j * 2 + 0) * Tp + p], b = h[(j * 2 + 1) * Tp + p];
    return Rec<float>{{a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w}};
}
__device__ __forceinline__ Rec<double> load_rec(const double* __restrict__ hist, long long j, int Tp, int p)
{
    const double2* h = reinterpret_cast<const double2*>(hist);
    const double2 a = h[(j * 4 + 0) * Tp + p], b = h[(j * 4 + 1) * Tp + p];
    const double2 c = h[(j * 4 + 2) * Tp + p], d = h[(j * 4 + 3) * Tp + p];
    return Rec<double>{{a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y}};
}

struct PointArgs {
    int nsx, nsy, nsz;
    int nox, noy;
    double shx, shy, shz;       // source spacing
    double ohx, ohy, ohz;       // obs spacing
    double d0x, d0y, d0z;       // obs origin - source origin (host fp64)
    double sox, soy, soz;       // source origin (for explicit point lists)
    double rcut2, inv_cdt;
    long long Ns, obs_begin, obs_count;
    int Tp, n1, origin;         // n1 = step + 1; ring origin of the packed history
    int obs_kind;
    const void* points;
    long long cells_per_chunk;
};

constexpr int kPointThreads = 128;

template <typename T>
__global__ void __launch_bounds__(kPointThreads)
fields_point_kernel(const T* __restrict__ hist, double* __restrict__ partial, PointArgs a)
{
    const long long i = (long long)blockIdx.x * kPointThreads + threadIdx.x;
    if (i >= a.obs_count) return;
    const long long gi = a.obs_begin + i;

    // observation position relative to the centre of source cell (0,0,0)
    T ox, oy, oz;
    double pdx = 0, pdy = 0, pdz = 0;       // the same in fp64 (point lists in fp32: near-tie lags)
    if (a.obs_kind == 0) {
        const int ix = (int)(gi % a.nox), iy = (int)((gi / a.nox) % a.noy);
        const int iz = (int)(gi / ((long long)a.nox * a.noy));
        ox = obs_coord<T>(a.d0x, ix, a.ohx); oy = obs_coord<T>(a.d0y, iy, a.ohy); oz = obs_coord<T>(a.d0z, iz, a.ohz);
    } else {
        const T* p = (const T*)a.points + 3 * gi;
        pdx = (double)p[0] - a.sox; pdy = (double)p[1] - a.soy; pdz = (double)p[2] - a.soz;
        ox = (T)pdx; oy = (T)pdy; oz = (T)pdz;
    }
    // fp32 on an explicit point list: pairs whose q is within tie_delta of a half-integer get
    // their lag from fp64 (tiled_common.cuh near_tie_lag); grids keep the lattice arithmetic
    const bool fix_ties = sizeof(T) == 4 && a.obs_kind == 1;
    float tie_lim = 0.f;
    if (fix_ties) {
        const double fx = fmax(fabs(pdx), fabs(pdx - (a.nsx - 1) * a.shx));
        const double fy = fmax(fabs(pdy), fabs(pdy - (a.nsy - 1) * a.shy));
        const double fz = fmax(fabs(pdz), fabs(pdz - (a.nsz - 1) * a.shz));
        tie_lim = 0.5f - tie_delta(sqrt(fx * fx + fy * fy + fz * fz) * a.inv_cdt);
    }
    const T inv_cdt_plain = (T)a.inv_cdt;
    const T shx = (T)a.shx, shy = (T)a.shy, shz = (T)a.shz;
    const T rcut2 = (T)a.rcut2, inv_cdt = -tie_biased_neg_inv_cdt<T>(a.inv_cdt);

    const long long cb = (long long)blockIdx.y * a.cells_per_chunk;
    long long ce = cb + a.cells_per_chunk;
    if (ce > a.Ns) ce = a.Ns;
    int sx = (int)(cb % a.nsx), sy = (int)((cb / a.nsx) % a.nsy);
    int sz = (int)(cb / ((long long)a.nsx * a.nsy));

    double tot[6] = {0, 0, 0, 0, 0, 0};
    long long j = cb;
    while (j < ce) {
        // one (part of a) source row: y, z fixed
        T dy, dz;
        const T ryz = row_ryz<T>(oy, oz, sy, sz, shy, shz, dy, dz);
        long long row_end = j + (a.nsx - sx);
        if (row_end > ce) row_end = ce;
        T ex = 0, ey = 0, ez = 0, bx = 0, by = 0, bz = 0;
        for (; j < row_end; ++j, ++sx) {
            T dx, rinv;
            int k;
            point_geo<T>(ox, sx, shx, ryz, rcut2, inv_cdt, dx, rinv, k);
            if (fix_ties) {
                const T e = (dx * dx + ryz) * rinv * inv_cdt_plain - (T)k;      // q - k in [-1/2, 1/2]
                if ((e < T(0) ? -e : e) >= (T)tie_lim && rinv != T(0))
                    k = near_tie_lag(pdx, pdy, pdz, sx, sy, sz, a.shx, a.shy, a.shz, a.inv_cdt);
            }
            int p = a.n1 - k;
            p = p < 0 ? 0 : p;
            const Rec<T> h = load_rec(hist, j, a.Tp, ring_slot(p, a.origin, a.Tp - 1));      // rho, rho', Jx, Jy, Jz, Jx', Jy', Jz'
            const T r2 = rinv * rinv;
            const T s  = (h.v[0] * rinv + h.v[1]) * r2;
            const T ux = (h.v[2] * rinv + h.v[5]) * r2;
            const T uy = (h.v[3] * rinv + h.v[6]) * r2;
            const T uz = (h.v[4] * rinv + h.v[7]) * r2;
            ex += dx * s - h.v[5] * rinv;
            ey += dy * s - h.v[6] * rinv;
            ez += dz * s - h.v[7] * rinv;
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

// step a6: fixed-order sum over the S source chunks, scale, store as component planes.
// One thread per (component, point); the S loads of a thread are independent (eight in flight).
template <typename T>
__global__ void __launch_bounds__(256)
reduce_scale_kernel(const double* __restrict__ partial, T* __restrict__ E, T* __restrict__ B,
                    long long count, int S, double scaleE, double scaleB)
{
    const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
    if (t >= 6 * count) return;
    const int c = (int)(t / count);
    const long long i = t - (long long)c * count;
    const double* src = partial + (long long)c * count + i;
    const long long stride = 6 * count;
    double acc = 0.0;
    int s = 0;
    for (; s + 8 <= S; s += 8) {
        double v[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) v[e] = src[(long long)(s + e) * stride];
#pragma unroll
        for (int e = 0; e < 8; ++e) acc += v[e];          // same order as a plain loop over s
    }
    for (; s < S; ++s) acc += src[(long long)s * stride];
    if (c < 3) E[(long long)c * count + i] = (T)(acc * scaleE);
    else       B[(long long)(c - 3) * count + i] = (T)(acc * scaleB);
}

}  // namespace

int launch_reduce_scale(const Params& P, jefi_dtype dt, const FieldsLaunch& L, int S)
{
    const double pi = 3.14159265358979323846;
    const double dV = P.sh[0] * P.sh[1] * P.sh[2];
    const double scaleE = dV / (4.0 * pi), scaleB = P.c * scaleE;
    const unsigned grid = (unsigned)((6 * L.obs_count + 255) / 256);
    if (dt == JEFI_F32)
        reduce_scale_kernel<float><<<grid, 256, 0, L.stream>>>(
            (const double*)L.scratch, (float*)L.E_out, (float*)L.B_out, L.obs_count, S, scaleE, scaleB);
    else
        reduce_scale_kernel<double><<<grid, 256, 0, L.stream>>>(
            (const double*)L.scratch, (double*)L.E_out, (double*)L.B_out, L.obs_count, S, scaleE, scaleB);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int launch_fields_point(const Params& P, jefi_dtype dt, const void* hist, const FieldsLaunch& L)
{
    PointArgs a;
    a.nsx = P.ns[0]; a.nsy = P.ns[1]; a.nsz = P.ns[2];
    a.nox = P.no[0]; a.noy = P.no[1];
    a.shx = P.sh[0]; a.shy = P.sh[1]; a.shz = P.sh[2];
    a.ohx = P.oh[0]; a.ohy = P.oh[1]; a.ohz = P.oh[2];
    a.d0x = P.oo[0] - P.so[0]; a.d0y = P.oo[1] - P.so[1]; a.d0z = P.oo[2] - P.so[2];
    a.sox = P.so[0]; a.soy = P.so[1]; a.soz = P.so[2];
    double hmin = P.sh[0] < P.sh[1] ? P.sh[0] : P.sh[1];
    hmin = hmin < P.sh[2] ? hmin : P.sh[2];
    a.rcut2 = 0.25 * hmin * hmin;
    a.inv_cdt = 1.0 / (P.c * P.dt);
    a.Ns = P.Ns; a.obs_begin = L.obs_begin; a.obs_count = L.obs_count;
    a.Tp = P.Tp; a.n1 = L.step + 1; a.origin = P.origin;
    a.obs_kind = P.obs_kind; a.points = P.obs_points;

    const long long blocks = (L.obs_count + kPointThreads - 1) / kPointThreads;
    long long S = (4LL * L.sm_count + blocks - 1) / blocks;
    if (S > 64) S = 64;
    if (S > P.Ns / 64) S = P.Ns / 64;
    if (S * 6 * L.obs_count > L.scratch_elems) S = L.scratch_elems / (6 * L.obs_count);
    if (S < 1) S = 1;
    a.cells_per_chunk = (P.Ns + S - 1) / S;
    S = (P.Ns + a.cells_per_chunk - 1) / a.cells_per_chunk;

    dim3 grid((unsigned)blocks, (unsigned)S);
    if (dt == JEFI_F32)
        fields_point_kernel<float><<<grid, kPointThreads, 0, L.stream>>>(
            (const float*)hist, (double*)L.scratch, a);
    else
        fields_point_kernel<double><<<grid, kPointThreads, 0, L.stream>>>(
            (const double*)hist, (double*)L.scratch, a);
    if (cudaPeekAtLastError() != cudaSuccess) return -1;
    if (launch_reduce_scale(P, dt, L, (int)S) < 0) return -1;
    return 2;
}

}  // namespace jefi
