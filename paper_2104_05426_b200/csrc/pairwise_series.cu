// pairwise_series.cu -- SURVEY.md 8(f) NEXT-1: NS consecutive output steps per (observation point,
// source cell) pair in one launch.  The paper's real workload is hundreds of snapshots on fixed
// grids (Table 2: 410 snapshots; BASELINE.json configs[3]: 128 output steps), and
// nothing in a pair's geometry -- d, R, 1/R, the retarded lag k (Eq. (6)) -- depends
// on the evaluation step n.  So a thread computes them ONCE per pair and then walks NS output
// steps n0 .. n0+NS-1, whose retarded steps m_i = n0 + i - k are CONSECUTIVE stored snapshots.
//
// What that buys.  The one-step kernel (pairwise_tiled.cu) gathers a 32-byte record {rho, rho_dot,
// J, J_dot} per pair through the shared-memory pipe, which ncu shows 89 % busy.  Here the history
// is kept as RAW 16-byte records {rho, Jx/c, Jy/c, Jz/c} per (cell, step) ("series layout", built
// from the packed history by series_layout_kernel below), a thread loads the NS+2 consecutive
// slots m_0-1 .. m_{NS-1}+1 and forms the time differences in registers: 16 (NS+2)/NS lane-bytes
// per (pair, step) -- 21.3 B at NS = 6 instead of 32 -- and the geometry (7 FMA-pipe
// instructions, the MUFU, the address) is paid once per NS steps.  With the gather relieved
// (shared pipe 54 % busy) the bound moves to the register file: an FFMA that reads two fresh
// registers and one reused one sustains 89 % of the FMA-pipe rate on this chip, three fresh ones
// 57 %, and this loop's 4 FADD + 14 FFMA per step 72 % on its own, 4.3 pair-steps per clock per SM
// with its loads (micro-benchmarks); the kernel reaches 3.7.
//
// Arithmetic per (pair, step), pre-scaled variables as in prepass.cu (E = sum d (rho/R^3 +
// rho_dot'/R^2) - J_dot''/R, B = c sum (J'/R^3 + J_dot''/R^2) x d with rho_dot' = rho_dot/c,
// J' = J/c, J_dot'' = J_dot/c^2).  With kappa = 1/(2 c dt) (centred) or 1/(c dt) (backward):
//   D = r[m+1] - r[m-1]   (centred;  backward: r[m] - r[m-1])        -> rho_dot' = kappa D.rho, J_dot'' = kappa D.J
//   ts' = rho wq + D.rho,  tJ' = J' wq + D.J,   wq = rinv / kappa    (so ts = kappa ts', tJ = kappa tJ')
//   Ex += ts' h;  S += ts' g;  E -= D.J rinv;  U += tJ' g;  Vy += tJy' h;  Vz += tJz' h      (g = rinv^2, h = dx g)
// per source row Ey += dy S, ... as in pairwise_tiled.cu; the common factor kappa is applied by
// the epilogue.  4 FADD + 14 FFMA per (pair, step) + 1 LDS.128, plus (7 FMA + MUFU + LEA + LDS
// (cell meta) + 2 LDS.128) / NS.
//
// History ends.  Series slot p = m + 2: p = 0 is all-zero (every m <= -2), p = 1 the ghost
// g(-1) = 2 f[0] - f[1], p = T + 2 the ghost g(T) = 2 f[T-1] - f[T-2], so that the centred
// difference of stored values reproduces the one-sided ends of the definition (SURVEY.md 8c:
// D(m=0) = (f[1]-f[0])/dt = kappa (f[1] - g(-1))); T = 1: both ghosts = f[0], D = 0.  Backward
// mode stores 0 at p = 1 (f[-1] = 0) and needs nothing else.  m < 0 contributes
// zero (Q4): in backward mode the zero slots do that by themselves (value 0, difference 0); in
// centred mode the ghost is not zero, so stages whose window reaches m < 0 are flagged EDGE by
// the producer and the consumers predicate each step on m_i >= 0.  Steps after the newest stored
// one never occur (n <= T-1, k >= 0).
#include "tiled_common.cuh"

namespace jefi {
namespace {

constexpr int kStageCells = 32;
constexpr unsigned kOffFull = 0, kOffEmpty = 64, kOffFlags = 128, kOffMeta = 256;

template <typename T> struct SPrec;
template <> struct SPrec<float>  { static constexpr int U = 1; };     // one float4 {rho, Jx', Jy', Jz'}
template <> struct SPrec<double> { static constexpr int U = 2; };     // double2 {rho, Jx'}, {Jy', Jz'}

struct SeriesArgs {
    int nsx, nsy, nsz;
    int nox, noy, noz;
    double shx, shy, shz;
    double ohx, ohy, ohz, d0x, d0y, d0z;
    double rcut2, inv_cdt, inv_kappa;
    int Tq;                                   // slots per (cell, unit) row: T + 3
    int step_begin, step_count;               // output steps of this launch
    int tiles_x, tiles_y, ntiles, z_first;
    long long obs_begin, obs_count;
    long long cells_per_chunk, Ns;
    int chunk_base, accumulate;
    int flush_stages, wcap, stages, stage_bytes, cps;
    double box_hx, box_hy, box_hz;
};

// ------------------------------------------------------------------ series layout from the packed history
// packed record (prepass.cu): { rho, rho_dot', Jx', Jy' | Jz', ... };  series record: { rho, Jx', Jy', Jz' }.
// One thread per (cell, slot); reads and writes are coalesced along the slot index (both layouts are
// [cell][unit][step]).  HBM-bound: 32 B read + 16 B written per record (fp32).
template <typename T>
__device__ __forceinline__ void packed_values(const T* __restrict__ packed, long long j, int Tp, int origin, int m, T (&f)[4])
{
    // values rho, Jx', Jy', Jz' of stored step m (packed step m + 1)
    constexpr int VPU = 16 / sizeof(T), U = 8 / VPU;
    const long long base = (j * U) * (long long)Tp + ring_slot(m + 1, origin, Tp - 1);
    constexpr int idx[4] = {0, 2, 3, 4};
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int u = idx[q] / VPU, e = idx[q] % VPU;
        f[q] = packed[(base + (long long)u * Tp) * VPU + e];
    }
}

template <typename T>
__global__ void __launch_bounds__(256)
series_layout_kernel(const T* __restrict__ packed, T* __restrict__ series, long long Ns, int Tsteps, int Tp, int Tq,
                     int backward, int origin)
{
    constexpr int VPU = 16 / sizeof(T), U = 4 / VPU;         // series units per record: 1 (fp32), 2 (fp64)
    const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
    if (t >= Ns * Tq) return;
    const long long j = t / Tq;
    const int p = (int)(t - j * Tq);
    T f[4] = {0, 0, 0, 0};
    const int m = p - 2;
    if (m >= 0 && m < Tsteps) {
        packed_values<T>(packed, j, Tp, origin, m, f);
    } else if (!backward && (m == -1 || m == Tsteps)) {
        // ghost: 2 f[end] - f[next to end] (one rounding); T = 1: f[0]
        const int e = m == -1 ? 0 : Tsteps - 1, e2 = m == -1 ? 1 : Tsteps - 2;
        T a[4], b[4];
        packed_values<T>(packed, j, Tp, origin, e, a);
        if (Tsteps >= 2) {
            packed_values<T>(packed, j, Tp, origin, e2, b);
#pragma unroll
            for (int q = 0; q < 4; ++q) f[q] = fma_t<T>(T(2), a[q], -b[q]);
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) f[q] = a[q];
        }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
        T* dst = series + ((j * U + u) * (long long)Tq + p) * VPU;
#pragma unroll
        for (int e = 0; e < VPU; ++e) dst[e] = f[u * VPU + e];
    }
}

// ------------------------------------------------------------------ consumers
template <typename T, int NS> struct SAcc {
    T ex[NS], ey[NS], ez[NS], bx[NS], by[NS], bz[NS];     // running sums over the chunk
    T s[NS], ux[NS], uy[NS], uz[NS], vy[NS], vz[NS];      // per source row
};

__device__ __forceinline__ void load_raw(unsigned addr, unsigned, float (&v)[4])
{
    const float4 a = lds128(addr);
    v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
}
__device__ __forceinline__ void load_raw(unsigned addr, unsigned unit_off, double (&v)[4])
{
    const double2 a = lds128d(addr), b = lds128d(addr + unit_off);
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}

// per-launch constants in the kernel's own precision (kernel parameters live in the constant
// bank: the FMA-pipe instructions take them as operands without a register read)
template <typename T> struct SConsts { T neg_inv_cdt, rcut2, inv_kappa, shy, shz; };

// geometry of one pair: the slot address of its first record, the screening weight, dx
template <typename T> struct SGeo { unsigned addr; T w, dx; int m0; };

template <typename T, bool SLOW, bool EDGE>
__device__ __forceinline__ SGeo<T> series_geo(T ox, T ryz, unsigned meta_addr, const SConsts<T>& k, int n0)
{
    unsigned C;
    T sx;
    if constexpr (sizeof(T) == 4) {
        const float4 mv = lds128(meta_addr);
        C = __float_as_uint(mv.x); sx = mv.y;
    } else {
        const double2 mv = lds128d(meta_addr);
        C = (unsigned)__double2loint(mv.x); sx = mv.y;
    }
    SGeo<T> G;
    unsigned bits;
    pair_geo<T, SLOW>(ox, sx, ryz, k.neg_inv_cdt, k.rcut2, G.dx, G.w, bits);
    G.addr = C + (bits << 4);
    G.m0 = EDGE ? n0 - lag_of_bits(bits, Prec<T>::kMagicLo) : 0;
    return G;
}

// one pair, NS steps.  NL = slots loaded: NS + 2 (centred), NS + 1 (backward)
template <typename T, int NS, bool EDGE, bool BACKWARD>
__device__ __forceinline__ void series_accumulate(SAcc<T, NS>& a, const SGeo<T>& G, T inv_kappa, unsigned unit_off,
                                                  const T (&r)[BACKWARD ? NS + 1 : NS + 2][4])
{
    const T w = G.w;
    const T g = w * w;
    const T h = G.dx * g;
    const T wq = w * inv_kappa;
#pragma unroll
    for (int i = 0; i < NS; ++i) {
        if (EDGE && G.m0 + i < 0) continue;          // before the stored history: zero contribution (Q4)
        const T* v = r[i + 1];
        T d[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) d[q] = BACKWARD ? v[q] - r[i][q] : r[i + 2][q] - r[i][q];
        const T ts = fma_t<T>(v[0], wq, d[0]);
        const T tx = fma_t<T>(v[1], wq, d[1]);
        const T ty = fma_t<T>(v[2], wq, d[2]);
        const T tz = fma_t<T>(v[3], wq, d[3]);
        a.ex[i] = fma_t<T>(ts, h, a.ex[i]);
        a.s[i]  = fma_t<T>(ts, g, a.s[i]);
        a.ex[i] = fma_t<T>(-d[1], w, a.ex[i]);
        a.ey[i] = fma_t<T>(-d[2], w, a.ey[i]);
        a.ez[i] = fma_t<T>(-d[3], w, a.ez[i]);
        a.ux[i] = fma_t<T>(tx, g, a.ux[i]);
        a.uy[i] = fma_t<T>(ty, g, a.uy[i]);
        a.uz[i] = fma_t<T>(tz, g, a.uz[i]);
        a.vy[i] = fma_t<T>(ty, h, a.vy[i]);
        a.vz[i] = fma_t<T>(tz, h, a.vz[i]);
    }
}

// One source row (or the part of it in this stage).  Software pipeline: the geometry of cell
// c+1 (meta load -> distance -> MUFU -> lag -> address: one long dependency chain) is computed
// beside the record loads and the accumulation of cell c.  The look-ahead past the last cell
// reads a meta slot that may be stale; its geometry is computed and never used.
template <typename T, int NS, bool SLOW, bool EDGE, bool BACKWARD>
__device__ __forceinline__ void row_series(SAcc<T, NS>& a, T ox, T ryz, unsigned meta_addr, int len,
                                           const SConsts<T>& k, int n0, unsigned unit_off)
{
    constexpr int NL = BACKWARD ? NS + 1 : NS + 2;
    SGeo<T> G = series_geo<T, SLOW, EDGE>(ox, ryz, meta_addr, k, n0);
#pragma unroll 1
    for (int c = 0; c < len; ++c) {
        T r[NL][4];
#pragma unroll
        for (int i = 0; i < NL; ++i) load_raw(G.addr + 16u * i, unit_off, r[i]);
        const SGeo<T> Gn = series_geo<T, SLOW, EDGE>(ox, ryz, meta_addr + (c + 1) * 16u, k, n0);
        series_accumulate<T, NS, EDGE, BACKWARD>(a, G, k.inv_kappa, unit_off, r);
        G = Gn;
    }
}

template <typename T, int NS>
__device__ __forceinline__ void fold_row_series(SAcc<T, NS>& a, T dy, T dz)
{
#pragma unroll
    for (int i = 0; i < NS; ++i) {
        a.ey[i] = fma_t<T>(dy, a.s[i], a.ey[i]);
        a.ez[i] = fma_t<T>(dz, a.s[i], a.ez[i]);
        a.bx[i] += a.uy[i] * dz - a.uz[i] * dy;
        a.by[i] += a.vz[i] - a.ux[i] * dz;
        a.bz[i] += a.ux[i] * dy - a.vy[i];
        a.s[i] = a.ux[i] = a.uy[i] = a.uz[i] = a.vy[i] = a.vz[i] = T(0);
    }
}

// A CTA = CW consumer warps (one observation point per thread: TX x TY x TZ = 32 CW points) + one
// producer warp; grid.x = tile + ntiles * (step block), grid.y = source chunk.
template <typename T, int NS, int TX, int TY, int TZ, int CW, int CTAS, bool BACKWARD>
__global__ void __launch_bounds__((CW + 1) * 32, CTAS)
fields_series_kernel(const uint4* __restrict__ hist, double* __restrict__ partial, const SeriesArgs a,
                     const SConsts<T> k)
{
    constexpr int U = SPrec<T>::U;
    static_assert(TX == 8 && TY % 4 == 0 && TX * TY * TZ == CW * 32, "a warp covers 8 x 4 points of one z layer");
    extern __shared__ __align__(128) unsigned char smem[];
    const unsigned sbase = smem_u32(smem);
    const unsigned data0 = sbase + kOffMeta + (unsigned)a.stages * kStageCells * 16u;
    const unsigned unit_off = (unsigned)a.wcap * 16u;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    const int tile = (int)(blockIdx.x % (unsigned)a.ntiles);
    const int blk = (int)(blockIdx.x / (unsigned)a.ntiles);
    const int n0 = a.step_begin + blk * NS;                       // first output step of this CTA
    const int ix0 = (tile % a.tiles_x) * TX;
    const int iy0 = ((tile / a.tiles_x) % a.tiles_y) * TY;
    const int iz0 = a.z_first + (tile / (a.tiles_x * a.tiles_y)) * TZ;
    const long long cb = (long long)(a.chunk_base + (int)blockIdx.y) * a.cells_per_chunk;
    const long long ce = (cb + a.cells_per_chunk < a.Ns) ? cb + a.cells_per_chunk : a.Ns;
    const int nst = (int)((ce - cb + a.cps - 1) / a.cps);

    if (tid == 0) {
        for (int s = 0; s < a.stages; ++s) {
            mbar_init(sbase + kOffFull + 8 * s, 32);
            mbar_init(sbase + kOffEmpty + 8 * s, CW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == CW) {
        // ------------------------------------------------------------ producer warp
        const double bx0 = a.d0x + ix0 * a.ohx, bx1 = bx0 + a.box_hx;
        const double by0 = a.d0y + iy0 * a.ohy, by1 = by0 + a.box_hy;
        const double bz0 = a.d0z + iz0 * a.ohz, bz1 = bz0 + a.box_hz;
        for (int it = 0; it < nst; ++it) {
            const int s = it % a.stages;
            if (it >= a.stages) mbar_wait_parked(sbase + kOffEmpty + 8 * s, ((it / a.stages) - 1) & 1);
            const long long j = cb + (long long)it * a.cps + lane;
            const bool valid = lane < a.cps && j < ce;
            int flags = 0, p_src = 0, cnt = 0, nz = 0;
            unsigned row0 = 0;
            if (valid) {
                const int jx = (int)(j % a.nsx), jy = (int)((j / a.nsx) % a.nsy);
                const int jz = (int)(j / ((long long)a.nsx * a.nsy));
                int kmin, kmax;
                double dmin2;
                cell_lag_bounds(jx * a.shx, jy * a.shy, jz * a.shz, bx0, bx1, by0, by1, bz0, bz1, a.inv_cdt, kmin, kmax,
                                dmin2);
                // window slot i <-> stored step m = n0 - kmax - 1 + i, i.e. series slot p = p_lo + i;
                // a pair with lag k reads slots (kmax - k) .. (kmax - k) + NS + 1
                const int p_lo = n0 - kmax + 1;
                int span = kmax - kmin + NS + 2;
                span = span > a.wcap ? a.wcap : span;
                if (dmin2 <= a.rcut2 * 1.001) flags |= 1;
                if (!BACKWARD && kmax > n0) flags |= 2;          // some pair may have m_0 < 0
                nz = p_lo < 0 ? -p_lo : 0;
                nz = nz > span ? span : nz;
                p_src = p_lo < 0 ? 0 : p_lo;
                int p_hi = p_lo + span - 1;
                p_hi = p_hi > a.Tq - 1 ? a.Tq - 1 : p_hi;
                cnt = p_hi >= p_src ? p_hi - p_src + 1 : 0;
                row0 = data0 + (unsigned)s * (unsigned)a.stage_bytes + (unsigned)lane * (unsigned)U * unit_off;
                const unsigned C = row0 + ((unsigned)kmax << 4) - (Prec<T>::kMagicLo << 4);
                if constexpr (sizeof(T) == 4) {
                    float4 m;
                    m.x = __uint_as_float(C); m.y = src_coord<T>(jx, a.shx); m.z = 0.f; m.w = 0.f;
                    *reinterpret_cast<float4*>(smem + kOffMeta + (s * kStageCells + lane) * 16) = m;
                } else {
                    double2 m;
                    m.x = __hiloint2double(0, (int)C); m.y = src_coord<T>(jx, a.shx);
                    *reinterpret_cast<double2*>(smem + kOffMeta + (s * kStageCells + lane) * 16) = m;
                }
                // slots before the stored history, and (ragged last step block only) after it
                for (int z = 0; z < span; ++z) {
                    if (z >= nz && z < nz + cnt) { z = nz + cnt - 1; continue; }
#pragma unroll
                    for (int u = 0; u < U; ++u) sts128_zero(row0 + u * unit_off + (unsigned)z * 16u);
                }
            }
            const unsigned any = __reduce_or_sync(0xffffffffu, (unsigned)flags);
            if (lane == 0) *reinterpret_cast<int*>(smem + kOffFlags + 4 * s) = (int)any;
            const unsigned bar = sbase + kOffFull + 8 * s;
            if (valid && cnt > 0) {
                const unsigned bytes = (unsigned)cnt * 16u;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                mbar_arrive_expect_tx(bar, (unsigned)U * bytes);
                const uint4* src = hist + ((size_t)j * U) * a.Tq + p_src;
#pragma unroll
                for (int u = 0; u < U; ++u)
                    bulk_g2s(row0 + u * unit_off + (unsigned)nz * 16u, src + (size_t)u * a.Tq, bytes, bar);
            } else {
                mbar_arrive(bar);
            }
        }
        return;
    }

    // ---------------------------------------------------------------- consumer warps
    // a quarter-warp (one LDS.128 wavefront) covers a compact 4 x 2 patch: lags within ~6 of each
    // other at dx/(c dt) = 2, so its 16-byte slots fall into distinct bank groups
    const int lx = (lane & 3) | ((lane >> 1) & 4);
    const int ly = ((lane >> 2) & 1) | ((lane >> 3) & 2);
    const int wy = warp % (TY / 4), wz = warp / (TY / 4);
    int ix = ix0 + lx, iy = iy0 + ly + 4 * wy, iz = iz0 + wz;
    const long long gi = ((long long)iz * a.noy + iy) * a.nox + ix - a.obs_begin;
    const bool wanted = ix < a.nox && iy < a.noy && iz < a.noz && gi >= 0 && gi < a.obs_count;
    if (!__any_sync(0xffffffffu, wanted)) {
        // a warp none of whose points is requested only keeps the stage protocol going
        for (int it = 0; it < nst; ++it) {
            const int s = it % a.stages;
            mbar_wait(sbase + kOffFull + 8 * s, (it / a.stages) & 1);
            __syncwarp();
            if (lane == 0) mbar_arrive(sbase + kOffEmpty + 8 * s);
        }
        return;
    }
    // lanes outside the grid compute a copy of an edge point (their lags must stay inside the
    // tile's windows) and store nothing
    ix = ix < a.nox ? ix : a.nox - 1; iy = iy < a.noy ? iy : a.noy - 1; iz = iz < a.noz ? iz : a.noz - 1;
    const T ox = obs_coord<T>(a.d0x, ix, a.ohx), oy = obs_coord<T>(a.d0y, iy, a.ohy), oz = obs_coord<T>(a.d0z, iz, a.ohz);
    SAcc<T, NS> acc;
#pragma unroll
    for (int i = 0; i < NS; ++i) {
        acc.ex[i] = acc.ey[i] = acc.ez[i] = acc.bx[i] = acc.by[i] = acc.bz[i] = T(0);
        acc.s[i] = acc.ux[i] = acc.uy[i] = acc.uz[i] = acc.vy[i] = acc.vz[i] = T(0);
    }
    int jx = (int)(cb % a.nsx), jy = (int)((cb / a.nsx) % a.nsy), jz = (int)(cb / ((long long)a.nsx * a.nsy));
    int since = 0;
    bool first = a.accumulate == 0;
    int nvalid = a.step_count - blk * NS;                          // steps of this block that exist
    nvalid = nvalid > NS ? NS : nvalid;

    for (int it = 0; it < nst; ++it) {
        const int s = it % a.stages;
        mbar_wait(sbase + kOffFull + 8 * s, (it / a.stages) & 1);
        const long long j0 = cb + (long long)it * a.cps;
        const int cnt = (int)((ce - j0) < a.cps ? (ce - j0) : a.cps);
        const int flags = *reinterpret_cast<volatile int*>(smem + kOffFlags + 4 * s);
        int pos = 0;
        while (pos < cnt) {
            int len = a.nsx - jx;
            len = len < cnt - pos ? len : cnt - pos;
            T dy, dz;
            const T ryz = row_ryz<T>(oy, oz, jy, jz, k.shy, k.shz, dy, dz);
            const unsigned meta_addr = sbase + kOffMeta + (unsigned)(s * kStageCells + pos) * 16u;
            switch (flags) {
                case 0:  row_series<T, NS, false, false, BACKWARD>(acc, ox, ryz, meta_addr, len, k, n0, unit_off); break;
                case 1:  row_series<T, NS, true,  false, BACKWARD>(acc, ox, ryz, meta_addr, len, k, n0, unit_off); break;
                case 2:  row_series<T, NS, false, true,  BACKWARD>(acc, ox, ryz, meta_addr, len, k, n0, unit_off); break;
                default: row_series<T, NS, true,  true,  BACKWARD>(acc, ox, ryz, meta_addr, len, k, n0, unit_off); break;
            }
            pos += len; jx += len;
            const bool row_done = jx == a.nsx;
            if (row_done || (it == nst - 1 && pos == cnt)) fold_row_series<T, NS>(acc, dy, dz);
            if (row_done) { jx = 0; if (++jy == a.nsy) { jy = 0; ++jz; } }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(sbase + kOffEmpty + 8 * s);

        // running sums -> double partial sums [chunk][step][6][point] of this launch (owned by
        // this thread: plain read-modify-write), every flush_stages stages in fp32
        if (++since == a.flush_stages || it == nst - 1) {
            since = 0;
            if (wanted) {
#pragma unroll
                for (int i = 0; i < NS; ++i) {
                    if (i < nvalid) {
                        double* out = partial + (((long long)blockIdx.y * a.step_count + (blk * NS + i)) * 6) * a.obs_count + gi;
                        const T v[6] = {acc.ex[i], acc.ey[i], acc.ez[i], acc.bx[i], acc.by[i], acc.bz[i]};
#pragma unroll
                        for (int c = 0; c < 6; ++c) {
                            double* q = out + (long long)c * a.obs_count;
                            *q = first ? (double)v[c] : *q + (double)v[c];
                        }
                    }
                }
            }
#pragma unroll
            for (int i = 0; i < NS; ++i)
                acc.ex[i] = acc.ey[i] = acc.ez[i] = acc.bx[i] = acc.by[i] = acc.bz[i] = T(0);
            first = false;
        }
    }
}

// step a6 for a series: fixed-order sum over the S source chunks, scale, store E[step][3][count]
template <typename T>
__global__ void __launch_bounds__(256)
reduce_scale_series_kernel(const double* __restrict__ partial, T* __restrict__ E, T* __restrict__ B, long long count,
                           int steps, int S, double scaleE, double scaleB)
{
    const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
    const long long per_step = 6 * count;
    if (t >= per_step * steps) return;
    const long long st = t / per_step;
    const long long r = t - st * per_step;
    const int c = (int)(r / count);
    const long long i = r - (long long)c * count;
    const double* src = partial + t;
    const long long stride = per_step * steps;
    double acc = 0.0;
    for (int s = 0; s < S; ++s) acc += src[(long long)s * stride];
    if (c < 3) E[(st * 3 + c) * count + i] = (T)(acc * scaleE);
    else       B[(st * 3 + (c - 3)) * count + i] = (T)(acc * scaleB);
}

template <typename T, int NS, int TX, int TY, int TZ, int CW, int CTAS, bool BACKWARD>
int launch_series_shape(const Params& P, jefi_dtype dt, const void* series, const FieldsLaunch& L, int step_begin,
                        int step_count)
{
    constexpr int U = SPrec<T>::U;
    constexpr int kThreads = (CW + 1) * 32;
    const long long plane = (long long)P.no[0] * P.no[1];
    const int z_first = (int)(L.obs_begin / plane);
    const int z_last = (int)((L.obs_begin + L.obs_count - 1) / plane);

    SeriesArgs a;
    a.nsx = P.ns[0]; a.nsy = P.ns[1]; a.nsz = P.ns[2];
    a.nox = P.no[0]; a.noy = P.no[1]; a.noz = P.no[2];
    a.shx = P.sh[0]; a.shy = P.sh[1]; a.shz = P.sh[2];
    a.ohx = P.oh[0]; a.ohy = P.oh[1]; a.ohz = P.oh[2];
    a.d0x = P.oo[0] - P.so[0]; a.d0y = P.oo[1] - P.so[1]; a.d0z = P.oo[2] - P.so[2];
    double hmin = P.sh[0] < P.sh[1] ? P.sh[0] : P.sh[1];
    hmin = hmin < P.sh[2] ? hmin : P.sh[2];
    a.rcut2 = 0.25 * hmin * hmin;
    a.inv_cdt = 1.0 / (P.c * P.dt);
    const double kappa = (BACKWARD ? 1.0 : 0.5) * a.inv_cdt;
    a.inv_kappa = 1.0 / kappa;
    SConsts<T> k;
    k.neg_inv_cdt = tie_biased_neg_inv_cdt<T>(a.inv_cdt); k.rcut2 = (T)a.rcut2; k.inv_kappa = (T)a.inv_kappa;
    k.shy = (T)P.sh[1]; k.shz = (T)P.sh[2];
    a.Tq = P.T + 3;
    a.tiles_x = (P.no[0] + TX - 1) / TX;
    a.tiles_y = (P.no[1] + TY - 1) / TY;
    a.z_first = z_first;
    const int tiles_z = (z_last - z_first + TZ) / TZ;
    a.ntiles = a.tiles_x * a.tiles_y * tiles_z;
    a.obs_begin = L.obs_begin; a.obs_count = L.obs_count;
    a.Ns = P.Ns;
    const double ex = (TX - 1) * P.oh[0], ey = (TY - 1) * P.oh[1], ez = (TZ - 1) * P.oh[2];
    a.box_hx = ex; a.box_hy = ey; a.box_hz = ez;

    // window capacity: the lag of one cell varies over a tile by at most diam/(c dt); +5 covers the
    // rounding of both ends and the margins; + NS + 1 more slots for the NS steps and their neighbours
    const double diam = sqrt(ex * ex + ey * ey + ez * ez);
    const double wd = floor(diam * a.inv_cdt) + 5.0 + NS + 1;
    if (wd > 1.0e6) return 0;
    const double far = sqrt(pow(fabs(a.d0x) + ex + P.no[0] * P.oh[0] + P.ns[0] * P.sh[0], 2) +
                            pow(fabs(a.d0y) + ey + P.no[1] * P.oh[1] + P.ns[1] * P.sh[1], 2) +
                            pow(fabs(a.d0z) + ez + P.no[2] * P.oh[2] + P.ns[2] * P.sh[2], 2));
    if (far * a.inv_cdt > kMaxLagSteps) return 0;
    a.wcap = ((int)wd + 7) / 8 * 8;

    const int cell_bytes = U * a.wcap * 16;
    const int budget = 227 * 1024 / CTAS - 2048;
    int cps = 0, stages = 0;
    for (int c = 32; c >= 1 && !cps; c = c > 4 ? c - 4 : c - 1) {
        const int st = (budget - (int)kOffMeta) / (c * cell_bytes + 512);
        if (st >= 2) { cps = c; stages = st > 4 ? 4 : st; }
    }
    if (!cps) return 0;
    a.flush_stages = sizeof(T) == 4 ? (2048 / cps > 0 ? 2048 / cps : 1) : (1 << 30);
    a.cps = cps; a.stages = stages; a.stage_bytes = cps * cell_bytes;
    const int smem = (int)kOffMeta + stages * 512 + stages * a.stage_bytes;

    auto kern = fields_series_kernel<T, NS, TX, TY, TZ, CW, CTAS, BACKWARD>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return -1;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kThreads, smem) != cudaSuccess) return -1;
    if (per_sm < 1) return 0;

    // steps per launch batch: the partial sums [S][steps][6][points] must fit the scratch
    long long sb = L.scratch_elems / (6 * L.obs_count);
    if (sb < 1) return 0;
    if (sb >= step_count) sb = step_count;
    else if (sb >= NS) sb = sb / NS * NS;
    const double pi = 3.14159265358979323846;
    const double dV = P.sh[0] * P.sh[1] * P.sh[2];
    const double scaleE = dV / (4.0 * pi) * kappa, scaleB = P.c * scaleE;

    int launches = 0;
    for (int b0 = 0; b0 < step_count; b0 += (int)sb) {
        const int steps = step_count - b0 < sb ? step_count - b0 : (int)sb;
        const int nblocks = (steps + NS - 1) / NS;
        a.step_begin = step_begin + b0; a.step_count = steps;
        // source chunks: (1) ~4 waves of CTAs when the problem is small, full last wave preferred;
        // (2) a chunk's series history below chunk_bytes (L2 sharing, see pairwise_tiled.cu);
        // (3) S chunks per launch must fit the scratch, the rest goes to accumulating launches
        const long long nct = (long long)a.ntiles * nblocks;
        const long long slots = (long long)L.sm_count * per_sm;
        long long smax = P.Ns / ((long long)cps * 2);
        if (smax > 65535) smax = 65535;
        if (smax < 1) smax = 1;
        long long s_launch = L.scratch_elems / (6 * L.obs_count * steps);
        if (s_launch < 1) s_launch = 1;
        long long s0 = (4 * slots + nct - 1) / nct;
        if (s0 > s_launch) s0 = s_launch;
        long long s_hi = 4 * s0 < s_launch ? 4 * s0 : s_launch;
        if (P.Ns < s0 * cps * 8) {
            s0 = slots / nct;
            if (s0 < 1) s0 = 1;
            if (s0 > s_launch) s0 = s_launch;
            s_hi = s0;
        }
        const double cell_hist_bytes = (double)U * (double)a.Tq * 16.0;
        const long long s_l2 = (long long)ceil((double)P.Ns * cell_hist_bytes / (double)L.chunk_bytes);
        if (s0 < s_l2) { s0 = s_l2; s_hi = 4 * s_l2; }
        if (s0 > smax) s0 = smax;
        if (s_hi > smax) s_hi = smax;
        long long S = s0;
        double best = -1.0;
        for (long long s = s0; s <= s_hi; ++s) {
            const double waves = (double)(nct * s) / (double)slots;
            const double eff = waves / ceil(waves);
            if (eff > best + 1e-9) { best = eff; S = s; }
        }
        a.cells_per_chunk = (P.Ns + S - 1) / S;
        a.cells_per_chunk = (a.cells_per_chunk + cps - 1) / cps * cps;
        S = (P.Ns + a.cells_per_chunk - 1) / a.cells_per_chunk;
        if (s_launch > S) s_launch = S;
        for (long long base = 0; base < S; base += s_launch) {
            const long long sl = S - base < s_launch ? S - base : s_launch;
            a.chunk_base = (int)base;
            a.accumulate = base > 0 ? 1 : 0;
            dim3 grid((unsigned)nct, (unsigned)sl);
            kern<<<grid, kThreads, smem, L.stream>>>((const uint4*)series, (double*)L.scratch, a, k);
            if (cudaPeekAtLastError() != cudaSuccess) return -1;
            ++launches;
        }
        const long long total = 6 * L.obs_count * steps;
        const size_t out_off = (size_t)b0 * 3 * (size_t)L.obs_count;
        reduce_scale_series_kernel<T><<<(unsigned)((total + 255) / 256), 256, 0, L.stream>>>(
            (const double*)L.scratch, (T*)L.E_out + out_off, (T*)L.B_out + out_off, L.obs_count, steps, (int)s_launch,
            scaleE, scaleB);
        if (cudaPeekAtLastError() != cudaSuccess) return -1;
        ++launches;
    }
    return launches;
}

template <typename T, int NS, int CTAS>
int launch_series_T(const Params& P, jefi_dtype dt, const void* series, const FieldsLaunch& L, int step_begin,
                    int step_count)
{
    const long long plane = (long long)P.no[0] * P.no[1];
    const long long nz = (L.obs_begin + L.obs_count - 1) / plane - L.obs_begin / plane + 1;
    const bool bw = P.deriv_mode == 1;
    if (nz <= 2) {
        return bw ? launch_series_shape<T, NS, 8, 16, 1, 4, CTAS, true>(P, dt, series, L, step_begin, step_count)
                  : launch_series_shape<T, NS, 8, 16, 1, 4, CTAS, false>(P, dt, series, L, step_begin, step_count);
    }
    return bw ? launch_series_shape<T, NS, 8, 4, 4, 4, CTAS, true>(P, dt, series, L, step_begin, step_count)
              : launch_series_shape<T, NS, 8, 4, 4, 4, CTAS, false>(P, dt, series, L, step_begin, step_count);
}

}  // namespace

int launch_series_layout(const Params& P, jefi_dtype dt, const void* packed, void* series, cudaStream_t stream)
{
    const int Tq = P.T + 3;
    const long long total = P.Ns * Tq;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    if (dt == JEFI_F32)
        series_layout_kernel<float><<<blocks, 256, 0, stream>>>((const float*)packed, (float*)series, P.Ns, P.T, P.Tp,
                                                                 Tq, P.deriv_mode, P.origin);
    else
        series_layout_kernel<double><<<blocks, 256, 0, stream>>>((const double*)packed, (double*)series, P.Ns, P.T,
                                                                  P.Tp, Tq, P.deriv_mode, P.origin);
    return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int series_block_steps(jefi_dtype dt) { return dt == JEFI_F32 ? 6 : 4; }

int launch_fields_series(const Params& P, jefi_dtype dt, const void* series, const FieldsLaunch& L, int step_begin,
                         int step_count)
{
    if (P.obs_kind != 0) return 0;
    // Block length NS and CTAs per SM, measured on c4 (128 steps, ms per series) and the paper's X1
    // series (411 steps on 15^3).  fp32, (NS, CTAs/SM, geometry look-ahead): (8,3,no) 894 / 10.5,
    // (8,3,yes: spills) 1026 / 10.2, (8,2,no) 929 / 9.9, (8,2,yes) 851 / 9.0, (6,3,no) 957 / 8.8,
    // (6,3,yes) 871 / 7.9, (4,3,no) 996; a 256-point tile, one CTA per SM: 933.  fp64 on c4:
    // (4,2,no) 1875, (4,2,yes) 1784, (2,3,yes) 1961, (6,1,yes) 1902, (4,1,yes) 2066, (3,2,yes) 1830.
    if (dt == JEFI_F32) return launch_series_T<float, 6, 3>(P, dt, series, L, step_begin, step_count);
    return launch_series_T<double, 4, 2>(P, dt, series, L, step_begin, step_count);
}

}  // namespace jefi
