// pairwise_list.cu -- steps a2-a5 for EXPLICIT OBSERVATION POINT LISTS (jefi_obs_desc kind 1) on
// the tiled fast path (lower item).  The tiled kernel of pairwise_tiled.cu gets
// its speed from one fact: the points of a CTA are close together, so for one source cell their
// retarded lags fall in a short window that a producer warp can stage in shared memory with one
// TMA bulk copy per unit.  A point list has no such structure by itself, so jefi_create gives it
// one: the points are binned on a regular 64^3 lattice over their bounding box, the bins are
// visited along a Hilbert curve, and every run of 512 (fp32) / 256 (fp64) points in that order
// becomes a tile with its own bounding box (list_* kernels below; once, at
// jefi_create -- the positions belong to the context like a grid does).  fields_list_kernel is
// then the tiled kernel with two differences: the tile's box comes from that table instead of
// index arithmetic, and every point of a thread has its own (y, z), so dy^2 + dz^2 and the
// per-row fold are per point instead of per thread.  Results are stored by ORIGINAL index: the
// partial sums, the epilogue and the caller never see the permutation.
//
// A quarter-warp (one LDS.128 wavefront) takes 8 consecutive points of that order, i.e.
// roughly one bin: their lags against one cell differ by a few steps, so their 16-byte slots
// fall in distinct bank groups most of the time, as in a grid tile.
#include <math.h>
#include "tiled_step.cuh"

namespace jefi {
namespace {

// ------------------------------------------------------------------ binning (jefi_create)
// order-preserving map double -> unsigned long long, for atomicMin/Max on coordinates
__device__ __forceinline__ unsigned long long ord(double x)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(x);
    return (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
}
__host__ __device__ inline double unord(unsigned long long u)
{
    const unsigned long long b = (u & 0x8000000000000000ull) ? (u & 0x7fffffffffffffffull) : ~u;
    double x;
    memcpy(&x, &b, sizeof(x));
    return x;
}

template <typename T>
__global__ void __launch_bounds__(256)
list_bbox_kernel(const T* __restrict__ pts, long long n, unsigned long long* __restrict__ mm /* [6]: min xyz, max xyz */)
{
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256)
        for (int a = 0; a < 3; ++a) {
            const double v = (double)pts[3 * i + a];
            // a NaN or Inf position makes the box infinite: build_tiles_T reports it
            if (!isfinite(v)) { lo[a] = -INFINITY; hi[a] = INFINITY; continue; }
            lo[a] = v < lo[a] ? v : lo[a]; hi[a] = v > hi[a] ? v : hi[a];
        }
    for (int a = 0; a < 3; ++a) {
        for (int o = 16; o; o >>= 1) {
            lo[a] = fmin(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = fmax(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
        }
        if ((threadIdx.x & 31) == 0) { atomicMin(mm + a, ord(lo[a])); atomicMax(mm + 3 + a, ord(hi[a])); }
    }
}

// Position of bin (x, y, z), 6 bits per axis, along the 3-D Hilbert curve (Skilling's transpose
// form of the published algorithm: inverse undo, Gray encode, interleave).  Unlike the Morton
// order, consecutive positions are always face-neighbours, so ANY run of consecutive bins is
// spatially compact -- a Morton run that crosses an octant boundary spans the whole domain
// (measured: the worst of the 128 tiles of 65 536 random points had a box diagonal of 18.7 of
// the domain's 22.2, which sets the window capacity of the whole launch).
__device__ __forceinline__ unsigned hilbert18(unsigned x, unsigned y, unsigned z)
{
    unsigned X[3] = {x, y, z};
    const unsigned M = 1u << 5;
    for (unsigned Q = M; Q > 1; Q >>= 1) {
        const unsigned Pm = Q - 1;
        for (int i = 0; i < 3; ++i) {
            if (X[i] & Q) X[0] ^= Pm;
            else { const unsigned t = (X[0] ^ X[i]) & Pm; X[0] ^= t; X[i] ^= t; }
        }
    }
    for (int i = 1; i < 3; ++i) X[i] ^= X[i - 1];
    unsigned t = 0;
    for (unsigned Q = M; Q > 1; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1;
    for (int i = 0; i < 3; ++i) X[i] ^= t;
    unsigned h = 0;
    for (int b = 5; b >= 0; --b)
        for (int i = 0; i < 3; ++i) h = (h << 1) | ((X[i] >> b) & 1u);
    return h;
}

struct BinArgs { double lo[3], inv[3]; int nb; };

template <typename T>
__global__ void __launch_bounds__(256)
list_key_kernel(const T* __restrict__ pts, long long n, BinArgs b, unsigned* __restrict__ key, unsigned* __restrict__ hist)
{
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    unsigned q[3];
    for (int a = 0; a < 3; ++a) {
        int v = (int)floor(((double)pts[3 * i + a] - b.lo[a]) * b.inv[a]);
        v = v < 0 ? 0 : (v >= b.nb ? b.nb - 1 : v);
        q[a] = (unsigned)v;
    }
    const unsigned k = hilbert18(q[0], q[1], q[2]);
    key[i] = k;
    atomicAdd(hist + k, 1u);
}

// exclusive scan of the (<= 2^18) bin counts, one block
__global__ void __launch_bounds__(1024) list_scan_kernel(unsigned* __restrict__ hist, int nbins)
{
    __shared__ unsigned part[1024];
    const int per = (nbins + 1023) / 1024;
    const int b0 = threadIdx.x * per, b1 = b0 + per < nbins ? b0 + per : nbins;
    unsigned s = 0;
    for (int i = b0; i < b1; ++i) s += hist[i];
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned run = 0;
        for (int i = 0; i < 1024; ++i) { const unsigned v = part[i]; part[i] = run; run += v; }
    }
    __syncthreads();
    unsigned run = part[threadIdx.x];
    for (int i = b0; i < b1; ++i) { const unsigned v = hist[i]; hist[i] = run; run += v; }
}

__global__ void __launch_bounds__(256)
list_scatter_kernel(const unsigned* __restrict__ key, long long n, unsigned* __restrict__ offs, int* __restrict__ perm)
{
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    perm[atomicAdd(offs + key[i], 1u)] = (int)i;
}

// bounding box of every tile of TP consecutive points of the sorted order, relative to the centre
// of source cell (0,0,0); the largest box diagonal goes to *diam2 (ordered bits, atomicMax)
template <typename T>
__global__ void __launch_bounds__(256)
list_tilebox_kernel(const T* __restrict__ pts, const int* __restrict__ perm, long long n, int TP, double sox, double soy,
                    double soz, double* __restrict__ boxes, unsigned long long* __restrict__ diam2)
{
    const long long t0 = (long long)blockIdx.x * TP;
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    const double so[3] = {sox, soy, soz};
    for (long long s = t0 + threadIdx.x; s < t0 + TP && s < n; s += 256)
        for (int a = 0; a < 3; ++a) {
            const double v = (double)pts[3 * (long long)perm[s] + a] - so[a];
            lo[a] = v < lo[a] ? v : lo[a]; hi[a] = v > hi[a] ? v : hi[a];
        }
    __shared__ double sl[8][3], sh[8][3];
    for (int a = 0; a < 3; ++a) {
        for (int o = 16; o; o >>= 1) {
            lo[a] = fmin(lo[a], __shfl_xor_sync(0xffffffffu, lo[a], o));
            hi[a] = fmax(hi[a], __shfl_xor_sync(0xffffffffu, hi[a], o));
        }
        if ((threadIdx.x & 31) == 0) { sl[threadIdx.x >> 5][a] = lo[a]; sh[threadIdx.x >> 5][a] = hi[a]; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double d2 = 0;
        for (int a = 0; a < 3; ++a) {
            double l = sl[0][a], h = sh[0][a];
            for (int w = 1; w < 8; ++w) { l = fmin(l, sl[w][a]); h = fmax(h, sh[w][a]); }
            boxes[6 * blockIdx.x + a] = l; boxes[6 * blockIdx.x + 3 + a] = h;
            d2 += (h - l) * (h - l);
        }
        atomicMax(diam2, ord(d2));
    }
}

// ------------------------------------------------------------------ the pairwise kernel
struct ListArgs {
    int nsx, nsy, nsz;
    double shx, shy, shz, sox, soy, soz;
    double rcut2, inv_cdt;
    int Tp, n1, origin;
    long long n_points, obs_count;            // the whole list is evaluated (obs_begin = 0)
    long long cells_per_chunk, Ns;
    int wcap_rt, chunk_base, accumulate, flush_stages;
    int wmax, stages, stage_bytes, cps;
    const void* points; const int* perm; const double* boxes;
    float tie_lim;                            // fp32: |q - k| >= tie_lim is "near a tie" (0.5 - tie_delta)
};

// fp32 near-tie pairs (tiled_common.cuh tie_delta): the few pairs whose q is within the fp32
// error of a half-integer take their lag from fp64 coordinate differences, as the contract's
// k = floor(q + 1/2) is defined (include/jefi.h).  The hot loop stays branch-free: it adds every
// pair with its fp32 lag and only MARKS the near-tie ones (three instructions and a predicated OR
// into a per-point bit mask, one bit per cell of the row segment); after the segment the marked
// pairs -- 4e-4 of all on the c3 geometry -- are revisited: fp64 lag (out of line, fed from seven
// doubles thread 0 parks in the unused bytes [160, 216) of the shared-memory map of
// tiled_step.cuh), and where it differs from the fp32 one (about one marked pair in four) the
// pair's terms are taken out again and added with the record of the right step.  (A branch
// around the pair inside the unrolled loop cost 48 % on c3_points: it stops the compiler from
// overlapping the gathers of neighbouring pairs.)
constexpr unsigned kOffTie = 160;
__device__ __noinline__ unsigned list_tie_bits(const double* tc, const float* p, int jx, int jy, int jz)
{
    const int k = near_tie_lag((double)p[0] - tc[0], (double)p[1] - tc[1], (double)p[2] - tc[2], jx, jy, jz, tc[3], tc[4],
                               tc[5], tc[6]);
    return Prec<float>::kMagicLo - (unsigned)k;
}
template <bool SLOW>
__device__ __forceinline__ void pair_update_mark(Acc<float>& a, float ox, float ryz, const CellMeta<float>& m,
                                                 float neg_inv_cdt, float rcut2, int n1, unsigned unit_off,
                                                 float neg_inv_plain, float tie_lim, unsigned& mask, unsigned bit)
{
    float dx, w, R;
    unsigned bits;
    pair_geo_r<float, SLOW>(ox, m.sx, ryz, neg_inv_cdt, rcut2, dx, w, bits, R);
    // bits = magic - k as a float pattern: e = k - q (without the tie bias), |e| <= 1/2
    const float e = fmaf(R, neg_inv_plain, 12582912.0f - __uint_as_float(bits));
    if (fabsf(e) >= tie_lim) mask |= bit;
    pair_accumulate<float>(a, dx, w, record_addr<float, SLOW>(m, bits, n1), unit_off);
}
// the marked pairs of one point over one row segment (cells jx0.. of row jy, jz; meta at meta_addr)
__device__ __forceinline__ void fix_marked_pairs(Acc<float>& a, unsigned mask, float ox, float ryz, unsigned meta_addr,
                                                 bool slow_stage, float neg_inv_cdt, float rcut2, int n1, unsigned unit_off,
                                                 const double* tc, const float* p, int jx0, int jy, int jz)
{
    while (mask) {
        const int c = __ffs(mask) - 1;
        mask &= mask - 1;
        const CellMeta<float> m = load_meta(meta_addr + c * 16u, 0.f);
        float dx, w, R;
        unsigned bits;
        pair_geo_r<float, true>(ox, m.sx, ryz, neg_inv_cdt, rcut2, dx, w, bits, R);     // as in the hot loop
        const unsigned good = list_tie_bits(tc, p, jx0 + c, jy, jz);
        if (good == bits || w == 0.f) continue;
        const unsigned was = slow_stage ? record_addr<float, true>(m, bits, n1) : record_addr<float, false>(m, bits, n1);
        const unsigned now = slow_stage ? record_addr<float, true>(m, good, n1) : record_addr<float, false>(m, good, n1);
        pair_accumulate<float, true>(a, dx, w, was, unit_off);
        pair_accumulate<float, false>(a, dx, w, now, unit_off);
    }
}

template <typename T, int WCAP, int CW, int CTAS>
__global__ void __launch_bounds__((CW + 1) * 32, CTAS)
fields_list_kernel(const uint4* __restrict__ hist, double* __restrict__ partial, const ListArgs a)
{
    constexpr int P = Prec<T>::P, U = Prec<T>::U, TP = P * CW * 32;
    const unsigned unit_off = WCAP > 0 ? (unsigned)WCAP * 16u : (unsigned)a.wcap_rt * 16u;
    extern __shared__ __align__(128) unsigned char smem[];
    const unsigned sbase = smem_u32(smem);
    const unsigned data0 = sbase + kOffMeta + (unsigned)a.stages * kStageCells * 16u;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int tile = blockIdx.x;
    const long long cb = (long long)(a.chunk_base + (int)blockIdx.y) * a.cells_per_chunk;
    const long long ce = (cb + a.cells_per_chunk < a.Ns) ? cb + a.cells_per_chunk : a.Ns;
    const int nst = (int)((ce - cb + a.cps - 1) / a.cps);

    if (tid == 0) {
        for (int s = 0; s < a.stages; ++s) {
            mbar_init(sbase + kOffFull + 8 * s, 32);
            mbar_init(sbase + kOffEmpty + 8 * s, CW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        double* tc = reinterpret_cast<double*>(smem + kOffTie);
        tc[0] = a.sox; tc[1] = a.soy; tc[2] = a.soz; tc[3] = a.shx; tc[4] = a.shy; tc[5] = a.shz; tc[6] = a.inv_cdt;
    }
    __syncthreads();

    if (warp == CW) {
        // ------------------------------------------------------------ producer warp (as in pairwise_tiled.cu,
        // the tile's box read from the table jefi_create built)
        const double* bx = a.boxes + 6 * (long long)tile;
        const double bx0 = bx[0], by0 = bx[1], bz0 = bx[2], bx1 = bx[3], by1 = bx[4], bz1 = bx[5];
        for (int it = 0; it < nst; ++it) {
            const int s = it % a.stages;
            if (it >= a.stages) mbar_wait_parked(sbase + kOffEmpty + 8 * s, ((it / a.stages) - 1) & 1);
            const long long j = cb + (long long)it * a.cps + lane;
            const bool valid = lane < a.cps && j < ce;
            bool slow = false;
            int p_src = 0, cnt = 0, nz = 0;
            unsigned row0 = 0;
            if (valid) {
                const int jx = (int)(j % a.nsx), jy = (int)((j / a.nsx) % a.nsy);
                const int jz = (int)(j / ((long long)a.nsx * a.nsy));
                int kmin, kmax;
                double dmin2;
                cell_lag_bounds(jx * a.shx, jy * a.shy, jz * a.shz, bx0, bx1, by0, by1, bz0, bz1, a.inv_cdt, kmin, kmax,
                                dmin2);
                const int p_lo = a.n1 - kmax;
                int span = kmax - kmin + 1;
                span = span > a.wmax ? a.wmax : span;
                slow = dmin2 <= a.rcut2 * 1.001;
                int p_hi = a.n1 - kmin;
                p_hi = p_hi > a.Tp - 1 ? a.Tp - 1 : p_hi;
                // slots for p <= 0 (the zero record and everything before it) are zero-filled here;
                // stored steps p >= 1 are copied from the ring
                nz = p_lo < 1 ? 1 - p_lo : 0;
                nz = nz > span ? span : nz;
                p_src = p_lo < 1 ? 1 : p_lo;
                cnt = p_hi >= p_src ? p_hi - p_src + 1 : 0;
                cnt = cnt > span - nz ? span - nz : cnt;
                row0 = data0 + (unsigned)s * (unsigned)a.stage_bytes + (unsigned)lane * (unsigned)U * unit_off;
                CellMeta<T> m;
                m.C = row0 + ((unsigned)(a.n1 - p_lo) << 4) - (Prec<T>::kMagicLo << 4);
                m.C2 = cnt > 0 ? row0 - ((unsigned)p_lo << 4) : row0;
                m.sx = src_coord<T>(jx, a.shx);
                *reinterpret_cast<CellMeta<T>*>(smem + kOffMeta + (s * kStageCells + lane) * 16) = m;
                for (int z = 0; z < nz; ++z) {
#pragma unroll
                    for (int u = 0; u < U; ++u) sts128_zero(row0 + u * unit_off + (unsigned)z * 16u);
                }
            }
            const bool any_slow = __any_sync(0xffffffffu, slow);
            if (lane == 0) *reinterpret_cast<int*>(smem + kOffFlags + 4 * s) = any_slow ? 1 : 0;
            const unsigned bar = sbase + kOffFull + 8 * s;
            if (valid && cnt > 0) {
                const unsigned bytes = (unsigned)cnt * 16u;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                mbar_arrive_expect_tx(bar, (unsigned)U * bytes);
                // the window is contiguous in p; in the ring it is one piece, or two when it wraps
                const int slot1 = ring_slot(p_src, a.origin, a.Tp - 1);
                const int len1 = cnt < a.Tp - slot1 ? cnt : a.Tp - slot1;
                const uint4* src = hist + ((size_t)j * U) * a.Tp;
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const unsigned dst = row0 + u * unit_off + (unsigned)nz * 16u;
                    bulk_g2s(dst, src + (size_t)u * a.Tp + slot1, (unsigned)len1 * 16u, bar);
                    if (len1 < cnt)
                        bulk_g2s(dst + (unsigned)len1 * 16u, src + (size_t)u * a.Tp + 1, (unsigned)(cnt - len1) * 16u, bar);
                }
            } else {
                mbar_arrive(bar);
            }
        }
        return;
    }

    // ---------------------------------------------------------------- consumer warps
    // point i of thread tid = entry tile*TP + i*(32 CW) + tid of the sorted order; entries past the
    // end of the list compute a copy of the last point and store nothing
    T ox[P], oy[P], oz[P];
    int gi[P];                                  // caller's index of the point (perm is int)
    unsigned okmask = 0;                        // bit i: entry i is a real point (stored at the end)
    Acc<T> acc[P];
    const T* pts = (const T*)a.points;
#pragma unroll
    for (int i = 0; i < P; ++i) {
        long long s = (long long)tile * TP + i * (CW * 32) + tid;
        const bool ok = s < a.n_points;
        s = ok ? s : a.n_points - 1;
        const int g = a.perm[s];
        gi[i] = g;
        okmask |= ok ? 1u << i : 0u;
        ox[i] = (T)((double)pts[3 * (long long)g + 0] - a.sox);
        oy[i] = (T)((double)pts[3 * (long long)g + 1] - a.soy);
        oz[i] = (T)((double)pts[3 * (long long)g + 2] - a.soz);
        acc[i] = Acc<T>{0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    }
    const T shy = (T)a.shy, shz = (T)a.shz, rcut2 = (T)a.rcut2;
    const T neg_inv_cdt = tie_biased_neg_inv_cdt<T>(a.inv_cdt);
    const float neg_inv_plain = (float)(-a.inv_cdt), tie_lim = a.tie_lim;
    unsigned tmask[P];                          // fp32: bit c = pair (point i, cell c of the row segment) is near a tie
#pragma unroll
    for (int i = 0; i < P; ++i) tmask[i] = 0;
    const double* tc = reinterpret_cast<const double*>(smem + kOffTie);
    int jx = (int)(cb % a.nsx), jy = (int)((cb / a.nsx) % a.nsy), jz = (int)(cb / ((long long)a.nsx * a.nsy));
    int since = 0;
    bool first = a.accumulate == 0;

    for (int it = 0; it < nst; ++it) {
        const int s = it % a.stages;
        mbar_wait(sbase + kOffFull + 8 * s, (it / a.stages) & 1);
        const long long j0 = cb + (long long)it * a.cps;
        const int cnt = (int)((ce - j0) < a.cps ? (ce - j0) : a.cps);
        const int slow = *reinterpret_cast<volatile int*>(smem + kOffFlags + 4 * s);
        int pos = 0;
        while (pos < cnt) {
            int len = a.nsx - jx;
            len = len < cnt - pos ? len : cnt - pos;
            T dy[P], dz[P], ryz[P];
#pragma unroll
            for (int i = 0; i < P; ++i) ryz[i] = row_ryz<T>(oy[i], oz[i], jy, jz, shy, shz, dy[i], dz[i]);
            const unsigned meta_addr = sbase + kOffMeta + (unsigned)(s * kStageCells + pos) * 16u;
            if (slow) {
#pragma unroll 2
                for (int c = 0; c < len; ++c) {
                    const CellMeta<T> m = load_meta(meta_addr + c * 16u, T(0));
#pragma unroll
                    for (int i = 0; i < P; ++i) {
                        if constexpr (sizeof(T) == 4)
                            pair_update_mark<true>(acc[i], ox[i], ryz[i], m, neg_inv_cdt, rcut2, a.n1, unit_off, neg_inv_plain,
                                                   tie_lim, tmask[i], 1u << c);
                        else
                            pair_update<T, true>(acc[i], ox[i], ryz[i], m, neg_inv_cdt, rcut2, a.n1, unit_off);
                    }
                }
            } else {
#pragma unroll 4
                for (int c = 0; c < len; ++c) {
                    const CellMeta<T> m = load_meta(meta_addr + c * 16u, T(0));
#pragma unroll
                    for (int i = 0; i < P; ++i) {
                        if constexpr (sizeof(T) == 4)
                            pair_update_mark<false>(acc[i], ox[i], ryz[i], m, neg_inv_cdt, rcut2, a.n1, unit_off, neg_inv_plain,
                                                    tie_lim, tmask[i], 1u << c);
                        else
                            pair_update<T, false>(acc[i], ox[i], ryz[i], m, neg_inv_cdt, rcut2, a.n1, unit_off);
                    }
                }
            }
            if constexpr (sizeof(T) == 4) {
                unsigned any = 0;
#pragma unroll
                for (int i = 0; i < P; ++i) any |= tmask[i];
                if (any) {
#pragma unroll
                    for (int i = 0; i < P; ++i) {
                        fix_marked_pairs(acc[i], tmask[i], ox[i], ryz[i], meta_addr, slow != 0, neg_inv_cdt, rcut2, a.n1,
                                         unit_off, tc, (const float*)pts + 3 * (long long)gi[i], jx, jy, jz);
                        tmask[i] = 0;
                    }
                }
            }
            pos += len; jx += len;
            const bool row_done = jx == a.nsx;
            if (row_done || (it == nst - 1 && pos == cnt)) {
#pragma unroll
                for (int i = 0; i < P; ++i) fold_row<T>(acc[i], dy[i], dz[i]);
            }
            if (row_done) { jx = 0; if (++jy == a.nsy) { jy = 0; ++jz; } }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(sbase + kOffEmpty + 8 * s);

        if (++since == a.flush_stages || it == nst - 1) {
            since = 0;
#pragma unroll
            for (int i = 0; i < P; ++i) {
                if (okmask >> i & 1u) {
                    double* out = partial + (long long)blockIdx.y * 6 * a.obs_count + gi[i];
                    const T v[6] = {acc[i].ex, acc[i].ey, acc[i].ez, acc[i].bx, acc[i].by, acc[i].bz};
#pragma unroll
                    for (int c = 0; c < 6; ++c) {
                        double* q = out + (long long)c * a.obs_count;
                        *q = first ? (double)v[c] : *q + (double)v[c];
                    }
                }
                acc[i].ex = acc[i].ey = acc[i].ez = acc[i].bx = acc[i].by = acc[i].bz = T(0);
            }
            first = false;
        }
    }
}

template <typename T, int WCAP, int CW, int CTAS>
int launch_list_cap(const Params& P, jefi_dtype dt, const void* hist, const FieldsLaunch& L, const PointTiles& pt)
{
    constexpr int U = Prec<T>::U;
    constexpr int kThreads = (CW + 1) * 32;
    ListArgs a;
    a.nsx = P.ns[0]; a.nsy = P.ns[1]; a.nsz = P.ns[2];
    a.shx = P.sh[0]; a.shy = P.sh[1]; a.shz = P.sh[2];
    a.sox = P.so[0]; a.soy = P.so[1]; a.soz = P.so[2];
    double hmin = P.sh[0] < P.sh[1] ? P.sh[0] : P.sh[1];
    hmin = hmin < P.sh[2] ? hmin : P.sh[2];
    a.rcut2 = 0.25 * hmin * hmin;
    a.inv_cdt = 1.0 / (P.c * P.dt);
    a.Tp = P.Tp; a.n1 = L.step + 1; a.origin = P.origin;
    a.n_points = P.n_obs; a.obs_count = L.obs_count;
    a.Ns = P.Ns;
    a.points = P.obs_points; a.perm = pt.perm; a.boxes = pt.boxes;

    const double wd = floor(pt.max_diam * a.inv_cdt) + 5.0;
    if (wd > 1.0e6 || pt.far * a.inv_cdt > kMaxLagSteps) return 0;
    a.wmax = (int)wd;
    a.tie_lim = 0.5f - tie_delta(pt.far * a.inv_cdt);
    if (WCAP > 0 && a.wmax > WCAP) return 0;
    const int wcap = WCAP > 0 ? WCAP : (a.wmax + 7) / 8 * 8;
    a.wcap_rt = wcap;
    const int cell_bytes = U * wcap * 16;
    const int budget3 = 227 * 1024 / CTAS - 2048, budget1 = 226 * 1024;
    int cps = 0, stages = 0;
    for (int c = 32; c >= 4 && !cps; c -= 4) {
        const int st = (budget3 - (int)kOffMeta) / (c * cell_bytes + 512);
        if (st >= 2) { cps = c; stages = st > 4 ? 4 : st; }
    }
    for (int c = 4; c >= 1 && !cps; c >>= 1) {
        const int st = (budget1 - (int)kOffMeta) / (c * cell_bytes + 512);
        if (st >= 2) { cps = c; stages = st > 4 ? 4 : st; }
    }
    if (!cps) return 0;
    a.flush_stages = sizeof(T) == 4 ? 2048 / cps : (1 << 30);
    a.cps = cps; a.stages = stages; a.stage_bytes = cps * cell_bytes;
    const int smem = (int)kOffMeta + stages * 512 + stages * a.stage_bytes;

    auto kern = fields_list_kernel<T, WCAP, CW, CTAS>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return -1;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kThreads, smem) != cudaSuccess) return -1;
    if (per_sm < 1) return 0;

    // source chunks: as in pairwise_tiled.cu (waves, L2 sharing, scratch)
    const long long ntiles = pt.ntiles;
    const long long slots = (long long)L.sm_count * per_sm;
    long long smax = P.Ns / ((long long)cps * 2);
    if (smax > 65535) smax = 65535;
    if (smax < 1) smax = 1;
    long long s_launch = L.scratch_elems / (6 * L.obs_count);
    if (s_launch < 1) s_launch = 1;
    long long s0 = (4 * slots + ntiles - 1) / ntiles;
    if (s0 > s_launch) s0 = s_launch;
    long long s_hi = 4 * s0 < s_launch ? 4 * s0 : s_launch;
    if (P.Ns < s0 * cps * 8) {
        s0 = slots / ntiles;
        if (s0 < 1) s0 = 1;
        if (s0 > s_launch) s0 = s_launch;
        s_hi = s0;
    }
    const double cell_hist_bytes = (double)U * (double)P.Tp * 16.0;
    const long long s_l2 = (long long)ceil((double)P.Ns * cell_hist_bytes / (double)L.chunk_bytes);
    if (s0 < s_l2) { s0 = s_l2; s_hi = 4 * s_l2; }
    if (s0 > smax) s0 = smax;
    if (s_hi > smax) s_hi = smax;
    long long S = s0;
    double best = -1.0;
    for (long long s = s0; s <= s_hi; ++s) {
        const double waves = (double)(ntiles * s) / (double)slots;
        const double eff = waves / ceil(waves);
        if (eff > best + 1e-9) { best = eff; S = s; }
    }
    a.cells_per_chunk = (P.Ns + S - 1) / S;
    a.cells_per_chunk = (a.cells_per_chunk + cps - 1) / cps * cps;
    S = (P.Ns + a.cells_per_chunk - 1) / a.cells_per_chunk;
    if (s_launch > S) s_launch = S;

    int launches = 0;
    for (long long base = 0; base < S; base += s_launch) {
        const long long sl = S - base < s_launch ? S - base : s_launch;
        a.chunk_base = (int)base;
        a.accumulate = base > 0 ? 1 : 0;
        dim3 grid((unsigned)ntiles, (unsigned)sl);
        kern<<<grid, kThreads, smem, L.stream>>>((const uint4*)hist, (double*)L.scratch, a);
        if (cudaPeekAtLastError() != cudaSuccess) return -1;
        ++launches;
    }
    if (launch_reduce_scale(P, dt, L, (int)s_launch) < 0) return -1;
    return launches + 1;
}

template <typename T>
int launch_list_T(const Params& P, jefi_dtype dt, const void* hist, const FieldsLaunch& L, const PointTiles& pt)
{
    int n = launch_list_cap<T, 32, 4, 3>(P, dt, hist, L, pt);
    if (n == 0) n = launch_list_cap<T, 64, 4, 3>(P, dt, hist, L, pt);
    if (n == 0) n = launch_list_cap<T, 96, 4, 3>(P, dt, hist, L, pt);
    if (n == 0) n = launch_list_cap<T, 0, 4, 3>(P, dt, hist, L, pt);
    return n;
}

template <typename T>
int build_tiles_T(const Params& P, PointTiles& pt, unsigned* key, unsigned* hist, unsigned long long* mm)
{
    const long long n = P.n_obs;
    const T* pts = (const T*)P.obs_points;
    unsigned long long init[7] = {~0ull, ~0ull, ~0ull, 0ull, 0ull, 0ull, 0ull};
    if (cudaMemcpy(mm, init, sizeof(init), cudaMemcpyHostToDevice) != cudaSuccess) return -1;
    const unsigned gb = (unsigned)((n + 255) / 256 < 1184 ? (n + 255) / 256 : 1184);
    list_bbox_kernel<T><<<gb, 256>>>(pts, n, mm);
    unsigned long long h[7];
    if (cudaMemcpy(h, mm, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    // bins: the full 64 per axis of the 18-bit curve keys, whatever n -- the finer the sort, the
    // closer the 8 points of a quarter-warp and the fewer bank conflicts among their slots
    // (no measurable difference between 32 and 64 on 65 536 random points: at that density the
    // 8 points already spread over more than 8 lag steps)
    const int nb = 64;
    BinArgs b;
    b.nb = nb;
    double far2 = 0;
    for (int a = 0; a < 3; ++a) {
        const double lo = unord(h[a]), hi = unord(h[3 + a]);
        if (!(lo <= hi) || !isfinite(lo) || !isfinite(hi)) return -2;            // NaN / Inf positions
        b.lo[a] = lo;
        b.inv[a] = hi > lo ? nb / (hi - lo) : 0.0;
        const double e0 = fabs(lo - P.so[a]), e1 = fabs(hi - P.so[a]);
        const double ext = (e0 > e1 ? e0 : e1) + P.ns[a] * P.sh[a];
        far2 += ext * ext;
    }
    pt.far = sqrt(far2);
    const int nbins = 1 << 18;
    if (cudaMemset(hist, 0, nbins * sizeof(unsigned)) != cudaSuccess) return -1;
    const unsigned g = (unsigned)((n + 255) / 256);
    list_key_kernel<T><<<g, 256>>>(pts, n, b, key, hist);
    list_scan_kernel<<<1, 1024>>>(hist, nbins);
    list_scatter_kernel<<<g, 256>>>(key, n, hist, pt.perm);
    list_tilebox_kernel<T><<<(unsigned)pt.ntiles, 256>>>(pts, pt.perm, n, pt.tile_points, P.so[0], P.so[1], P.so[2],
                                                         pt.boxes, mm + 6);
    if (cudaMemcpy(h, mm, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
    if (cudaGetLastError() != cudaSuccess) return -1;
    pt.max_diam = sqrt(unord(h[6]));
    return 5;
}

}  // namespace

int list_tile_points(jefi_dtype dt) { return dt == JEFI_F32 ? Prec<float>::P * 128 : Prec<double>::P * 128; }

// jefi_create, kind 1: permutation + tile boxes (synchronous; default stream).  Scratch for the
// keys, the bin histogram and the min/max words is allocated and freed here.
int build_point_tiles(const Params& P, jefi_dtype dt, PointTiles& pt)
{
    unsigned *key = nullptr, *hist = nullptr;
    unsigned long long* mm = nullptr;
    int rc = -1;
    if (cudaMalloc(&key, (size_t)P.n_obs * sizeof(unsigned)) == cudaSuccess &&
        cudaMalloc(&hist, (size_t)(1 << 18) * sizeof(unsigned)) == cudaSuccess &&
        cudaMalloc(&mm, 7 * sizeof(unsigned long long)) == cudaSuccess)
        rc = dt == JEFI_F32 ? build_tiles_T<float>(P, pt, key, hist, mm) : build_tiles_T<double>(P, pt, key, hist, mm);
    cudaFree(key); cudaFree(hist); cudaFree(mm);
    return rc;
}

int launch_fields_list(const Params& P, jefi_dtype dt, const void* hist, const FieldsLaunch& L, const PointTiles& pt)
{
    if (P.obs_kind != 1 || !pt.perm || L.obs_begin != 0 || L.obs_count != P.n_obs) return 0;
    return dt == JEFI_F32 ? launch_list_T<float>(P, dt, hist, L, pt) : launch_list_T<double>(P, dt, hist, L, pt);
}

}  // namespace jefi
