// tiled_step.cuh -- the one-step record arithmetic shared by the tiled kernel for regular
// observation grids (pairwise_tiled.cu) and the one for explicit point lists (pairwise_list.cu):
// the per-cell meta record the producer writes, the 12 running sums of a point, the per-pair update
// (Eq. (4)-(6), pre-scaled variables) and the per-row fold.  Internal to libjefi.so.
#pragma once
#include "tiled_common.cuh"

namespace jefi {

constexpr int kStageCells = 32;       // meta slots per stage; a stage holds a.cps <= 32 cells (one producer lane each)
// shared-memory map (dynamic): [0,64) full barriers, [64,128) empty barriers, [128,160) stage
// flags, [256, 256 + stages*512) cell meta, then stages * stage_bytes of history windows
constexpr unsigned kOffFull = 0, kOffEmpty = 64, kOffFlags = 128, kOffMeta = 256;

// per-cell record written by the producer, read (broadcast) by every consumer thread
template <typename T> struct CellMeta;
template <> struct alignas(16) CellMeta<float> {
    unsigned C;        // fast path: slot address = C + (lag_bits << 4)
    float    sx;       // cell centre x relative to source cell (0,0,0)
    unsigned C2;       // slow path: slot address = C2 + (p << 4), p = max(n1 - k, 0)
    unsigned pad;
};
template <> struct alignas(16) CellMeta<double> {
    unsigned C, C2;
    double   sx;
};
__device__ __forceinline__ CellMeta<float> load_meta(unsigned addr, float)
{
    const float4 mv = lds128(addr);
    CellMeta<float> m;
    m.C = __float_as_uint(mv.x); m.sx = mv.y; m.C2 = __float_as_uint(mv.z); m.pad = 0;
    return m;
}
__device__ __forceinline__ CellMeta<double> load_meta(unsigned addr, double)
{
    const double2 mv = lds128d(addr);
    CellMeta<double> m;
    m.C = (unsigned)__double2loint(mv.x); m.C2 = (unsigned)__double2hiint(mv.x); m.sx = mv.y;
    return m;
}

template <typename T> struct Acc {
    T ex, ey, ez, bx, by, bz;     // running sums over the chunk
    T s, ux, uy, uz, vy, vz;      // per source row
};

// shared-memory address of the record a pair reads: fast path straight from the lag bits, slow
// path (stages that may hold p <= 0 or screened pairs) through the clamped packed step
template <typename T, bool SLOW>
__device__ __forceinline__ unsigned record_addr(const CellMeta<T>& m, unsigned bits, int n1)
{
    if (SLOW) {
        int p = n1 - lag_of_bits(bits, Prec<T>::kMagicLo);
        p = p < 0 ? 0 : p;
        return m.C2 + ((unsigned)p << 4);
    }
    return m.C + (bits << 4);
}
// gather the record and add the pair's terms to the running sums (NEG: take them out again --
// every term is a product with g, h or w, so negating those three negates the pair)
template <typename T, bool NEG = false>
__device__ __forceinline__ void pair_accumulate(Acc<T>& a, T dx, T w, unsigned addr, unsigned unit_off)
{
    T v[8];
    load_record(addr, unit_off, v);
    T g = w * w;
    T h = dx * g;
    const T ts = fma_t<T>(v[0], w, v[1]);
    const T tx = fma_t<T>(v[2], w, v[5]);
    const T ty = fma_t<T>(v[3], w, v[6]);
    const T tz = fma_t<T>(v[4], w, v[7]);
    if (NEG) { g = -g; h = -h; w = -w; }
    a.ex = fma_t<T>(ts, h, a.ex);
    a.s  = fma_t<T>(ts, g, a.s);
    a.ex = fma_t<T>(-v[5], w, a.ex);
    a.ey = fma_t<T>(-v[6], w, a.ey);
    a.ez = fma_t<T>(-v[7], w, a.ez);
    a.ux = fma_t<T>(tx, g, a.ux);
    a.uy = fma_t<T>(ty, g, a.uy);
    a.uz = fma_t<T>(tz, g, a.uz);
    a.vy = fma_t<T>(ty, h, a.vy);
    a.vz = fma_t<T>(tz, h, a.vz);
}

template <typename T, bool SLOW>
__device__ __forceinline__ void pair_update(Acc<T>& a, T ox, T ryz, const CellMeta<T>& m, T neg_inv_cdt, T rcut2, int n1,
                                            unsigned unit_off)
{
    T dx, w;
    unsigned bits;
    pair_geo<T, SLOW>(ox, m.sx, ryz, neg_inv_cdt, rcut2, dx, w, bits);
    pair_accumulate<T>(a, dx, w, record_addr<T, SLOW>(m, bits, n1), unit_off);
}

template <typename T>
__device__ __forceinline__ void fold_row(Acc<T>& a, T dy, T dz)
{
    a.ey = fma_t<T>(dy, a.s, a.ey);
    a.ez = fma_t<T>(dz, a.s, a.ez);
    a.bx += a.uy * dz - a.uz * dy;
    a.by += a.vz - a.ux * dz;
    a.bz += a.ux * dy - a.vy;
    a.s = a.ux = a.uy = a.uz = a.vy = a.vz = T(0);
}


}  // namespace jefi
