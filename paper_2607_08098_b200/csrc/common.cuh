// common.cuh -- device helpers shared by the EVIS kernels (sm_100a).
//
// Arithmetic contract: everything that decides an integer is IEEE binary32
// with an explicit operation order (__fmaf_rn / __fmul_rn / __fadd_rn / __fsub_rn / __fdiv_rn), so
// the compiler cannot contract or reassociate.  No fast-math anywhere in this library.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/evis.h"

namespace evis {

constexpr unsigned long long KEY_EMPTY = 0xFFFFFFFFFFFFFFFFull;
constexpr unsigned long long KEY_DIR_A = 0x8000000000000000ull;   // direction bit: B = 0 < A = 1
constexpr uint32_t           IDX_NONE  = 0xFFFFFFFFu;

// Per-substep time weights f_i = (float)i / (float)S and g_i = 1 - f_i (Eq. 5),
// computed on the host with IEEE binary32 division and subtraction, index i in 0..S.
struct SubstepTable {
    float f[256];
    float g[256];
};

struct EventParams {
    float c_pos, c_neg;   // C+, C-            (Eq. 4, R4)
    float dt;             // T / S  (binary32 division on the host)
    uint32_t kf;          // interval index of this step
};

// Where the compacted stream goes (a8).  Space in the arrival buffer is handed out by `alloc`
// (one atomicAdd per chunk on the global path, one per SLAB of events on the persistent tile path);
// `counter` accumulates the true number of events.  directory[d] = (arrival offset, count) of chunk d;
// order.cu lays the chunks out in d order.
struct EventSink {
    uint4 *arrival;                 // [arrival_cap] events in arrival order
    unsigned long long arrival_cap; // < 2^32
    unsigned long long *alloc;      // next free arrival slot
    unsigned long long *counter;    // total events of this step
    uint2 *directory;               // [num_entries] (arrival offset, count)
};

__device__ __forceinline__ unsigned long long umin64(unsigned long long a, unsigned long long b)
{
    return a < b ? a : b;
}

// ---- Eq. 5-7: one source offered to the z-buffer at one substep ---------------------------------
// q = p + w * disp (Eq. 5);  zt = f * zb + g * za (Eq. 7, g*za rounded first);  footprint = the
// integer pixels with positive bilinear weight (R14).  Returns false when the source is skipped
// (invalid depth R17, off-image R18).  cls: bit0 = positive weight on x0+1, bit1 = on y0+1.
struct Landing {
    int x0, y0;
    int cls;
    unsigned long long key;    // [dir:1 | zt bits:31 | source index:32]  (R15)
};

__device__ __forceinline__ bool land(float x, float y, float dx, float dy, float w, float f, float g,
                                     float za, float zb, uint32_t src, unsigned long long dirbit,
                                     int W, int H, Landing &o)
{
    const float qx = __fmaf_rn(w, dx, x);
    const float qy = __fmaf_rn(w, dy, y);
    const float zt = __fmaf_rn(f, zb, __fmul_rn(g, za));
    const uint32_t zbits = __float_as_uint(zt);
    // valid depth: 0 < zt < +inf  <=>  0 < bits < 0x7f800000 (sign bit clear)
    if (zbits - 1u >= 0x7f7fffffu) return false;
    const float x0f = floorf(qx), y0f = floorf(qy);
    if (!(x0f >= -1.0f && x0f <= (float)(W - 1) && y0f >= -1.0f && y0f <= (float)(H - 1))) return false;
    o.x0 = (int)x0f;
    o.y0 = (int)y0f;
    o.cls = (qx > x0f ? 1 : 0) | (qy > y0f ? 2 : 0);
    o.key = dirbit | ((unsigned long long)zbits << 32) | src;
    return true;
}

// Depth of the far endpoint of the correspondence (Eq. 7, R16): nearest pixel of the other
// keyframe, or the source's own depth when it falls outside the image.
__device__ __forceinline__ float far_depth(const float *__restrict__ z_other, float x, float y, float dx,
                                           float dy, float z_own, int W, int H)
{
    const float jx = floorf(__fadd_rn(__fadd_rn(x, dx), 0.5f));
    const float jy = floorf(__fadd_rn(__fadd_rn(y, dy), 0.5f));
    if (jx >= 0.0f && jx <= (float)(W - 1) && jy >= 0.0f && jy <= (float)(H - 1))
        return __ldg(z_other + (int)jy * W + (int)jx);
    return z_own;
}

// ---- Eq. 4: number of threshold crossings of one pixel at one substep ---------
// n = floor(|dL| / C), capped at 255 (R7).  |dL| < C  <=>  the correctly rounded quotient is < 1,
// so the division is skipped for the common silent pixel.
__device__ __forceinline__ int event_count(float l_hat, float l_ref, float c_pos, float c_neg, int &pol,
                                           float &c)
{
    const float d = __fsub_rn(l_hat, l_ref);
    if (d > 0.0f)      { c = c_pos; pol = +1; }
    else if (d < 0.0f) { c = c_neg; pol = -1; }
    else               { c = 1.0f; pol = 0; return 0; }
    const float ad = fabsf(d);
    if (ad < c) return 0;
    const float r = floorf(__fdiv_rn(ad, c));
    return r >= 255.0f ? 255 : (int)r;
}

// Timestamp of the k-th crossing (R8): linear in log intensity between L_prev and L_hat.
__device__ __forceinline__ float event_time(int k, int pol, float c, float l_ref, float l_prev, float l_hat,
                                            int substep, float dt)
{
    const float lev = __fmaf_rn((float)(pol * k), c, l_ref);
    const float den = __fsub_rn(l_hat, l_prev);
    // timestamps decide nothing (compared within 1e-7 s; the step is ~1e-3 s): approximate division
    // (2 ulp) unless the denominator is so small that the fast reciprocal would overflow
    float fr = 1.0f;
    if (fabsf(den) > 1e-30f) fr = __fdividef(__fsub_rn(lev, l_prev), den);
    else if (den != 0.0f) fr = __fdiv_rn(__fsub_rn(lev, l_prev), den);
    fr = fminf(fmaxf(fr, 0.0f), 1.0f);          // NaN -> 0 like the oracle's !(fr >= 0)
    return __fmaf_rn(fr, dt, __fmul_rn((float)(substep - 1), dt));
}

// ---- a8: compaction ------------------------------------------------------------------------------
// 16-byte event record from the crossing index k of one pixel-substep.
__device__ __forceinline__ uint4 make_event(int k, int pol, float c, float l_ref, float l_prev, float l_hat,
                                            uint32_t xy, int env, int substep, const EventParams &ep)
{
    uint4 r;
    r.x = xy;
    r.y = (uint32_t)env | (((uint32_t)pol & 0xFFu) << 16) | ((uint32_t)substep << 24);
    r.z = __float_as_uint(event_time(k, pol, c, l_ref, l_prev, l_hat, substep, ep.dt));
    r.w = ep.kf;
    return r;
}

// Warp-cooperative emission.  Every lane of a converged warp calls this with the n >= 0 crossings of
// ITS pixel at this substep; the warp's events go to arrival[off ...] in (lane, k) order and the
// number written is returned (warp-uniform).  n <= 1 everywhere: ballot/popc ranks, each firing lane
// stores its own record.  Otherwise: shuffle scan of n, then the lanes take the warp's events 32 at a
// time -- lane e finds its owner by a 5-step search over the scan and fetches the owner's values by
// shuffle -- so a pixel with many crossings costs the warp one pass, not n divergent ones.
__device__ __forceinline__ int warp_emit(const EventSink &sink, unsigned long long off, int n, int pol, float c,
                                         float l_ref, float l_prev, float l_hat, uint32_t xy, int env, int substep,
                                         const EventParams &ep)
{
    constexpr unsigned FULL = 0xFFFFFFFFu;
    const unsigned fire = __ballot_sync(FULL, n > 0);
    if (!fire) return 0;
    const int lane = threadIdx.x & 31;
    if (!__ballot_sync(FULL, n > 1)) {
        const unsigned long long o = off + __popc(fire & ((1u << lane) - 1u));
        if (n && o < sink.arrival_cap) sink.arrival[o] = make_event(1, pol, c, l_ref, l_prev, l_hat, xy, env, substep, ep);
        return __popc(fire);
    }
    int incl = n;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(FULL, incl, d);
        if (lane >= d) incl += v;
    }
    const int excl = incl - n, total = __shfl_sync(FULL, incl, 31);
    const float cs = pol < 0 ? -c : c;                      // polarity rides on the sign of the threshold
    for (int base = 0; base < total; base += 32) {
        const int e = base + lane;
        int s = 0;                                          // owner: the last lane whose first event is <= e
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) {
            const int t = __shfl_sync(FULL, excl, s + d);
            if (t <= e) s += d;
        }
        const int k = e - __shfl_sync(FULL, excl, s) + 1;
        const float ocs = __shfl_sync(FULL, cs, s), oref = __shfl_sync(FULL, l_ref, s);
        const float oprev = __shfl_sync(FULL, l_prev, s), ohat = __shfl_sync(FULL, l_hat, s);
        const uint32_t oxy = __shfl_sync(FULL, xy, s);
        const unsigned long long o = off + e;
        if (e < total && o < sink.arrival_cap)
            sink.arrival[o] = make_event(k, ocs < 0.0f ? -1 : +1, fabsf(ocs), oref, oprev, ohat, oxy, env, substep, ep);
    }
    return total;
}

// Exclusive prefix of this warp among the per-warp event totals s_tot[0..NW) of a block, and the block
// total.  Every warp computes both from the same array, so no second barrier is needed.
template <int NW>
__device__ __forceinline__ uint32_t warp_prefix(const volatile uint32_t *s_tot, uint32_t &block_total)
{
    static_assert(NW <= 32, "one lane per warp");
    constexpr unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t v = lane < NW ? s_tot[lane] : 0u;
    uint32_t incl = v;
#pragma unroll
    for (int d = 1; d < NW; d <<= 1) {
        const uint32_t u = __shfl_up_sync(FULL, incl, d);
        if (lane >= d) incl += u;
    }
    block_total = __shfl_sync(FULL, incl, NW - 1);
    return __shfl_sync(FULL, incl - v, warp);
}

}  // namespace evis
