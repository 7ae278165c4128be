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

// Where the compacted stream goes (a8).
struct EventSink {
    uint4 *arrival;                 // [capacity] events in arrival order
    unsigned long long capacity;
    unsigned long long *counter;    // total events of this step
    uint2 *directory;               // [num_entries] (arrival offset, count); capacity < 2^32; see order.cu
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

// 16-byte event record, layout of evis_event.
__device__ __forceinline__ uint4 pack_event(int x, int y, int env, int pol, int substep, float t_off,
                                            uint32_t kf)
{
    uint4 r;
    r.x = (uint32_t)x | ((uint32_t)y << 16);
    r.y = (uint32_t)env | (((uint32_t)pol & 0xFFu) << 16) | ((uint32_t)substep << 24);
    r.z = __float_as_uint(t_off);
    r.w = kf;
    return r;
}

// Timestamp of the k-th crossing (R8): linear in log intensity between L_prev and L_hat.
__device__ __forceinline__ float event_time(int k, int pol, float c, float l_ref, float l_prev, float l_hat,
                                            int substep, float dt)
{
    const float lev = __fmaf_rn((float)(pol * k), c, l_ref);
    const float den = __fsub_rn(l_hat, l_prev);
    float fr = 1.0f;
    if (den != 0.0f) fr = __fdiv_rn(__fsub_rn(lev, l_prev), den);
    fr = fminf(fmaxf(fr, 0.0f), 1.0f);          // NaN -> 0 like the oracle's !(fr >= 0)
    return __fmaf_rn(fr, dt, __fmul_rn((float)(substep - 1), dt));
}

// ---- a8: block-level compaction ------------------------------------------------------------------
// Every thread of the block calls this once per (tile, substep) with its number of events n.
// Warp shuffle scan -> block scan over warp totals -> ONE global atomic per block -> each thread
// gets the arrival offset of its first event.  The (offset, count) of the block's chunk goes to
// directory[dir_index]; order.cu later lays the chunks out in directory order, which makes the
// stream deterministic although the atomics arrive in any order.
// Returns the global arrival offset of this thread's first event; `any` tells whether the block
// emitted anything (uniform across the block).  NT = threads per block (multiple of 32, <= 1024).
template <int NT>
__device__ __forceinline__ unsigned long long block_reserve(int n, const EventSink &sink, uint32_t dir_index,
                                                            uint32_t *s_warp /* [NT/32 + 2] */, bool &any)
{
    constexpr int NW = NT / 32;
    any = __syncthreads_or(n > 0) != 0;
    if (!any) return 0;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int incl = n;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(0xFFFFFFFFu, incl, d);
        if (lane >= d) incl += v;
    }
    if (lane == 31) s_warp[warp] = (uint32_t)incl;
    __syncthreads();
    __shared__ unsigned long long s_base;
    if (warp == 0) {
        uint32_t w = lane < NW ? s_warp[lane] : 0u;
        uint32_t wi = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, wi, d);
            if (lane >= d) wi += v;
        }
        if (lane < NW) s_warp[lane] = wi - w;             // exclusive warp offsets
        if (lane == 31) {
            const unsigned long long base = atomicAdd(sink.counter, (unsigned long long)wi);
            s_base = base;
            // chunks that start beyond 2^32 lie beyond any capacity: mark them unreachable
            sink.directory[dir_index] = make_uint2(base < 0xFFFFFFFFull ? (uint32_t)base : 0xFFFFFFFFu, wi);
        }
    }
    __syncthreads();
    return s_base + s_warp[warp] + (uint32_t)(incl - n);
}

__device__ __forceinline__ void write_events(const EventSink &sink, unsigned long long off, int n, int pol,
                                             float c, float l_ref, float l_prev, float l_hat, int x, int y,
                                             int env, int substep, const EventParams &ep)
{
    for (int k = 1; k <= n; ++k, ++off) {
        if (off < sink.capacity)
            sink.arrival[off] = pack_event(x, y, env, pol, substep,
                                           event_time(k, pol, c, l_ref, l_prev, l_hat, substep, ep.dt), ep.kf);
    }
}

}  // namespace evis
