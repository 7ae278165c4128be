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
// (one atomicAdd per group of substeps of a resolve block);
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

}  // namespace evis
