// order.cu -- row a8, second half: deterministic ordering of the compacted event stream.
//
// The compaction kernels reserve space with one global atomic per (tile, substep) chunk, so chunks
// land in the arrival buffer in scheduling order.  Each chunk left (arrival offset, count) in
// directory[d], d = ((env * S + substep-1) * tiles_y + tile_y) * tiles_x + tile_x.  Here the chunks
// are laid out in directory order: exclusive scan of the counts (three small kernels) and a
// chunk-by-chunk 128-bit copy.  Inside a chunk the order is the block scan order of the producer
// (pixel rank in the tile, then crossing index k), which is deterministic as well.
#include "kernels.h"

namespace evis {

constexpr int ORD_NT = 256, ORD_PER_THREAD = 2, ORD_PER_BLOCK = ORD_NT * ORD_PER_THREAD;
static_assert(ORD_PER_BLOCK == ORDER_ENTRIES_PER_BLOCK, "api.cu sizes the block-sum array with this");

__device__ __forceinline__ unsigned long long block_scan_excl(unsigned long long v, unsigned long long *s_w,
                                                              unsigned long long &total)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned long long incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned long long u = __shfl_up_sync(0xFFFFFFFFu, incl, d);
        if (lane >= d) incl += u;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        const int nw = blockDim.x >> 5;
        unsigned long long w = lane < nw ? s_w[lane] : 0ull, wi = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned long long u = __shfl_up_sync(0xFFFFFFFFu, wi, d);
            if (lane >= d) wi += u;
        }
        if (lane < nw) s_w[lane] = wi - w;
        if (lane == 31) s_w[32] = wi;
    }
    __syncthreads();
    total = s_w[32];
    const unsigned long long r = s_w[warp] + incl - v;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(ORD_NT)
k_dir_blocksum(const uint2 *__restrict__ dir, uint32_t n, unsigned long long *__restrict__ bsum)
{
    __shared__ unsigned long long s_w[33];
    const uint32_t base = blockIdx.x * ORD_PER_BLOCK + threadIdx.x * ORD_PER_THREAD;
    unsigned long long v = 0;
#pragma unroll
    for (int j = 0; j < ORD_PER_THREAD; ++j)
        if (base + j < n) v += dir[base + j].y;
    unsigned long long total;
    block_scan_excl(v, s_w, total);
    if (threadIdx.x == 0) bsum[blockIdx.x] = total;
}

// single block: exclusive scan of the per-block sums in place
__global__ void __launch_bounds__(1024)
k_dir_scan_bsum(unsigned long long *__restrict__ bsum, uint32_t nb, const unsigned long long *__restrict__ step_events,
                unsigned long long *__restrict__ total_events)
{
    if (threadIdx.x == 0) *total_events += *step_events;
    __shared__ unsigned long long s_w[33];
    const uint32_t per = (nb + blockDim.x - 1) / blockDim.x;
    const uint32_t lo = threadIdx.x * per, hi = min(lo + per, nb);
    unsigned long long v = 0;
    for (uint32_t j = lo; j < hi; ++j) v += bsum[j];
    unsigned long long total;
    unsigned long long run = block_scan_excl(v, s_w, total);
    for (uint32_t j = lo; j < hi; ++j) { const unsigned long long c = bsum[j]; bsum[j] = run; run += c; }
}

// Balanced copy: the block's chunks form one contiguous output range of `total` events; the threads
// stride over that range (coalesced 16-byte loads and stores) and walk the chunk table forward, so
// a block's time depends on its event count, not on how the events are split into chunks.
__global__ void __launch_bounds__(ORD_NT)
k_dir_copy(const uint2 *__restrict__ dir, uint32_t n, const unsigned long long *__restrict__ bsum,
           const uint4 *__restrict__ arrival, unsigned long long arrival_cap, uint4 *__restrict__ ordered,
           unsigned long long cap)
{
    __shared__ unsigned long long s_w[33];
    __shared__ uint32_t s_rel[ORD_PER_BLOCK + 1];     // first output position of chunk e, relative to the block
    __shared__ uint32_t s_src[ORD_PER_BLOCK];         // its arrival offset
    const uint32_t blk = blockIdx.x * ORD_PER_BLOCK;
    const uint32_t base = blk + threadIdx.x * ORD_PER_THREAD;
    uint32_t cnt[ORD_PER_THREAD];
    unsigned long long v = 0;
#pragma unroll
    for (int j = 0; j < ORD_PER_THREAD; ++j) {
        uint2 d = make_uint2(0u, 0u);
        if (base + j < n) d = dir[base + j];
        cnt[j] = d.y;
        v += d.y;
        s_src[threadIdx.x * ORD_PER_THREAD + j] = d.x;
    }
    unsigned long long total;
    unsigned long long run = block_scan_excl(v, s_w, total);
    if (total == 0) return;
#pragma unroll
    for (int j = 0; j < ORD_PER_THREAD; ++j) { s_rel[threadIdx.x * ORD_PER_THREAD + j] = run < 0xFFFFFFFFull ? (uint32_t)run : 0xFFFFFFFFu; run += cnt[j]; }
    if (threadIdx.x == ORD_NT - 1) s_rel[ORD_PER_BLOCK] = 0xFFFFFFFFu;           // sentinel: the walk stops here
    __syncthreads();
    const unsigned long long out0 = bsum[blockIdx.x];
    if (out0 >= cap) return;
    const uint32_t tot = (uint32_t)(total < cap - out0 ? total : cap - out0);   // positions this block may store
    uint32_t e = 0;
    constexpr int U = 4;
    for (uint32_t o0 = threadIdx.x; o0 < tot; o0 += U * ORD_NT) {
        uint4 val[U];
        bool ok[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t o = o0 + u * ORD_NT;
            ok[u] = false;
            if (o < tot) {
                while (s_rel[e + 1] <= o) ++e;                      // chunk holding output position o
                const unsigned long long src = (unsigned long long)s_src[e] + (o - s_rel[e]);
                ok[u] = s_src[e] != 0xFFFFFFFFu && src < arrival_cap;
                if (ok[u]) val[u] = __ldcs(arrival + src);
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
            if (ok[u]) ordered[out0 + o0 + u * ORD_NT] = val[u];
    }
}

cudaError_t launch_order(const EventSink &sink, uint32_t n, unsigned long long *bsum, uint4 *ordered,
                         unsigned long long capacity, const unsigned long long *step_events,
                         unsigned long long *total_events, cudaStream_t st)
{
    const uint32_t nb = (n + ORD_PER_BLOCK - 1) / ORD_PER_BLOCK;
    k_dir_blocksum<<<nb, ORD_NT, 0, st>>>(sink.directory, n, bsum);
    k_dir_scan_bsum<<<1, 1024, 0, st>>>(bsum, nb, step_events, total_events);
    k_dir_copy<<<nb, ORD_NT, 0, st>>>(sink.directory, n, bsum, sink.arrival, sink.arrival_cap, ordered, capacity);
    return cudaGetLastError();
}

}  // namespace evis
