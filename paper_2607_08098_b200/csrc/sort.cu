// sort.cu -- the time-sorted per-environment stream (the stream E = {(u_k, t_k, p_k)}).
//
// The ordered stream of a step is grouped by environment and, inside an environment, laid out by (substep, tile, y, x,
// k).  evis_set_time_sorted makes the order stage sort every environment's segment by the events' timestamps t_off:
// a segmented, STABLE least-significant-digit radix sort on the 32 bits of t_off (a non-negative binary32: its bit
// pattern orders like its value), four passes of 8 bits, ping-ponging between the ordered buffer and the step's
// (by then free) arrival buffer.  Stable: events with equal stamps keep the ordered stream's order, so the result is
// deterministic.  The segment is the ENVIRONMENT, not (env, substep): binary32 rounding can put the last stamp of
// substep i one ulp above the first of substep i + 1.
//
// A segment is cut into tiles of SORT_TILE events, one block each (a block never spans two segments):
//   k_seg_counts    events per environment from the directory (its entries are env-major)
//   k_seg_scan      segment starts in the stream and first block of every segment (one block)
// and per pass (the blocks hold other events after every pass, so their histograms are taken again; counting the next
// pass's digit per destination block with global atomics inside the scatter was measured slower than the extra read):
//   k_sort_hist     per block: histogram of the pass's digit
//   k_sort_scan     per segment: where each block's run of each digit goes (digit-major, block-minor: stable)
//   k_sort_scatter  stable rank of every event inside its block's digit run, then the move
#include "kernels.h"

namespace evis {

constexpr int SORT_NT = 256, SORT_TILE = 4096, SORT_ROUNDS = SORT_TILE / SORT_NT, SORT_BINS = 256, SORT_PASSES = 4;

// events of env e = sum of its directory entries' event counts.  shift: see k_dir_blocksum (order.cu)
__global__ void __launch_bounds__(SORT_NT)
k_seg_counts(const uint2 *__restrict__ dir, uint32_t entries_per_env, int shift, unsigned long long *__restrict__ seg_count)
{
    __shared__ unsigned long long s_w[SORT_NT / 32];
    const uint2 *d = dir + (size_t)blockIdx.x * entries_per_env;
    unsigned long long v = 0;
    for (uint32_t i = threadIdx.x; i < entries_per_env; i += SORT_NT) v += d[i].y >> shift;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
        for (int w = 0; w < SORT_NT / 32; ++w) t += s_w[w];
        seg_count[blockIdx.x] = t;
    }
}

// one thread: exclusive scans over the E segments (E <= 65535): start of the segment in the stream (cut at `cap`
// stored events) and its first block.  seg_start[E] / seg_block[E] = totals.
__global__ void k_seg_scan(const unsigned long long *__restrict__ seg_count, uint32_t E, unsigned long long cap,
                           unsigned long long *__restrict__ seg_start, uint32_t *__restrict__ seg_block)
{
    if (threadIdx.x || blockIdx.x) return;
    unsigned long long run = 0;
    uint32_t blk = 0;
    for (uint32_t e = 0; e < E; ++e) {
        const unsigned long long a = run < cap ? run : cap;
        run += seg_count[e];
        const unsigned long long b = run < cap ? run : cap;
        seg_start[e] = a;
        seg_block[e] = blk;
        blk += (uint32_t)((b - a + SORT_TILE - 1) / SORT_TILE);
    }
    seg_start[E] = run < cap ? run : cap;
    seg_block[E] = blk;
}

// block -> (segment, first event, events) through a search over seg_block; false: no such block
__device__ __forceinline__ bool sort_block(const unsigned long long *__restrict__ seg_start, const uint32_t *__restrict__ seg_block,
                                           uint32_t E, uint32_t blk, uint32_t &seg, unsigned long long &first, uint32_t &n)
{
    if (blk >= seg_block[E]) return false;
    uint32_t lo = 0, hi = E - 1;                    // last segment with seg_block <= blk that owns blocks
    while (lo < hi) {
        const uint32_t mid = (lo + hi + 1) >> 1;
        if (seg_block[mid] <= blk) lo = mid; else hi = mid - 1;
    }
    seg = lo;
    const unsigned long long s0 = seg_start[seg], s1 = seg_start[seg + 1];
    first = s0 + (unsigned long long)(blk - seg_block[seg]) * SORT_TILE;
    const unsigned long long left = s1 - first;
    n = (uint32_t)(left < SORT_TILE ? left : SORT_TILE);
    return true;
}

// hist[block][digit] of the pass's digit
__global__ void __launch_bounds__(SORT_NT)
k_sort_hist(const uint4 *__restrict__ src, const unsigned long long *__restrict__ seg_start, const uint32_t *__restrict__ seg_block,
            uint32_t E, uint32_t *__restrict__ hist, int pass)
{
    __shared__ uint32_t s_h[SORT_BINS];
    uint32_t seg, n;
    unsigned long long first;
    if (!sort_block(seg_start, seg_block, E, blockIdx.x, seg, first, n)) return;
    s_h[threadIdx.x] = 0;
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < n; i += SORT_NT) atomicAdd(&s_h[(src[first + i].z >> (8 * pass)) & 0xFFu], 1u);
    __syncthreads();
    hist[(size_t)blockIdx.x * SORT_BINS + threadIdx.x] = s_h[threadIdx.x];
}

// one block per segment, one thread per digit: hist[block][digit] (counts) -> where the block's run of that digit
// starts, relative to the segment: all smaller digits of the segment + the same digit in the segment's earlier blocks
__global__ void __launch_bounds__(SORT_BINS)
k_sort_scan(const uint32_t *__restrict__ seg_block, uint32_t *__restrict__ hist)
{
    __shared__ uint32_t s_tot[SORT_BINS];
    const uint32_t seg = blockIdx.x, b0 = seg_block[seg], b1 = seg_block[seg + 1], d = threadIdx.x;
    if (b0 == b1) return;
    uint32_t tot = 0;
    for (uint32_t b = b0; b < b1; ++b) tot += hist[(size_t)b * SORT_BINS + d];
    s_tot[d] = tot;
    __syncthreads();
    uint32_t base = 0;
    for (uint32_t q = 0; q < d; ++q) base += s_tot[q];              // 256 adds per thread: negligible beside the scatter
    for (uint32_t b = b0; b < b1; ++b) {
        const uint32_t c = hist[(size_t)b * SORT_BINS + d];
        hist[(size_t)b * SORT_BINS + d] = base;
        base += c;
    }
}

// One pass: stable scatter of the block's events by the pass's digit.  Warp w owns the tile's events
// [w * 512, (w + 1) * 512) and ranks them round by round (32 consecutive events per round) against its own row of digit
// counters -- __match_any_sync groups the lanes of a round by digit --, keeping events and ranks in registers; one block
// barrier later the rows are turned into the start of every (warp, digit) run inside the block's run of that digit, and
// the events are moved.  Order inside a digit = (warp, round, lane) = the order in the tile: stable.
__global__ void __launch_bounds__(SORT_NT)
k_sort_scatter(const uint4 *__restrict__ src, uint4 *__restrict__ dst, const unsigned long long *__restrict__ seg_start,
               const uint32_t *__restrict__ seg_block, uint32_t E, const uint32_t *__restrict__ hist, int pass)
{
    constexpr int NW = SORT_NT / 32, PER_WARP = SORT_TILE / NW;
    __shared__ uint32_t s_cnt[NW][SORT_BINS];
    uint32_t seg, n;
    unsigned long long first;
    if (!sort_block(seg_start, seg_block, E, blockIdx.x, seg, first, n)) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int w = 0; w < NW; ++w) s_cnt[w][threadIdx.x] = 0;
    __syncthreads();
    uint4 ev[SORT_ROUNDS];
    uint32_t rk[SORT_ROUNDS];                        // rank among the warp's events of the same digit | digit << 16
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; ++r) {
        const uint32_t i = (uint32_t)(warp * PER_WARP + r * 32 + lane);
        ev[r] = i < n ? __ldcs(src + first + i) : make_uint4(0u, 0u, 0u, 0u);
    }
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; ++r) {
        const uint32_t i = (uint32_t)(warp * PER_WARP + r * 32 + lane);
        const bool have = i < n;
        const uint32_t digit = have ? (ev[r].z >> (8 * pass)) & 0xFFu : 0x100u;
        const unsigned peers = __match_any_sync(0xFFFFFFFFu, digit);
        uint32_t before = 0;
        if (have) before = s_cnt[warp][digit];
        __syncwarp();
        if (have && (peers & lt) == 0u) s_cnt[warp][digit] = before + __popc(peers);
        __syncwarp();
        rk[r] = (before + __popc(peers & lt)) | (digit << 16);
    }
    __syncthreads();
    {
        uint32_t base = hist[(size_t)blockIdx.x * SORT_BINS + threadIdx.x];      // the block's run of digit threadIdx.x
#pragma unroll
        for (int w = 0; w < NW; ++w) { const uint32_t c = s_cnt[w][threadIdx.x]; s_cnt[w][threadIdx.x] = base; base += c; }
    }
    __syncthreads();
    const unsigned long long seg0 = seg_start[seg];
#pragma unroll
    for (int r = 0; r < SORT_ROUNDS; ++r) {
        const uint32_t digit = rk[r] >> 16;
        if (digit < 0x100u) dst[seg0 + s_cnt[warp][digit] + (rk[r] & 0xFFFFu)] = ev[r];
    }
}

// ws: workspace of sort_workspace_bytes(E, capacity): seg_count [E+1] u64 | seg_start [E+1] u64 | seg_block [E+1] u32 |
// hist [max_blocks][256] u32.  `a` holds the ordered stream and receives the sorted one (an even number of
// passes); `b` is scratch of the same size.
static size_t sort_hist_offset(uint32_t E) { return ((size_t)(E + 1) * 20 + 15) & ~(size_t)15; }

size_t sort_workspace_bytes(uint32_t E, unsigned long long capacity)
{
    const size_t max_blocks = (size_t)(capacity / SORT_TILE) + E + 1;
    return sort_hist_offset(E) + max_blocks * SORT_BINS * sizeof(uint32_t);
}

cudaError_t launch_time_sort(const uint2 *directory, uint32_t num_entries, int dir_shift, uint32_t E, unsigned long long capacity,
                             uint4 *a, uint4 *b, void *ws, cudaStream_t st)
{
    const uint32_t max_blocks = (uint32_t)(capacity / SORT_TILE) + E + 1;
    unsigned long long *seg_count = reinterpret_cast<unsigned long long *>(ws);
    unsigned long long *seg_start = seg_count + (E + 1);
    uint32_t *seg_block = reinterpret_cast<uint32_t *>(seg_start + (E + 1));
    uint32_t *hist = reinterpret_cast<uint32_t *>(reinterpret_cast<unsigned char *>(ws) + sort_hist_offset(E));
    k_seg_counts<<<E, SORT_NT, 0, st>>>(directory, num_entries / E, dir_shift, seg_count);
    k_seg_scan<<<1, 32, 0, st>>>(seg_count, E, capacity, seg_start, seg_block);
    for (int p = 0; p < SORT_PASSES; ++p) {
        const uint4 *src = p & 1 ? b : a;
        k_sort_hist<<<max_blocks, SORT_NT, 0, st>>>(src, seg_start, seg_block, E, hist, p);
        k_sort_scan<<<E, SORT_BINS, 0, st>>>(seg_block, hist);
        k_sort_scatter<<<max_blocks, SORT_NT, 0, st>>>(src, p & 1 ? a : b, seg_start, seg_block, E, hist, p);
    }
    return cudaGetLastError();
}

}  // namespace evis
