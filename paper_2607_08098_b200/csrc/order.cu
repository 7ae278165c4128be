// order.cu -- row a8, second half: deterministic ordering of the compacted event stream.
//
// The compaction kernels reserve space with one global atomic per (tile, substep) chunk, so chunks
// land in the arrival buffer in scheduling order.  Each chunk left (arrival offset, count) in
// directory[d], d = ((env * S + substep-1) * tiles_y + tile_y) * tiles_x + tile_x.  Here the chunks
// are laid out in directory order: exclusive scan of the counts (three small kernels) and a
// chunk-by-chunk 128-bit copy.  Inside a chunk the order is the block scan order of the producer
// (pixel rank in the tile, then crossing index k), which is deterministic as well.
#include <mutex>

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

// One event into the voxel grid (kernels.h): xy = cropped pixel, w1 = env | polarity << 16 | substep << 24.
__device__ __forceinline__ void voxel_add(const VoxelSink &vox, uint32_t xy, uint32_t w1, float t_off)
{
    const float tau = fminf(__fmul_rn(__fadd_rn(vox.t_base, t_off), vox.scale), (float)(vox.bins - 1u));
    const float b0f = floorf(tau);
    const uint32_t b0 = (uint32_t)b0f;
    const unsigned long long q = __float2ull_rd(__fmul_rn(__fsub_rn(tau, b0f), 4294967296.0f));      // w in 32.32, exact
    const uint32_t ch = ((w1 >> 16) & 0xFFu) == 0x01u ? 0u : 1u;
    const size_t plane = (size_t)vox.hc * vox.wc;
    const size_t cell = (((size_t)(w1 & 0xFFFFu) * 2u + ch) * vox.bins + b0) * plane + (size_t)(xy >> 16) * vox.wc + (xy & 0xFFFFu);
    atomicAdd(vox.v + cell, 0x100000000ull - q);
    if (q && b0 + 1u < vox.bins) atomicAdd(vox.v + cell + plane, q);
}

// The 8-byte event of include/evis.h (evis_event8): x | y << 12 | env << 24 | substep << 40 | frac << 48 | ON << 63, frac =
// min(32767, floor(fr 2^15)) with fr in [0, 1] the stamp's position inside its substep.
__device__ __forceinline__ unsigned long long pack_event8(uint32_t xy, uint32_t w1, float fr)
{
    const uint32_t frac = min(32767u, (uint32_t)__float2uint_rd(__fmul_rn(fminf(fmaxf(fr, 0.0f), 1.0f), 32768.0f)));
    const unsigned long long on = ((w1 >> 16) & 0xFFu) == 0x01u ? 1ull : 0ull;
    return (unsigned long long)(xy & 0xFFFu) | ((unsigned long long)((xy >> 16) & 0xFFFu) << 12) |
           ((unsigned long long)(w1 & 0xFFFFu) << 24) | ((unsigned long long)(w1 >> 24) << 40) |
           ((unsigned long long)frac << 48) | (on << 63);
}

// shift: 0 = the entry's .y is an event count (direct mode: the chunk holds events), DIR_EV_SHIFT = records | events << shift
__global__ void __launch_bounds__(ORD_NT)
k_dir_blocksum(const uint2 *__restrict__ dir, uint32_t n, unsigned long long *__restrict__ bsum, int shift)
{
    __shared__ unsigned long long s_w[33];
    const uint32_t base = blockIdx.x * ORD_PER_BLOCK + threadIdx.x * ORD_PER_THREAD;
    unsigned long long v = 0;
#pragma unroll
    for (int j = 0; j < ORD_PER_THREAD; ++j)
        if (base + j < n) v += dir[base + j].y >> shift;
    unsigned long long total;
    block_scan_excl(v, s_w, total);
    if (threadIdx.x == 0) bsum[blockIdx.x] = total;
}

// single block: exclusive scan of the per-block sums in place
__global__ void __launch_bounds__(1024)
k_dir_scan_bsum(unsigned long long *__restrict__ bsum, uint32_t nb, const unsigned long long *__restrict__ step_events,
                unsigned long long *__restrict__ total_events, const unsigned long long *__restrict__ alloc,
                unsigned long long arrival_cap, unsigned long long capacity, unsigned long long *__restrict__ overflow_steps)
{
    if (threadIdx.x == 0) {
        *total_events += *step_events;
        if (*step_events > capacity || *alloc > arrival_cap) *overflow_steps += 1ull;      // sticky: evis_info.overflow_steps
    }
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
           unsigned long long cap, const VoxelSink vox)
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
    if (out0 >= cap && !vox.v) return;
    // positions this block may store; the voxel grid takes every event, stored or not
    const uint32_t tot_store = out0 >= cap ? 0u : (uint32_t)(total < cap - out0 ? total : cap - out0);
    const uint32_t tot = vox.v ? (uint32_t)total : tot_store;
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
            if (ok[u]) {
                const bool st_ = o0 + u * ORD_NT < tot_store;
                if (st_ && vox.store_events == 1) ordered[out0 + o0 + u * ORD_NT] = val[u];
                else if (st_ && vox.store_events == 2) {
                    // direct mode stamps in seconds: back to the fraction of the substep
                    const float t0 = __fmul_rn((float)((val[u].y >> 24) - 1u), vox.dt);
                    reinterpret_cast<unsigned long long *>(ordered)[out0 + o0 + u * ORD_NT] =
                        pack_event8(val[u].x, val[u].y, __fdividef(__fsub_rn(__uint_as_float(val[u].z), t0), vox.dt));
                }
                if (vox.v) voxel_add(vox, val[u].x, val[u].y, __uint_as_float(val[u].z));
            }
    }
}

// ---- global path: records -> events ------------------------------------------------------------------
// A block owns ORD_PER_BLOCK consecutive directory entries = one contiguous range of the ordered stream;
// the directory holds each chunk's event count, so the block scan of those counts places every chunk.
// Then the warps take chunks one at a time (shared counter): 32 records per pass -- one coalesced 16-byte
// load per lane --, warp scan of the crossing counts n, and the warp writes the pass's events 32 at a time, one per
// lane, found by a search over the scan (a7: timestamp of the k-th crossing, R8: linear in log intensity between
// L_prev and L_hat).
__global__ void __launch_bounds__(ORD_NT)
k_expand(const uint2 *__restrict__ dir, uint32_t n, const unsigned long long *__restrict__ bsum,
         const uint4 *__restrict__ arrival, unsigned long long arrival_cap, uint4 *__restrict__ ordered,
         unsigned long long cap, const EventParams ep, const Thresholds th, uint32_t W, uint32_t HW, uint32_t margin,
         uint32_t tiles_x, uint32_t tiles, uint32_t S, const VoxelSink vox)
{
    constexpr unsigned FULL = 0xFFFFFFFFu;
    __shared__ unsigned long long s_w[33];
    __shared__ uint32_t s_rel[ORD_PER_BLOCK];         // first output position of chunk e, relative to the block
    __shared__ uint2 s_dir[ORD_PER_BLOCK];            // its directory entry (arrival offset, records | events << shift)
    __shared__ uint32_t s_next;
    const uint32_t blk = blockIdx.x * ORD_PER_BLOCK;
    const uint32_t base = blk + threadIdx.x * ORD_PER_THREAD;
    constexpr uint32_t RMASK = (1u << DIR_EV_SHIFT) - 1u;
    uint32_t cnt[ORD_PER_THREAD];
    unsigned long long v = 0;
#pragma unroll
    for (int j = 0; j < ORD_PER_THREAD; ++j) {
        uint2 e = make_uint2(0u, 0u);
        if (base + j < n) e = dir[base + j];
        cnt[j] = e.y >> DIR_EV_SHIFT;
        v += cnt[j];
        s_dir[threadIdx.x * ORD_PER_THREAD + j] = e;
    }
    if (threadIdx.x == 0) s_next = 0;
    unsigned long long total;
    unsigned long long run = block_scan_excl(v, s_w, total);
    if (total == 0) return;
#pragma unroll
    for (int j = 0; j < ORD_PER_THREAD; ++j) { s_rel[threadIdx.x * ORD_PER_THREAD + j] = (uint32_t)run; run += cnt[j]; }
    __syncthreads();
    const unsigned long long out0 = bsum[blockIdx.x];
    if (out0 >= cap && !vox.v) return;
    const int lane = threadIdx.x & 31;
    for (;;) {
        uint32_t e = 0;
        if (lane == 0) e = atomicAdd(&s_next, 1u);
        e = __shfl_sync(FULL, e, 0);
        if (e >= ORD_PER_BLOCK) break;
        const uint2 de = s_dir[e];
        const uint32_t nrec = de.y & RMASK;
        if (nrec == 0) continue;
        // chunk d = (env * S + substep - 1) * tiles + tile
        const uint32_t d = blk + e;
        const uint32_t es = d / tiles, tile = d - es * tiles;
        const uint32_t env = es / S, sub = es - env * S + 1u;
        const uint32_t ty = tile / tiles_x, tx = tile - ty * tiles_x;
        const uint32_t org = (tx * G_TILE_W) | ((ty * G_TILE_H) << 16);
        const float t0 = __fmul_rn((float)(sub - 1u), ep.dt);
        unsigned long long first = out0 + s_rel[e];
        for (uint32_t r0 = 0; r0 < nrec; r0 += 32) {
            const uint32_t r = r0 + lane;
            uint4 rec = make_uint4(0u, 0u, 0u, 0u);
            const unsigned long long src = (unsigned long long)de.x + r;
            if (r < nrec && de.x != 0xFFFFFFFFu && src < arrival_cap) rec = __ldcs(arrival + src);
            const uint32_t nev = rec.w >> 16;
            uint32_t incl = nev;
#pragma unroll
            for (int dd = 1; dd < 32; dd <<= 1) {
                const uint32_t u = __shfl_up_sync(FULL, incl, dd);
                if (lane >= dd) incl += u;
            }
            const uint32_t excl = incl - nev, total_ev = __shfl_sync(FULL, incl, 31);
            // per record, in its own lane: polarity and threshold, cropped position, reciprocal of the denominator
            const float l_ref = __uint_as_float(rec.x), l_prev = __uint_as_float(rec.y), l_hat = __uint_as_float(rec.z);
            const bool up = __fsub_rn(l_hat, l_ref) > 0.0f;
            const uint32_t pos = rec.w & 0xFFFFu;
            const uint32_t xy = org + (pos % G_TILE_W) + ((pos / G_TILE_W) << 16);
            float pc = up ? ep.c_pos : -ep.c_neg;                        // p C
            if (th.on && nev) {                                          // Eq. 8: the pixel's own thresholds
                const size_t pix = (size_t)env * HW + (size_t)(xy >> 16) * W + (xy & 0xFFFFu);
                pc = up ? __ldg(th.on + pix) : -__ldg(th.off + pix);
            }
            const uint32_t xyc = xy - (margin | (margin << 16));         // coordinates in the cropped frame (R27)
            const uint32_t w1 = env | ((up ? 0x01u : 0xFFu) << 16) | (sub << 24);
            // fr_k = (L_ref + k p C - L_prev) / (L_hat - L_prev), clamped to [0, 1]; 1 when the denominator is 0.
            // Timestamps decide nothing (compared within 1e-7 s; a substep is ~1e-3 s): reciprocal once per record.
            // A zero denominator (fr = 1) is encoded as rden = +inf with L_prev = -inf: (lev + inf) * inf clamps to 1;
            // a NaN denominator (non-finite L) gives fr = NaN -> 0, like the oracle's !(fr >= 0).
            const float den = __fsub_rn(l_hat, l_prev);
            const bool flat = den == 0.0f;
            const float rden = flat ? __int_as_float(0x7F800000) : __fdividef(1.0f, den);
            const float l_prev_e = flat ? __int_as_float(0xFF800000) : l_prev;
            // the pass's events, 32 at a time, one per lane: event e belongs to the last lane s with excl[s] <= e
            // (a 5-step search over the scan), is its crossing k = e - excl[s] + 1, and goes to first + e -- the
            // stores of a warp are contiguous
            for (uint32_t e0 = 0; e0 < total_ev; e0 += 32) {
                const uint32_t e = e0 + lane;
                int sl = 0;
#pragma unroll
                for (int dd = 16; dd >= 1; dd >>= 1) {
                    const uint32_t tt = __shfl_sync(FULL, excl, sl + dd);
                    if (tt <= e) sl += dd;
                }
                const float kf = (float)(e - __shfl_sync(FULL, excl, sl) + 1u);
                const float o_ref = __shfl_sync(FULL, l_ref, sl), o_prev = __shfl_sync(FULL, l_prev_e, sl);
                const float o_pc = __shfl_sync(FULL, pc, sl), o_rden = __shfl_sync(FULL, rden, sl);
                const uint32_t o_xy = __shfl_sync(FULL, xyc, sl), o_w1 = __shfl_sync(FULL, w1, sl);
                float fr = __fmul_rn(__fsub_rn(__fmaf_rn(kf, o_pc, o_ref), o_prev), o_rden);
                fr = fminf(fmaxf(fr, 0.0f), 1.0f);
                const unsigned long long o = first + e;
                if (e < total_ev) {
                    const float t_off = __fmaf_rn(fr, ep.dt, t0);
                    if (o < cap) {
                        if (vox.store_events == 1) ordered[o] = make_uint4(o_xy, o_w1, __float_as_uint(t_off), ep.kf);
                        else if (vox.store_events == 2) reinterpret_cast<unsigned long long *>(ordered)[o] = pack_event8(o_xy, o_w1, fr);
                    }
                    if (vox.v) voxel_add(vox, o_xy, o_w1, t_off);        // the grid takes every event, stored or not
                }
            }
            first += total_ev;
        }
    }
}

cudaError_t launch_expand(const EventSink &sink, uint32_t n, unsigned long long *bsum, uint4 *ordered,
                          unsigned long long capacity, const unsigned long long *step_events,
                          unsigned long long *total_events, unsigned long long *overflow_steps, const EventParams &ep, const Thresholds &th, uint32_t W,
                          uint32_t HW, uint32_t margin, uint32_t tiles_x, uint32_t tiles, uint32_t S, const VoxelSink &vox, cudaStream_t st)
{
    const uint32_t nb = (n + ORD_PER_BLOCK - 1) / ORD_PER_BLOCK;
    k_dir_blocksum<<<nb, ORD_NT, 0, st>>>(sink.directory, n, bsum, DIR_EV_SHIFT);
    k_dir_scan_bsum<<<1, 1024, 0, st>>>(bsum, nb, step_events, total_events, sink.alloc, sink.arrival_cap, capacity, overflow_steps);
    k_expand<<<nb, ORD_NT, 0, st>>>(sink.directory, n, bsum, sink.arrival, sink.arrival_cap, ordered, capacity, ep, th,
                                    W, HW, margin, tiles_x, tiles, S, vox);
    return cudaGetLastError();
}

cudaError_t launch_order(const EventSink &sink, uint32_t n, unsigned long long *bsum, uint4 *ordered,
                         unsigned long long capacity, const unsigned long long *step_events,
                         unsigned long long *total_events, unsigned long long *overflow_steps, const VoxelSink &vox, cudaStream_t st)
{
    const uint32_t nb = (n + ORD_PER_BLOCK - 1) / ORD_PER_BLOCK;
    k_dir_blocksum<<<nb, ORD_NT, 0, st>>>(sink.directory, n, bsum, 0);
    k_dir_scan_bsum<<<1, 1024, 0, st>>>(bsum, nb, step_events, total_events, sink.alloc, sink.arrival_cap, capacity, overflow_steps);
    k_dir_copy<<<nb, ORD_NT, 0, st>>>(sink.directory, n, bsum, sink.arrival, sink.arrival_cap, ordered, capacity, vox);
    return cudaGetLastError();
}

// V (32.32 fixed point) -> float32; one block per (env, channel, bin) plane; normalize: divided by the plane's maximum
__global__ void __launch_bounds__(256)
k_voxel_finish(const unsigned long long *__restrict__ v, float *__restrict__ out, uint32_t cells, int normalize)
{
    __shared__ unsigned long long s_m[8];
    const unsigned long long *pv = v + (size_t)blockIdx.x * cells;
    float *po = out + (size_t)blockIdx.x * cells;
    double inv = 1.0 / 4294967296.0;
    if (normalize) {
        unsigned long long m = 0;
        for (uint32_t i = threadIdx.x; i < cells; i += blockDim.x) { const unsigned long long x = pv[i]; m = x > m ? x : m; }
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) { const unsigned long long o = __shfl_xor_sync(0xFFFFFFFFu, m, d); m = o > m ? o : m; }
        if ((threadIdx.x & 31) == 0) s_m[threadIdx.x >> 5] = m;
        __syncthreads();
        m = 0;
        for (int w = 0; w < 8; ++w) m = s_m[w] > m ? s_m[w] : m;
        if (m) inv = 1.0 / (double)m;
    }
    for (uint32_t i = threadIdx.x; i < cells; i += blockDim.x) po[i] = (float)((double)pv[i] * inv);
}

cudaError_t launch_voxel_finish(const unsigned long long *v, float *out, uint32_t planes, uint32_t cells, int normalize,
                                cudaStream_t st)
{
    k_voxel_finish<<<planes, 256, 0, st>>>(v, out, cells, normalize);
    return cudaGetLastError();
}

// ---- evis_voxelize_static: the voxel grid of a finished event stream, with no device allocation (include/evis.h) ------
//
// For callers that must not allocate on the device while they run: a rollout loop whose simulator, renderer and learner
// have divided the GPU's memory among their own pools up front (a cudaMalloc there can fail, and cudaMalloc / cudaFree
// make every stream of the device wait), or a consumer that holds events but no evis_ctx.  evis_set_voxels allocates its
// accumulator; this entry point keeps ONE accumulator of fixed size in the library's image instead.
//
// g_voxel_static is that accumulator (scratch: 32.32 fixed-point sums, like evis_ctx::vox_v): every GPU that loads the
// library holds its EVIS_VOXELIZE_STATIC_MAX_CELLS * 8 bytes = 16 MiB from the moment the module is loaded until the
// process exits.  In HOST code the name g_voxel_static is only a handle for the runtime, not a device address (a kernel
// handed it would fault or touch the wrong memory): voxel_static_address() asks the runtime for the address on the
// current device, once per device, and the kernels get that pointer.
__device__ __align__(256) static unsigned long long g_voxel_static[EVIS_VOXELIZE_STATIC_MAX_CELLS];

constexpr int VOXEL_STATIC_MAX_DEVICES = 64;
static unsigned long long *g_voxel_static_ptr[VOXEL_STATIC_MAX_DEVICES];      // per device ordinal; null = not asked yet
static std::mutex g_voxel_static_mu;

// device address of g_voxel_static on the CURRENT device (set-up on the first call per device)
static cudaError_t voxel_static_address(unsigned long long **out)
{
    int dev = -1;
    cudaError_t rc = cudaGetDevice(&dev);
    if (rc != cudaSuccess) return rc;
    if (dev < 0 || dev >= VOXEL_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_voxel_static_mu);
    if (!g_voxel_static_ptr[dev]) {
        unsigned long long *p = nullptr;
        rc = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_voxel_static);
        if (rc != cudaSuccess) return rc;
        if (!p) return cudaErrorInvalidSymbol;
        g_voxel_static_ptr[dev] = p;
    }
    *out = g_voxel_static_ptr[dev];
    return cudaSuccess;
}

// The accumulation of k_expand / k_dir_copy (voxel_add) as a kernel of its own over finished 16-byte events: the
// event's interval index places it in the window, t = (kf - first_kf) T + t_off.  Events outside the window, the
// frame or the env range add nothing.
__global__ void __launch_bounds__(256)
k_voxel_events(const uint4 *__restrict__ events, unsigned long long n, uint32_t E, uint32_t first_kf, uint32_t window_steps,
               float T, const VoxelSink vox)
{
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const uint4 ev = __ldcs(events + i);              // x | y << 16, env | p << 16 | substep << 24, t_off, kf
        const uint32_t j = ev.w - first_kf;
        if (j >= window_steps || (ev.x & 0xFFFFu) >= vox.wc || (ev.x >> 16) >= vox.hc || (ev.y & 0xFFFFu) >= E) continue;
        VoxelSink v = vox;
        v.t_base = __fmul_rn((float)j, T);
        voxel_add(v, ev.x, ev.y, __uint_as_float(ev.z));
    }
}

}  // namespace evis

extern "C" int evis_voxelize_static(const evis_event *events, uint64_t n_events, int32_t num_envs, int32_t height, int32_t width,
                                    int32_t bins, int32_t window_steps, float keyframe_dt, uint32_t first_kf, int normalize,
                                    float *grid, void *cuda_stream, int *cuda_error)
{
    using namespace evis;
    if (cuda_error) *cuda_error = 0;
    if (!grid || (!events && n_events) || num_envs <= 0 || num_envs > 65535 || height <= 0 || height > 32767 || width <= 0 ||
        width > 32767 || bins < 1 || window_steps < 1 || !(keyframe_dt > 0.0f) || !(keyframe_dt <= 3.0e38f))
        return EVIS_ERR_INVALID_ARG;
    const unsigned long long plane = (unsigned long long)height * (unsigned long long)width;
    const unsigned long long planes = 2ull * (unsigned long long)num_envs * (unsigned long long)bins;     // < 2^48
    if (planes > EVIS_VOXELIZE_STATIC_MAX_CELLS || plane * planes > EVIS_VOXELIZE_STATIC_MAX_CELLS) return EVIS_ERR_TOO_LARGE;
    const unsigned long long cells = plane * planes;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned long long *acc = nullptr;
    cudaError_t rc = voxel_static_address(&acc);
    // the array keeps what the last call left in it: the part this call uses starts at zero
    if (rc == cudaSuccess) rc = cudaMemsetAsync(acc, 0, cells * sizeof(unsigned long long), st);
    if (rc == cudaSuccess && n_events) {
        VoxelSink vs{};
        vs.v = acc;
        vs.bins = (uint32_t)bins; vs.hc = (uint32_t)height; vs.wc = (uint32_t)width;
        volatile float sc = (float)(bins - 1) / ((float)window_steps * keyframe_dt);      // as evis_step forms it
        vs.scale = sc;
        const unsigned long long want = (n_events + 255ull) / 256ull;
        const unsigned blocks = (unsigned)(want < 148ull * 16ull ? want : 148ull * 16ull);
        k_voxel_events<<<blocks, 256, 0, st>>>(reinterpret_cast<const uint4 *>(events), n_events, (uint32_t)num_envs, first_kf,
                                               (uint32_t)window_steps, keyframe_dt, vs);
        rc = cudaGetLastError();
    }
    if (rc == cudaSuccess) rc = launch_voxel_finish(acc, grid, (uint32_t)planes, (uint32_t)plane, normalize, st);
    if (rc != cudaSuccess) {
        if (cuda_error) *cuda_error = (int)rc;
        return EVIS_ERR_CUDA;
    }
    return EVIS_OK;
}
