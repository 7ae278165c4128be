// tile_path.cu -- rows a2-a8 fused per target tile, z-buffers in shared memory (bounded motion).
//
// Persistent kernel: one CTA per SM takes (env, tile) work items from a global counter.  For its
// tile (tw x th <= 64 x 32 target pixels) a CTA runs ALL S substeps of the keyframe interval, so the
// keyframes are read once, L_ref / L_prev stay in registers and only events are written
// (north_star).  Sources that can reach the tile lie inside the tile grown by the halo
// h = ceil(max_motion_px) + 1 ("halo sized from the motion bound").
//
//   stage      once per tile and direction: scan the halo region, keep the sources whose swept
//              landing box can touch the tile ("candidates": position, displacement, own depth, far
//              endpoint depth of Eq. 7) in shared memory.  Direction A is staged lazily, only when
//              some substep of this tile has a pixel B does not reach (A fills holes).
//   splat      per substep: every candidate computes q (Eq. 5), Zt (Eq. 7), its footprint class (R14)
//              and offers the packed key [dir | Zt bits | source index] (R15) to the shared z-buffer.
//              A source with positive weight on all four pixels is filed once under its floor cell
//              (cell buffer zc), otherwise under its 1-2 target pixels (zd) -- as in global_path.cu.
//              64-bit shared atomicMin is a CAS loop on sm_100a and ATOMS runs at ~2 cycles/lane, so
//              the minimum is taken OPTIMISTICALLY with plain 64-bit loads/stores: store if smaller,
//              barrier, re-check; a round in which no thread had to store proves every cell holds
//              the minimum of the keys offered to it (each thread only ever lowers a cell, and every
//              candidate re-checks its own key after the last store).  Deterministic: the result is
//              the minimum, whatever the interleaving.  Direction A only offers the candidates that
//              land inside the bounding box of this substep's holes.
//   resolve    per target pixel: minimum over zd and the four cells that can cover it, composite
//              (the direction bit makes "B primary, A fills holes" a plain minimum), gather L.
//   events     Eq. 4 + timestamps (R8).  Per-warp totals -> one barrier -> every warp derives its own
//              offset inside the (tile, substep) chunk; the chunk's space comes from a slab of the
//              arrival buffer the CTA owns (one global atomic per T_SLAB events, not per chunk);
//              warp-cooperative writes (common.cuh).  directory[(env, substep, tile)] records the
//              chunk so that order.cu can lay the stream out deterministically.
//
// Barriers per substep in the common case (no hole, no z conflict): after the z clear, after the
// optimistic stores, after check + gather + event count.
//
// A tile whose candidates all have zero motion and valid depth is static: every substep reproduces
// L_B, no splat is needed (bit-identical to the general path).
#include <cstdlib>

#include "kernels.h"

namespace evis {

constexpr int T_NT = 512;                       // threads per CTA
constexpr int T_NW = T_NT / 32;
constexpr int T_MAX_TW = 64, T_MAX_TH = 32;
constexpr int T_TPT = T_MAX_TW * T_MAX_TH / T_NT;   // targets per thread (4)
constexpr int T_CAP = 4608;                     // resident candidates per direction
constexpr int T_CPT = T_CAP / T_NT;             // candidates per thread (9)
constexpr int T_SLAB = 8192;                    // events per arrival slab
constexpr uint32_t A_NONE = 0xFFFFFFFFu;
static_assert(T_CAP % T_NT == 0 && T_TPT * T_NT == T_MAX_TW * T_MAX_TH, "tile constants");

struct TileArgs {
    Geom g;
    int tw, th, halo, tiles_x, tiles_y, force_direct;
    uint32_t num_items;                 // E * tiles_y * tiles_x
    unsigned long long *next_item;      // work counter (reset every step)
    const float *LA, *LB, *ZA, *ZB;
    const float2 *mvA, *fwdA, *mvB;     // fwdA nullable (R12)
    const SubstepTable *tab;
    float *l_ref, *l_prev;
    EventParams ep;
    EventSink sink;
    unsigned long long *holes;
    DebugOut dbg;
};

// Candidate pool in shared memory, structure of arrays; direction B uses [0, T_CAP), A [T_CAP, 2 T_CAP).
struct Pool {
    uint32_t *pos;      // x | y << 16 (pixel of the env)
    float *dx, *dy;     // displacement field of the direction (m_B, or -m_A / explicit forward field)
    float *zo, *zf;     // own depth, depth at the far endpoint of the correspondence (Eq. 7, R16)
};

struct TileGeo {
    int X0, Y0;         // tile origin
    int tw, th;         // tile size (clipped targets are those with X0+tx < W, Y0+ty < H)
    int RX0, RY0, RW, RH;  // halo region clipped to the image
    int zc_off;         // offset of the cell buffer inside the z-buffer array (= tw * th)
    int zc_w;           // cell row stride (= tw + 1)
    int W, H;
};

__device__ __forceinline__ bool zput(volatile unsigned long long *z, uint32_t a, unsigned long long key)
{
    const unsigned long long cur = z[a];
    if (key < cur) { z[a] = key; return true; }
    return false;
}

// Where a landing goes inside the tile's z-buffer: a0 (and a1 for a two-pixel footprint).
__device__ __forceinline__ void tile_addr(const Landing &L, const TileGeo &t, uint32_t &a0, uint32_t &a1)
{
    a0 = a1 = A_NONE;
    const int cx = L.x0 + 1 - t.X0, cy = L.y0 + 1 - t.Y0;          // cell coordinates
    if (L.cls == 3) {
        if ((unsigned)cx <= (unsigned)t.tw && (unsigned)cy <= (unsigned)t.th) a0 = t.zc_off + cy * t.zc_w + cx;
        return;
    }
    const int tx = cx - 1, ty = cy - 1;
    const bool in_y0 = (unsigned)ty < (unsigned)t.th, in_x0 = (unsigned)tx < (unsigned)t.tw;
    if (in_x0 && in_y0) a0 = ty * t.tw + tx;
    if (L.cls == 1) { if ((unsigned)(tx + 1) < (unsigned)t.tw && in_y0) a1 = ty * t.tw + tx + 1; }
    else if (L.cls == 2) { if ((unsigned)(ty + 1) < (unsigned)t.th && in_x0) a1 = (ty + 1) * t.tw + tx; }
}

// One source of the halo region: does its swept landing box touch the tile?  Loads its record.
// dir 0 = B (disp m_B, far endpoint in A), dir 1 = A (disp -m_A or explicit forward, far endpoint in B).
__device__ __forceinline__ bool candidate(const TileArgs &a, const TileGeo &t, size_t eoff, int dir, int x, int y,
                                          float &dx, float &dy, float &zo, float &zf)
{
    const int p = y * t.W + x;
    float2 m;
    if (dir == 0) m = __ldg(a.mvB + eoff + p);
    else if (a.fwdA) m = __ldg(a.fwdA + eoff + p);
    else { const float2 b = __ldg(a.mvA + eoff + p); m = make_float2(-b.x, -b.y); }
    dx = m.x; dy = m.y;
    const float fx = (float)x, fy = (float)y;
    const float ex = fx + dx, ey = fy + dy;
    // q = x + w dx, w in [0,1], lies between x and x+dx; the footprint is floor(q) and floor(q)+1, so it
    // touches the tile columns [X0, X0+tw-1] only if max(x, x+dx) >= X0 - 1 and min(x, x+dx) < X0 + tw.
    // 1/16 px of slack absorbs the rounding of q and of x+dx (coordinates < 2^15: ulp <= 2^-8).
    const bool hit = fmaxf(fx, ex) >= (float)(t.X0 - 1) - 0.0625f && fminf(fx, ex) <= (float)(t.X0 + t.tw) + 0.0625f &&
                     fmaxf(fy, ey) >= (float)(t.Y0 - 1) - 0.0625f && fminf(fy, ey) <= (float)(t.Y0 + t.th) + 0.0625f;
    if (!hit) return false;                         // also rejects NaN displacements (dropped, R18)
    const float *Zs = (dir == 0 ? a.ZB : a.ZA) + eoff, *Zo = (dir == 0 ? a.ZA : a.ZB) + eoff;
    zo = __ldg(Zs + p);
    zf = far_depth(Zo, fx, fy, dx, dy, zo, t.W, t.H);
    return true;
}

// q of Eq. 5 for a candidate of direction DIR at time weights (f, g): B moves by g m_B, A by f d_A.
template <int DIR>
__device__ __forceinline__ bool land_dir(float x, float y, float dx, float dy, float zo, float zf, float f, float g,
                                         uint32_t src, int W, int H, Landing &L)
{
    // B: q = p + (1-f) m_B, Za = far, Zb = own.   A: q = p + f d_A, Za = own, Zb = far.   (Eq. 5, 7)
    if (DIR == 0) return land(x, y, dx, dy, g, f, g, zf, zo, src, 0ull, W, H, L);
    return land(x, y, dx, dy, f, f, g, zo, zf, src, KEY_DIR_A, W, H, L);
}

__device__ __forceinline__ unsigned long long tile_gather(const volatile unsigned long long *z, const TileGeo &t,
                                                          int tx, int ty)
{
    unsigned long long k = z[ty * t.tw + tx];
    const volatile unsigned long long *c = z + t.zc_off + ty * t.zc_w + tx;
    k = umin64(k, c[0]);
    k = umin64(k, c[1]);
    k = umin64(k, c[t.zc_w]);
    k = umin64(k, c[t.zc_w + 1]);
    return k;
}

// ---- stage: compact the candidates of one direction into the pool --------------------------------
// Unordered compaction (warp ballot + one shared atomicAdd per warp and pass): the slot order is
// irrelevant because the key carries the source's global index.  Returns the number of candidates
// (block-uniform); more than T_CAP means the direction is not resident.  `flags` accumulates, per
// thread, bit 0 = "a candidate moves or has a depth the static shortcut cannot take".
__device__ int stage(const TileArgs &a, const TileGeo &t, size_t eoff, int dir, const Pool &pool, int base,
                     uint32_t *s_count, uint32_t &flags)
{
    if (threadIdx.x == 0) *s_count = 0;
    __syncthreads();
    const int nR = t.RW * t.RH;
    const int lane = threadIdx.x & 31;
    int ly = threadIdx.x / t.RW, lx = threadIdx.x - ly * t.RW;
    const int sy = T_NT / t.RW, sx = T_NT - sy * t.RW;
    for (int r0 = 0; r0 < nR; r0 += T_NT) {
        const int r = r0 + threadIdx.x;
        bool pass = false;
        float dx = 0.f, dy = 0.f, zo = 0.f, zf = 0.f;
        const int x = t.RX0 + lx, y = t.RY0 + ly;
        if (r < nR) pass = candidate(a, t, eoff, dir, x, y, dx, dy, zo, zf);
        const unsigned m = __ballot_sync(0xFFFFFFFFu, pass);
        if (m) {
            const int leader = __ffs(m) - 1;
            int b = 0;
            if (lane == leader) b = (int)atomicAdd(s_count, (uint32_t)__popc(m));
            b = __shfl_sync(0xFFFFFFFFu, b, leader);
            if (pass) {
                const int slot = b + __popc(m & ((1u << lane) - 1u));
                if (slot < T_CAP) {
                    pool.pos[base + slot] = (uint32_t)x | ((uint32_t)y << 16);
                    pool.dx[base + slot] = dx; pool.dy[base + slot] = dy;
                    pool.zo[base + slot] = zo; pool.zf[base + slot] = zf;
                }
                const bool plain = dx == 0.0f && dy == 0.0f && zo > 1e-30f && zo < 1e30f && zf > 1e-30f && zf < 1e30f;
                if (!plain) flags |= 1u;
            }
        }
        lx += sx; ly += sy;
        if (lx >= t.RW) { lx -= t.RW; ++ly; }
    }
    __syncthreads();
    return (int)*s_count;
}

// ---- splat of one resident direction at one substep: optimistic stores, then the re-checks ---------
// Hole box of direction A (float, inclusive): only sources with q inside it can cover a hole.
struct Box { float x0, y0, x1, y1; };

template <int DIR>
__device__ __forceinline__ void splat_store(volatile unsigned long long *z, const Pool &pool, int base, int n, float f,
                                            float g, const TileGeo &t, const Box &box, unsigned long long (&key)[T_CPT],
                                            uint32_t (&adr)[T_CPT])
{
#pragma unroll
    for (int j = 0; j < T_CPT; ++j) {
        const int s = j * T_NT + threadIdx.x;
        adr[j] = 0xFFFFFFFFu;                   // a0 | a1 << 16, 0xFFFF = none
        key[j] = KEY_EMPTY;
        if (s < n) {
            const uint32_t pos = pool.pos[base + s];
            const int x = (int)(pos & 0xFFFFu), y = (int)(pos >> 16);
            const float dx = pool.dx[base + s], dy = pool.dy[base + s];
            if (DIR == 1) {                     // cheap reject: lands outside the hole box (same q as land())
                const float qx = __fmaf_rn(f, dx, (float)x), qy = __fmaf_rn(f, dy, (float)y);
                if (!(qx >= box.x0 && qx <= box.x1 && qy >= box.y0 && qy <= box.y1)) continue;
            }
            Landing L;
            if (land_dir<DIR>((float)x, (float)y, dx, dy, pool.zo[base + s], pool.zf[base + s], f, g,
                              (uint32_t)(y * t.W + x), t.W, t.H, L)) {
                uint32_t a0, a1;
                tile_addr(L, t, a0, a1);
                adr[j] = (a0 & 0xFFFFu) | (a1 << 16);
                key[j] = L.key;
                if (a0 != A_NONE) zput(z, a0, L.key);
                if (a1 != A_NONE) zput(z, a1, L.key);
            }
        }
    }
}

__device__ __forceinline__ bool splat_check(volatile unsigned long long *z, const unsigned long long (&key)[T_CPT],
                                            const uint32_t (&adr)[T_CPT])
{
    bool fail = false;
#pragma unroll
    for (int j = 0; j < T_CPT; ++j) {
        const uint32_t a0 = adr[j] & 0xFFFFu, a1 = adr[j] >> 16;
        if (a0 != 0xFFFFu) fail |= zput(z, a0, key[j]);
        if (a1 != 0xFFFFu) fail |= zput(z, a1, key[j]);
    }
    return fail;
}

// Non-resident direction (more candidates than the pool holds): walk the halo region every round.
// Leaves the final minima in z (ends with a barrier).
template <int DIR>
__device__ void splat_direct(volatile unsigned long long *z, const TileArgs &a, const TileGeo &t, size_t eoff,
                             float f, float g)
{
    const int nR = t.RW * t.RH;
    bool fail;
    do {
        __syncthreads();
        fail = false;
        for (int r = threadIdx.x; r < nR; r += T_NT) {
            const int ly = r / t.RW, lx = r - ly * t.RW;
            const int x = t.RX0 + lx, y = t.RY0 + ly;
            float dx, dy, zo, zf;
            if (!candidate(a, t, eoff, DIR, x, y, dx, dy, zo, zf)) continue;
            Landing L;
            if (!land_dir<DIR>((float)x, (float)y, dx, dy, zo, zf, f, g, (uint32_t)(y * t.W + x), t.W, t.H, L)) continue;
            uint32_t a0, a1;
            tile_addr(L, t, a0, a1);
            if (a0 != A_NONE) fail |= zput(z, a0, L.key);
            if (a1 != A_NONE) fail |= zput(z, a1, L.key);
        }
    } while (__syncthreads_or(fail));
}

// ---- the fused tile kernel -------------------------------------------------------------------------
__global__ void __launch_bounds__(T_NT, 1) k_tile(const TileArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_tot[2][T_NW];         // per-warp event totals (parity of the substep)
    __shared__ uint32_t s_flag[2][2];           // [parity][0 = a z re-check stored, 1 = a target is a hole]
    __shared__ int s_box[4];                    // hole bounding box of the substep (tile coordinates)
    __shared__ uint32_t s_count;
    __shared__ unsigned long long s_item, s_slab;

    const int zn = a.tw * a.th + (a.tw + 1) * (a.th + 1);
    volatile unsigned long long *z = reinterpret_cast<volatile unsigned long long *>(smem_raw);
    Pool pool;
    {
        unsigned char *p = smem_raw + (size_t)((zn + 1) & ~1) * 8;
        pool.pos = reinterpret_cast<uint32_t *>(p); p += 2 * T_CAP * 4;
        pool.dx = reinterpret_cast<float *>(p); p += 2 * T_CAP * 4;
        pool.dy = reinterpret_cast<float *>(p); p += 2 * T_CAP * 4;
        pool.zo = reinterpret_cast<float *>(p); p += 2 * T_CAP * 4;
        pool.zf = reinterpret_cast<float *>(p);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr unsigned FULL = 0xFFFFFFFFu;
    // arrival slab owned by this CTA: [cursor, slab_end); replicated in every thread (block-uniform)
    unsigned long long cursor = 0, slab_end = 0;
    uint32_t my_holes = 0;
    const uint32_t tiles_per_env = (uint32_t)(a.tiles_x * a.tiles_y);

    for (;;) {
        if (threadIdx.x == 0) s_item = atomicAdd(a.next_item, 1ull);
        __syncthreads();
        const unsigned long long item64 = s_item;
        if (item64 >= a.num_items) break;
        const uint32_t item = (uint32_t)item64;
        const int env = (int)(item / tiles_per_env);
        const uint32_t tile_id = item - (uint32_t)env * tiles_per_env;
        const int by = (int)(tile_id / (uint32_t)a.tiles_x), bx = (int)(tile_id - (uint32_t)by * a.tiles_x);

        TileGeo t;
        t.W = a.g.W; t.H = a.g.H;
        t.tw = a.tw; t.th = a.th;
        t.X0 = bx * a.tw; t.Y0 = by * a.th;
        t.RX0 = max(t.X0 - a.halo, 0); t.RY0 = max(t.Y0 - a.halo, 0);
        t.RW = min(t.X0 + a.tw + a.halo, t.W) - t.RX0;
        t.RH = min(t.Y0 + a.th + a.halo, t.H) - t.RY0;
        t.zc_off = a.tw * a.th; t.zc_w = a.tw + 1;
        const size_t eoff = (size_t)env * a.g.HW;
        const float *la = a.LA + eoff, *lb = a.LB + eoff;

        // my target pixels (lane-consecutive: conflict-free shared-memory access)
        int tx[T_TPT], ty[T_TPT], tp[T_TPT];
        bool in[T_TPT];
        float l_ref[T_TPT], l_prev[T_TPT];
#pragma unroll
        for (int j = 0; j < T_TPT; ++j) {
            const int tt = j * T_NT + threadIdx.x;
            ty[j] = tt / a.tw; tx[j] = tt - ty[j] * a.tw;
            in[j] = tt < t.zc_off && t.X0 + tx[j] < t.W && t.Y0 + ty[j] < t.H;
            tp[j] = (t.Y0 + ty[j]) * t.W + t.X0 + tx[j];
            l_ref[j] = l_prev[j] = 0.f;
            if (in[j]) { l_ref[j] = a.l_ref[eoff + tp[j]]; l_prev[j] = a.l_prev[eoff + tp[j]]; }
        }

        uint32_t flags = 0;
        int nB = stage(a, t, eoff, 0, pool, 0, &s_count, flags);
        if (a.force_direct) nB = T_CAP + 1;
        int nA = -1;
        // static tile: every candidate rests (zero displacement, ordinary depth).  Then each pixel of the
        // tile is reached by itself alone (single-pixel footprint, R14), at every substep: L_hat = L_B.
        const bool is_static = !__syncthreads_or((int)flags);

        for (int i = 1; i <= a.g.S; ++i) {
            const int par = i & 1;
            const float f = a.tab->f[i], g = a.tab->g[i];
            unsigned long long key[T_TPT];
            bool any_hole = false;
            if (is_static) {
#pragma unroll
                for (int j = 0; j < T_TPT; ++j) key[j] = in[j] ? (unsigned long long)(uint32_t)tp[j] : KEY_EMPTY;
            } else {
                for (int k = threadIdx.x; k < zn; k += T_NT) z[k] = KEY_EMPTY;
                if (threadIdx.x == 0) {
                    s_flag[par][0] = 0u; s_flag[par][1] = 0u;
                    s_box[0] = 0x7FFFFFFF; s_box[1] = 0x7FFFFFFF; s_box[2] = -1; s_box[3] = -1;
                }
                __syncthreads();
                bool fail = false;
                if (nB <= T_CAP) {
                    unsigned long long ck[T_CPT];
                    uint32_t ca[T_CPT];
                    const Box none = {0.f, 0.f, 0.f, 0.f};
                    splat_store<0>(z, pool, 0, nB, f, g, t, none, ck, ca);
                    __syncthreads();
                    fail = splat_check(z, ck, ca);
                    if (fail) s_flag[par][0] = 1u;
                    // gather optimistically: final unless some re-check stored (then redone below)
                    bool hole = false;
#pragma unroll
                    for (int j = 0; j < T_TPT; ++j) {
                        key[j] = in[j] ? tile_gather(z, t, tx[j], ty[j]) : 0ull;
                        hole |= key[j] == KEY_EMPTY;
                    }
                    if (hole) s_flag[par][1] = 1u;
                    __syncthreads();
                    if (s_flag[par][0]) {                       // rare: finish the fixed point, gather again
                        do { fail = splat_check(z, ck, ca); } while (__syncthreads_or(fail));
                        hole = false;
#pragma unroll
                        for (int j = 0; j < T_TPT; ++j) {
                            key[j] = in[j] ? tile_gather(z, t, tx[j], ty[j]) : 0ull;
                            hole |= key[j] == KEY_EMPTY;
                        }
                        any_hole = __syncthreads_or(hole) != 0;
                    } else any_hole = s_flag[par][1] != 0u;
                } else {
                    splat_direct<0>(z, a, t, eoff, f, g);
                    bool hole = false;
#pragma unroll
                    for (int j = 0; j < T_TPT; ++j) {
                        key[j] = in[j] ? tile_gather(z, t, tx[j], ty[j]) : 0ull;
                        hole |= key[j] == KEY_EMPTY;
                    }
                    any_hole = __syncthreads_or(hole) != 0;
                }
                if (any_hole) {                                 // A fills only B's holes
                    if (nA < 0) { nA = stage(a, t, eoff, 1, pool, T_CAP, &s_count, flags); if (a.force_direct) nA = T_CAP + 1; }
                    // bounding box of the holes (tile coordinates)
                    int hx0 = 0x7FFFFFFF, hy0 = 0x7FFFFFFF, hx1 = -1, hy1 = -1;
#pragma unroll
                    for (int j = 0; j < T_TPT; ++j)
                        if (in[j] && key[j] == KEY_EMPTY) {
                            hx0 = min(hx0, tx[j]); hx1 = max(hx1, tx[j]); hy0 = min(hy0, ty[j]); hy1 = max(hy1, ty[j]);
                        }
                    hx0 = __reduce_min_sync(FULL, hx0); hy0 = __reduce_min_sync(FULL, hy0);
                    hx1 = __reduce_max_sync(FULL, hx1); hy1 = __reduce_max_sync(FULL, hy1);
                    if (lane == 0 && hx1 >= 0) {
                        atomicMin(&s_box[0], hx0); atomicMin(&s_box[1], hy0); atomicMax(&s_box[2], hx1); atomicMax(&s_box[3], hy1);
                    }
                    __syncthreads();
                    if (nA <= T_CAP) {
                        // a source covers pixel h iff floor(q) is h-1 or h: q in [h-1, h+1)
                        const Box box = {(float)(t.X0 + s_box[0] - 1), (float)(t.Y0 + s_box[1] - 1),
                                         (float)(t.X0 + s_box[2] + 1), (float)(t.Y0 + s_box[3] + 1)};
                        unsigned long long ck[T_CPT];
                        uint32_t ca[T_CPT];
                        splat_store<1>(z, pool, T_CAP, nA, f, g, t, box, ck, ca);
                        do { __syncthreads(); fail = splat_check(z, ck, ca); } while (__syncthreads_or(fail));
                    } else splat_direct<1>(z, a, t, eoff, f, g);
#pragma unroll
                    for (int j = 0; j < T_TPT; ++j)
                        if (in[j] && key[j] == KEY_EMPTY) key[j] = tile_gather(z, t, tx[j], ty[j]);
                }
            }
            // composite (a5) + event model (a6)
            float l_hat[T_TPT], c[T_TPT];
            int n[T_TPT], pol[T_TPT], n_tot = 0;
#pragma unroll
            for (int j = 0; j < T_TPT; ++j) {
                n[j] = 0; pol[j] = 0; c[j] = 1.f; l_hat[j] = l_prev[j];
                if (!in[j]) continue;
                uint32_t widx = IDX_NONE;
                int wdir = 3;
                if (key[j] != KEY_EMPTY) {
                    widx = (uint32_t)key[j];
                    wdir = (int)(key[j] >> 63);
                    l_hat[j] = __ldg((wdir ? la : lb) + widx);
                } else ++my_holes;                            // R20: hold the previous value
                if (a.dbg.win) {
                    const size_t o = ((size_t)(i - 1) * a.g.E + env) * a.g.HW + tp[j];
                    a.dbg.win[o] = widx; a.dbg.dir[o] = (uint8_t)wdir; a.dbg.l_hat[o] = l_hat[j];
                }
                n[j] = event_count(l_hat[j], l_ref[j], a.ep.c_pos, a.ep.c_neg, pol[j], c[j]);   // Eq. 4
                n_tot += n[j];
            }
            // a8: per-warp totals -> one barrier -> offsets inside the (tile, substep) chunk
            const uint32_t wtot = (uint32_t)__reduce_add_sync(FULL, n_tot);
            if (lane == 0) s_tot[par][warp] = wtot;
            __syncthreads();
            uint32_t btot;
            const uint32_t wbase = warp_prefix<T_NW>(s_tot[par], btot);
            if (btot) {                                         // block-uniform
                if (cursor + btot > slab_end) {                 // block-uniform: take a new slab
                    const unsigned long long want = btot > (uint32_t)T_SLAB ? btot : (unsigned long long)T_SLAB;
                    if (threadIdx.x == 0) s_slab = atomicAdd(a.sink.alloc, want);
                    __syncthreads();
                    cursor = s_slab; slab_end = cursor + want;
                }
                unsigned long long off = cursor + wbase;
                if (threadIdx.x == 0) {
                    const uint32_t dir_index = ((uint32_t)env * a.g.S + (i - 1)) * tiles_per_env + tile_id;
                    a.sink.directory[dir_index] = make_uint2(cursor < 0xFFFFFFFFull ? (uint32_t)cursor : 0xFFFFFFFFu, btot);
                    atomicAdd(a.sink.counter, (unsigned long long)btot);
                }
                cursor += btot;
                if (wtot) {                                     // warp-uniform
#pragma unroll
                    for (int j = 0; j < T_TPT; ++j) {
                        off += warp_emit(a.sink, off, n[j], pol[j], c[j], l_ref[j], l_prev[j], l_hat[j],
                                         (uint32_t)(t.X0 + tx[j]) | ((uint32_t)(t.Y0 + ty[j]) << 16), env, i, a.ep);
                        if (n[j] > 0) l_ref[j] = __fmaf_rn((float)(pol[j] * n[j]), c[j], l_ref[j]);
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < T_TPT; ++j) l_prev[j] = l_hat[j];
            // static tile: once a substep is silent nothing changes any more (same L_hat, same L_ref)
            if (is_static && !btot && !a.dbg.win) break;
        }
#pragma unroll
        for (int j = 0; j < T_TPT; ++j)
            if (in[j]) { a.l_ref[eoff + tp[j]] = l_ref[j]; a.l_prev[eoff + tp[j]] = l_prev[j]; }
        __syncthreads();        // s_item, s_tot, the pool and z are reused by the next item
    }
    my_holes = __reduce_add_sync(FULL, my_holes);
    if (lane == 0 && my_holes) atomicAdd(a.holes, (unsigned long long)my_holes);
}

// ---- host side ----------------------------------------------------------------------------------------
static int tile_smem_bytes(int tw, int th)
{
    const int zn = tw * th + (tw + 1) * (th + 1);
    return ((zn + 1) & ~1) * 8 + 5 * 2 * T_CAP * 4;
}

bool plan_tile(const Geom &g, float max_motion_px, TilePlan *plan)
{
    if (g.mode != EVIS_COMPOSITE_B_PRIMARY) return false;      // blend needs both winners everywhere
    if (!(max_motion_px > 0.0f) || max_motion_px > 23.0f) return false;   // halo region too large to scan
    const int halo = (int)ceilf(max_motion_px) + 1;
    // equal tiles (no ragged last column), shrunk until the candidates of a uniformly translating scene
    // at the motion bound -- the tile swept by the motion, plus a one-pixel fringe -- fit the pool
    int nx = (g.W + T_MAX_TW - 1) / T_MAX_TW, ny = (g.H + T_MAX_TH - 1) / T_MAX_TH;
    for (;;) {
        plan->tw = (g.W + nx - 1) / nx;
        plan->th = (g.H + ny - 1) / ny;
        const float need = ((float)plan->tw + max_motion_px + 2.0f) * ((float)plan->th + max_motion_px + 2.0f);
        if (need <= (float)T_CAP || (plan->tw <= 16 && plan->th <= 16)) break;
        if (plan->tw >= plan->th) ++nx; else ++ny;
    }
    plan->tiles_x = (g.W + plan->tw - 1) / plan->tw;
    plan->tiles_y = (g.H + plan->th - 1) / plan->th;
    plan->halo = halo;
    plan->threads = T_NT;
    plan->cand_cap = T_CAP;
    plan->smem_bytes = tile_smem_bytes(plan->tw, plan->th);
    plan->slab = T_SLAB;
    const char *fd = getenv("EVIS_TILE_FORCE_DIRECT");
    plan->force_direct = fd && fd[0] == '1';
    return true;
}

cudaError_t tile_setup(const Geom &, TilePlan &plan, int device)
{
    cudaError_t e = cudaFuncSetAttribute(k_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.smem_bytes);
    if (e != cudaSuccess) return e;
    int sms = 0, per_sm = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_tile, T_NT, plan.smem_bytes);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    plan.ctas = sms * per_sm;                       // persistent: every CTA is resident
    return cudaSuccess;
}

cudaError_t launch_tile(const Geom &g, const TilePlan &plan, const Keyframe &A, const Keyframe &B,
                        const SubstepTable *tab, float *l_ref, float *l_prev, const EventParams &ep,
                        const EventSink &sink, unsigned long long *holes, unsigned long long *next_item,
                        const DebugOut &dbg, cudaStream_t st)
{
    TileArgs a;
    a.g = g;
    a.tw = plan.tw; a.th = plan.th; a.halo = plan.halo; a.tiles_x = plan.tiles_x; a.tiles_y = plan.tiles_y;
    a.force_direct = plan.force_direct;
    a.num_items = (uint32_t)g.E * (uint32_t)plan.tiles_x * (uint32_t)plan.tiles_y;
    a.next_item = next_item;
    a.LA = A.L; a.LB = B.L; a.ZA = A.Z; a.ZB = B.Z;
    a.mvA = A.mv; a.fwdA = A.has_fwd ? A.fwd : nullptr; a.mvB = B.mv;
    a.tab = tab; a.l_ref = l_ref; a.l_prev = l_prev; a.ep = ep; a.sink = sink; a.holes = holes; a.dbg = dbg;
    const unsigned grid = a.num_items < (uint32_t)plan.ctas ? a.num_items : (uint32_t)plan.ctas;
    k_tile<<<grid, T_NT, plan.smem_bytes, st>>>(a);
    return cudaGetLastError();
}

}  // namespace evis
