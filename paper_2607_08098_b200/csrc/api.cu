// api.cu -- the C ABI of include/evis.h: context, argument checks, launch sequencing.
// No step of the path runs on the host: this file only allocates, validates and enqueues kernels.
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "kernels.h"

using namespace evis;

static_assert(sizeof(evis_event) == 16, "evis_event is a 16-byte record");
static_assert(sizeof(evis_config) == 64 && sizeof(evis_info) == 80, "ABI struct layout (binding.py mirrors it)");

struct evis_ctx {
    evis_config cfg;
    Geom g;
    cudaStream_t own_stream;          // evis_step_host, state/debug copies
    cudaStream_t last_stream;
    int last_cuda;

    Keyframe kf[3];                   // three, so that the prep of step k + 1 can overwrite the oldest while the chunk
                                      // kernels of step k still read the other two
    int cur;                          // kf[cur] receives the next keyframe; kf[(cur + 2) % 3] is A
    float *l_ref, *l_prev;
    float *th_on, *th_off;            // Eq. 8 maps [E*H*W] (owned), in force when th_active
    bool th_active;
    evis_noise noise; bool noise_on;  // noise events (Eq. 9-10), parameters as given
    unsigned char *hot;               // hot-pixel set [E*H*W] (owned) or null
    int channel; bool channel_set;    // colour events: log of one channel instead of the luminance
    float *t_last;                    // refractory state [E*H*W] (owned), in force when tau_r > 0
    float tau_r;
    SubstepTable *tab;                // device
    SubstepTable h_tab;               // host copy (kernel parameter of the global path)
    EventParams ep;

    // global path z-buffers
    // nreg regions of zmem_bytes each; region r serves the env chunks c with c % nreg == r, on its own
    // stream when nreg > 1, so that several chunks small enough for the L2 are in flight together
    static constexpr int MAX_REG = 8;
    unsigned long long *zmem;         // one allocation: nreg * zmem_bytes
    size_t zmem_bytes;                // one region (a multiple of 256 bytes)
    int nreg;
    int chunk_ne, chunk_ni, nset;
    alignas(64) unsigned char tmap_d[MAX_REG][TMAP_BYTES], tmap_c[MAX_REG][TMAP_BYTES];   // CUtensorMap of zd / zc per region
    bool have_tmap;
    int idx_bits;                     // 24: tagged keys (H*W <= 2^24), 32: untagged
    int ztag[MAX_REG];                // tag of the region's last chunk; 0 or less: the region must be cleared
    cudaStream_t reg_stream[MAX_REG];
    cudaEvent_t ev_fork, ev_join[MAX_REG];

    // event stream
    // The order stage of step k runs on `ord_stream` while the chunk phase of step k + 1 runs on the caller's
    // stream (it is bound by HBM, the chunk phase by instruction issue), so the buffers the two share are doubled:
    // slot = step & 1 (slot 1 aliases slot 0 when EVIS_NO_OVERLAP=1).  `ordered`, `bsum` and the sticky counters
    // are touched by the order stream only.
    uint4 *arrival, *ordered;         // arrival = slot 0
    uint2 *directory;                 // slot 0
    uint4 *arrival_s[2];
    uint2 *directory_s[2];
    unsigned long long *counters_s[2];
    cudaStream_t ord_stream;
    cudaStream_t copy_stream;         // evis_read_events_begin: device -> host copy of the ordered stream
    cudaEvent_t ev_copy;
    bool copy_pending;
    // `ordered` is doubled like the arrival buffers (slot = step & 1; one buffer without the overlap), so that the order
    // stage of step k + 1 does not wait for step k's stream to be copied out.  copy_slot: the slot the pending copy
    // reads (-1: the voxel image).  h_copy (pinned): [0], [1] = events copied and overflow code of the deferred read;
    // from H_SLOT + slot * H_SLOT_WORDS on, a mirror of each slot's per-step counters C_EVENTS .. C_ALLOC (the deferred read
    // of the step before the last needs that step's counts while h_counters already belongs to the last step).
    uint4 *ordered_s[2];
    int copy_slot;
    bool deferred;
    unsigned long long *h_copy;
    static constexpr int H_SLOT = 8, H_SLOT_WORDS = 40;
    cudaEvent_t ev_chunks[2], ev_order[2];
    bool ord_pending[2];
    bool overlap;
    int last_slot;
    uint32_t dir_entries;
    unsigned long long *bsum;
    // device counters.  Reset every step: [0] events, [1] holes, [2] arrival slots handed out,
    // [3] unused.  Sticky: [4] motion-bound violations, [5] events over all steps.
    unsigned long long *counters;
    unsigned long long *h_counters;   // pinned host mirror
    unsigned long long arrival_cap;   // slots of the arrival buffer (capacity + slab slack)
    DebugOut dbg;

    // defocus (evis_set_defocus, R31): taps, the keyframes' linear intensity (one allocation, A and B
    // alternate like kf[].L), the carried unblurred frame and the warped linear frames of one chunk per region
    bool defocus;
    BlurTaps taps;
    float *lin[3];
    float *i_prev;
    float *frames;                    // nreg regions of frames_elems floats
    size_t frames_elems;

    // weighted front-surface splat (composite mode 2, R32): per region the front depth and the sums of one chunk
    uint32_t *zfront;
    long long *wacc;
    size_t wchunk_elems;              // chunk_ne * chunk_ni * HW

    bool graph_mode;                  // EVIS_GRAPH=1 (measurement hook): every step is captured and launched as one CUDA graph
    bool compact;                     // evis_set_compact_events: the stored stream holds 8-byte events

    // time-sorted stream (evis_set_time_sorted): workspace of the segmented radix sort
    bool time_sorted;
    void *sort_ws;
    size_t sort_ws_bytes;

    // voxel grid (evis_set_voxels): V in 32.32 fixed point, its float32 image for the read calls
    bool vox_on, vox_restart;
    evis_voxel_config vox;
    unsigned long long *vox_v;
    float *vox_out;
    uint32_t vox_j;                   // intervals accumulated in the current window
    size_t vox_cells;                 // E * 2 * bins * H' * W'

    // host-buffer entry point staging
    // two staging sets: the keyframe of step k + 1 goes up (up_stream) while step k computes (own_stream)
    float *st_rad[2], *st_mv[2], *st_fwd[2], *st_depth[2];
    cudaStream_t up_stream;
    cudaEvent_t ev_up[2], ev_used[2];     // set uploaded / the step that read the set has been enqueued and has run
    bool set_used[2];
    uint64_t host_steps;

    uint64_t steps, launches, device_bytes;
    uint32_t kf_next;                 // index the next closed interval gets (evis_set_interval_index)
    uint32_t env_offset;              // index of this context's env 0 in the whole batch (evis_set_env_offset): noise keys
    uint64_t last_events, last_holes;
    int last_overflow, last_motion;
    bool have_events;

    // stage timing (evis_profile_*)
    bool prof_on;
    struct ProfSpan { int stage; cudaEvent_t a, b; };
    std::vector<ProfSpan> prof_spans;     // recorded, not yet read
    std::vector<cudaEvent_t> prof_free;   // event pool
    evis_profile prof_acc;
};

namespace {

// Device counters, one per 128-byte line: the arrival reservation (C_ALLOC) is on every resolve block's critical
// path and must not queue behind the event / hole tallies in the same L2 sector.  [0, C_STEP_END) are reset
// every step; C_MOTION, C_TOTAL and C_OVERFLOW (steps whose events did not all fit) are sticky.
enum { C_EVENTS = 0, C_HOLES = 16, C_ALLOC = 32, C_ITEM = 48, C_STEP_END = 64, C_MOTION = 64, C_TOTAL = 80, C_OVERFLOW = 96, NCOUNTERS = 112 };

struct DeviceGuard {
    int prev;
    bool ok;
    explicit DeviceGuard(int dev) : prev(-1), ok(true)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

#define CU(call)                                                        \
    do {                                                                \
        cudaError_t e_ = (call);                                        \
        if (e_ != cudaSuccess) {                                        \
            ctx->last_cuda = (int)e_;                                   \
            cudaGetLastError();                                         \
            return e_ == cudaErrorMemoryAllocation ? EVIS_ERR_OOM : EVIS_ERR_CUDA; \
        }                                                               \
    } while (0)

template <typename T>
cudaError_t dalloc(evis_ctx *ctx, T **p, size_t count)
{
    const size_t bytes = count * sizeof(T);
    cudaError_t e = cudaMalloc((void **)p, bytes ? bytes : 1);
    if (e == cudaSuccess) ctx->device_bytes += bytes;
    return e;
}

cudaEvent_t prof_event(evis_ctx *ctx)
{
    cudaEvent_t e = nullptr;
    if (!ctx->prof_free.empty()) { e = ctx->prof_free.back(); ctx->prof_free.pop_back(); }
    else if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return e;
}

// drain recorded spans into the accumulators (synchronises on the spans' events)
void prof_drain(evis_ctx *ctx)
{
    for (auto &sp : ctx->prof_spans) {
        float ms = 0.f;
        if (cudaEventSynchronize(sp.b) == cudaSuccess && cudaEventElapsedTime(&ms, sp.a, sp.b) == cudaSuccess)
            ctx->prof_acc.ms[sp.stage] += (double)ms;
        else cudaGetLastError();
        ctx->prof_free.push_back(sp.a);
        ctx->prof_free.push_back(sp.b);
    }
    ctx->prof_spans.clear();
}

// RAII span: records an event pair around the launches of one stage when profiling is on
struct Span {
    evis_ctx *ctx; cudaStream_t st; int stage; cudaEvent_t a;
    Span(evis_ctx *c, cudaStream_t s, int stg, int launches, bool timed = true) : ctx(c), st(s), stage(stg), a(nullptr)
    {
        ctx->launches += launches;
        if (!ctx->prof_on || !timed) return;
        ctx->prof_acc.launches[stage] += launches;
        a = prof_event(ctx);
        if (a) cudaEventRecord(a, st);
    }
    ~Span()
    {
        if (!a) return;
        cudaEvent_t b = prof_event(ctx);
        if (!b) { ctx->prof_free.push_back(a); return; }
        cudaEventRecord(b, st);
        ctx->prof_spans.push_back({stage, a, b});
    }
};

unsigned long long host_mix64(unsigned long long z)      // splitmix64 output function (R29)
{
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}

size_t env_size_mb(const char *name, size_t dflt)
{
    const char *v = getenv(name);
    if (!v || !*v) return dflt;
    const long long x = atoll(v);
    return x > 0 ? (size_t)x : dflt;
}

void free_all(evis_ctx *ctx)
{
    for (int k = 0; k < 3; ++k) {
        if (k == 0) cudaFree(ctx->kf[k].L);
        cudaFree(ctx->kf[k].mv); cudaFree(ctx->kf[k].fwd); cudaFree(ctx->kf[k].Z);
    }
    cudaFree(ctx->l_ref); cudaFree(ctx->l_prev); cudaFree(ctx->th_on); cudaFree(ctx->th_off); cudaFree(ctx->t_last); cudaFree(ctx->hot); cudaFree(ctx->tab); cudaFree(ctx->zmem);
    cudaFree(ctx->arrival); cudaFree(ctx->ordered); cudaFree(ctx->directory); cudaFree(ctx->bsum);
    cudaFree(ctx->counters); cudaFree(ctx->dbg.win); cudaFree(ctx->dbg.dir); cudaFree(ctx->dbg.l_hat);
    cudaFree(ctx->vox_v); cudaFree(ctx->vox_out); cudaFree(ctx->sort_ws);
    cudaFree(ctx->lin[0]); cudaFree(ctx->i_prev); cudaFree(ctx->frames);
    cudaFree(ctx->zfront); cudaFree(ctx->wacc);
    for (int k = 0; k < 2; ++k) {
        cudaFree(ctx->st_rad[k]); cudaFree(ctx->st_mv[k]); cudaFree(ctx->st_fwd[k]); cudaFree(ctx->st_depth[k]);
        if (ctx->ev_up[k]) cudaEventDestroy(ctx->ev_up[k]);
        if (ctx->ev_used[k]) cudaEventDestroy(ctx->ev_used[k]);
    }
    if (ctx->up_stream) cudaStreamDestroy(ctx->up_stream);
    if (ctx->h_counters) cudaFreeHost(ctx->h_counters);
    prof_drain(ctx);
    for (cudaEvent_t e : ctx->prof_free) cudaEventDestroy(e);
    ctx->prof_free.clear();
    if (ctx->arrival_s[1] != ctx->arrival_s[0]) {
        cudaFree(ctx->arrival_s[1]); cudaFree(ctx->directory_s[1]); cudaFree(ctx->counters_s[1]);
    }
    if (ctx->ordered_s[1] != ctx->ordered_s[0]) cudaFree(ctx->ordered_s[1]);
    if (ctx->h_copy) cudaFreeHost(ctx->h_copy);
    if (ctx->ord_stream) cudaStreamDestroy(ctx->ord_stream);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->ev_copy) cudaEventDestroy(ctx->ev_copy);
    for (int k = 0; k < 2; ++k) {
        if (ctx->ev_chunks[k]) cudaEventDestroy(ctx->ev_chunks[k]);
        if (ctx->ev_order[k]) cudaEventDestroy(ctx->ev_order[k]);
    }
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    for (int r = 0; r < evis_ctx::MAX_REG; ++r) {
        if (ctx->reg_stream[r]) cudaStreamDestroy(ctx->reg_stream[r]);
        if (ctx->ev_join[r]) cudaEventDestroy(ctx->ev_join[r]);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
}

int create_impl(evis_ctx *ctx)
{
    const evis_config &c = ctx->cfg;
    Geom &g = ctx->g;
    g.E = c.num_envs; g.H = c.height; g.W = c.width; g.S = c.substeps;
    g.HW = c.height * c.width;
    g.Wp = (c.width + 2) & ~1; g.HWp = (c.height + 1) * g.Wp;
    g.mode = c.composite_mode;
    const size_t P = (size_t)g.E * g.HW;
    if (P >= ((size_t)1 << 31)) return EVIS_ERR_INVALID_ARG;    // the kernels keep pixel offsets between planes in 32 bits

    CU(cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking));
    // the L planes share one allocation: the resolve kernel addresses the winner's value from one base
    CU(dalloc(ctx, &ctx->kf[0].L, 3 * P));
    ctx->kf[1].L = ctx->kf[0].L + P;
    ctx->kf[2].L = ctx->kf[0].L + 2 * P;
    for (int k = 0; k < 3; ++k) {
        CU(dalloc(ctx, &ctx->kf[k].mv, P));
        CU(dalloc(ctx, &ctx->kf[k].Z, P));
    }
    CU(dalloc(ctx, &ctx->l_ref, P));
    CU(dalloc(ctx, &ctx->l_prev, P));

    // substep weights f_i = i/S, g_i = 1 - f_i in IEEE binary32 (same expression as the paper's f = i/K)
    SubstepTable &h = ctx->h_tab;
    memset(&h, 0, sizeof h);
    for (int i = 0; i <= g.S; ++i) {
        volatile float f = (float)i / (float)g.S;
        volatile float gg = 1.0f - f;
        h.f[i] = f; h.g[i] = gg;
    }
    CU(dalloc(ctx, &ctx->tab, 1));
    CU(cudaMemcpy(ctx->tab, &h, sizeof h, cudaMemcpyHostToDevice));
    volatile float dt = c.keyframe_dt / (float)g.S;
    ctx->ep.c_pos = c.c_pos; ctx->ep.c_neg = c.c_neg; ctx->ep.dt = dt; ctx->ep.kf = 0;

    ctx->nset = g.mode == EVIS_COMPOSITE_BLEND ? 2 : 1;
    uint32_t tiles_x, tiles_y;
    {
        // chunk = envs x substeps whose z-buffers fit one region's budget.  Defaults (measured on B200, DESIGN.md
        // Sec. 6): 4 regions on 4 streams; 24 MiB regions when one env's S substeps fit (the live keys stay in the
        // L2 and small grids overlap across streams), else 512 MiB / regions (substep chunks re-read the sources and carry
        // L_ref / L_prev through memory, so they should be long); an env whose whole interval does not even fit that
        // share (cfg 3: 488 MB) gets 2 regions of 256 MiB (cfg 3: 17.8 -> 16.4 ms).  EVIS_ZBUF_MB / EVIS_STREAMS override.
        const size_t unit = (size_t)ctx->nset * 8u * 2u * (size_t)g.HWp;
        const bool huge = unit * g.S > ((size_t)128 << 20);
        const size_t default_regions = huge ? 2 : 4;
        const size_t share = (size_t)512 / ((size_t)g.E < default_regions ? (size_t)g.E : default_regions);   // of 512 MiB
        size_t budget = env_size_mb("EVIS_ZBUF_MB", unit * g.S <= ((size_t)24 << 20) ? 24 : share) << 20;
        if (budget > ((size_t)8 << 30)) budget = (size_t)8 << 30;    // the kernels index a chunk with 32-bit offsets
        if (unit * g.S <= budget) {
            ctx->chunk_ni = g.S;
            size_t ne = budget / (unit * g.S);
            ctx->chunk_ne = (int)(ne > (size_t)g.E ? g.E : ne);
        } else {
            ctx->chunk_ne = 1;
            size_t ni = budget / unit;
            ctx->chunk_ni = (int)(ni < 1 ? 1 : (ni > (size_t)g.S ? g.S : ni));
        }
        {   // experiment hooks: explicit chunk shape
            const size_t ni = env_size_mb("EVIS_CHUNK_NI", 0), ne = env_size_mb("EVIS_CHUNK_NE", 0);
            if (ni) ctx->chunk_ni = (int)(ni > (size_t)g.S ? g.S : ni);
            if (ne) ctx->chunk_ne = (int)(ne > (size_t)g.E ? g.E : ne);
            else if (ni) {
                size_t n2 = budget / (unit * ctx->chunk_ni);
                ctx->chunk_ne = (int)(n2 < 1 ? 1 : (n2 > (size_t)g.E ? g.E : n2));
            }
        }
        ctx->zmem_bytes = (unit * ctx->chunk_ne * ctx->chunk_ni + 255) & ~(size_t)255;
        {   // concurrent regions (EVIS_STREAMS): never more than there are env chunks
            const size_t nchunks = ((size_t)g.E + ctx->chunk_ne - 1) / ctx->chunk_ne;
            size_t nr = env_size_mb("EVIS_STREAMS", default_regions);
            if (nr > (size_t)evis_ctx::MAX_REG) nr = evis_ctx::MAX_REG;
            if (nr > nchunks) nr = nchunks;
            ctx->nreg = (int)(nr < 1 ? 1 : nr);
        }
        const char *nt = getenv("EVIS_NO_ZTAG");                      // test hook: force untagged keys
        ctx->idx_bits = (g.HW <= (1 << 24) && !(nt && nt[0] == '1')) ? 24 : 32;
        CU(cudaMalloc((void **)&ctx->zmem, ctx->zmem_bytes * ctx->nreg));
        ctx->device_bytes += ctx->zmem_bytes * ctx->nreg;
        {
            const size_t planes = (size_t)ctx->nset * ctx->chunk_ni * ctx->chunk_ne;
            const char *nt2 = getenv("EVIS_NO_TMA");                  // test hook: direct loads in the resolve kernel
            ctx->have_tmap = !(nt2 && nt2[0] == '1');
            for (int r = 0; r < ctx->nreg; ++r) {
                unsigned long long *zr = ctx->zmem + (size_t)r * (ctx->zmem_bytes / 8);
                ctx->ztag[r] = 0;
                if (ctx->have_tmap && !make_z_tensor_maps(g, zr, zr + planes * g.HWp, planes, ctx->tmap_d[r], ctx->tmap_c[r]))
                    ctx->have_tmap = false;
            }
        }
        if (ctx->nreg > 1) {
            CU(cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming));
            for (int r = 0; r < ctx->nreg; ++r) {
                CU(cudaStreamCreateWithFlags(&ctx->reg_stream[r], cudaStreamNonBlocking));
                CU(cudaEventCreateWithFlags(&ctx->ev_join[r], cudaEventDisableTiming));
            }
        }
        tiles_x = (g.W + G_TILE_W - 1) / G_TILE_W;
        tiles_y = (g.H + G_TILE_H - 1) / G_TILE_H;
    }
    const unsigned long long ent = (unsigned long long)g.E * g.S * tiles_x * tiles_y;
    if (ent >= 0xFFFFFFFFull) return EVIS_ERR_INVALID_ARG;
    ctx->dir_entries = (uint32_t)ent;
    CU(dalloc(ctx, &ctx->directory, (size_t)ent));
    CU(dalloc(ctx, &ctx->bsum, (size_t)(ent / ORDER_ENTRIES_PER_BLOCK + 2)));
    // arrival buffer: the chunks of records (or events, in direct mode) are packed densely
    ctx->arrival_cap = c.event_capacity;
    if (ctx->arrival_cap > 0xFFFFFFF0ull) ctx->arrival_cap = 0xFFFFFFF0ull;
    CU(dalloc(ctx, &ctx->arrival, (size_t)ctx->arrival_cap));
    CU(dalloc(ctx, &ctx->ordered, (size_t)c.event_capacity));
    CU(dalloc(ctx, &ctx->counters, NCOUNTERS));
    CU(cudaMemset(ctx->counters, 0, NCOUNTERS * sizeof(unsigned long long)));
    CU(cudaHostAlloc((void **)&ctx->h_counters, NCOUNTERS * sizeof(unsigned long long), cudaHostAllocDefault));
    memset(ctx->h_counters, 0, NCOUNTERS * sizeof(unsigned long long));
    {
        const char *gm = getenv("EVIS_GRAPH");
        ctx->graph_mode = gm && gm[0] == '1';
        const char *no = getenv("EVIS_NO_OVERLAP");       // test hook: order stage serialised with the next step
        ctx->overlap = !(no && no[0] == '1');
        ctx->arrival_s[0] = ctx->arrival; ctx->directory_s[0] = ctx->directory; ctx->counters_s[0] = ctx->counters;
        ctx->arrival_s[1] = ctx->arrival; ctx->directory_s[1] = ctx->directory; ctx->counters_s[1] = ctx->counters;
        ctx->ordered_s[0] = ctx->ordered_s[1] = ctx->ordered;
        if (ctx->overlap) CU(dalloc(ctx, &ctx->ordered_s[1], (size_t)c.event_capacity));
        ctx->copy_slot = -1;
        CU(cudaHostAlloc((void **)&ctx->h_copy, (evis_ctx::H_SLOT + 2 * evis_ctx::H_SLOT_WORDS) * sizeof(unsigned long long), cudaHostAllocDefault));
        memset(ctx->h_copy, 0, (evis_ctx::H_SLOT + 2 * evis_ctx::H_SLOT_WORDS) * sizeof(unsigned long long));
        if (ctx->overlap) {
            CU(dalloc(ctx, &ctx->arrival_s[1], (size_t)ctx->arrival_cap));
            CU(dalloc(ctx, &ctx->directory_s[1], (size_t)ent));
            CU(dalloc(ctx, &ctx->counters_s[1], NCOUNTERS));
            CU(cudaMemset(ctx->counters_s[1], 0, NCOUNTERS * sizeof(unsigned long long)));
        }
        CU(cudaStreamCreateWithFlags(&ctx->ord_stream, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        CU(cudaEventCreateWithFlags(&ctx->ev_copy, cudaEventDisableTiming));
        for (int k = 0; k < 2; ++k) {
            CU(cudaEventCreateWithFlags(&ctx->ev_chunks[k], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&ctx->ev_order[k], cudaEventDisableTiming));
        }
    }
    if (g.mode == EVIS_COMPOSITE_WEIGHTED) {
        ctx->wchunk_elems = (size_t)ctx->chunk_ne * ctx->chunk_ni * g.HW;
        CU(dalloc(ctx, &ctx->zfront, ctx->wchunk_elems * ctx->nreg));
        CU(dalloc(ctx, &ctx->wacc, 2 * ctx->wchunk_elems * ctx->nreg));
    }
    if (c.debug_capture) {
        CU(dalloc(ctx, &ctx->dbg.win, P * g.S));
        CU(dalloc(ctx, &ctx->dbg.dir, P * g.S));
        CU(dalloc(ctx, &ctx->dbg.l_hat, P * g.S));
    }
    return EVIS_OK;
}

// everything this context has enqueued: the caller's stream of the last step, then the order stream
cudaError_t sync_all(evis_ctx *ctx)
{
    cudaError_t e = cudaSuccess;
    if (ctx->last_stream || ctx->steps) e = cudaStreamSynchronize(ctx->last_stream);
    if (e == cudaSuccess && ctx->ord_stream) e = cudaStreamSynchronize(ctx->ord_stream);
    return e;
}

int fetch_counters(evis_ctx *ctx)
{
    CU(sync_all(ctx));
    ctx->last_events = ctx->h_counters[C_EVENTS];
    ctx->last_holes = ctx->h_counters[C_HOLES];
    ctx->last_motion = ctx->h_counters[C_MOTION] != 0;
    // 2: records were dropped in arrival order, the stored stream has gaps and is unusable; 1: a valid prefix is stored
    ctx->last_overflow = ctx->h_counters[C_ALLOC] > ctx->arrival_cap ? 2 : (ctx->last_events > ctx->cfg.event_capacity ? 1 : 0);
    return EVIS_OK;
}

// Events of the last step that the ordered stream validly holds (after fetch_counters): all of them; the first
// event_capacity when there were more (a true prefix of the deterministic order); none when the ARRIVAL buffer
// overflowed -- records were then dropped in scheduling order and the ordered stream has gaps.
uint64_t stored_events(const evis_ctx *ctx)
{
    if (ctx->last_overflow == 2) return 0;
    return ctx->last_events < ctx->cfg.event_capacity ? ctx->last_events : ctx->cfg.event_capacity;
}

}  // namespace

extern "C" {

const char *evis_version(void) { return "evis-b200 0.1 (sm_100a)"; }

const char *evis_strerror(int s)
{
    switch (s) {
        case EVIS_OK: return "ok";
        case EVIS_ERR_INVALID_ARG: return "invalid argument";
        case EVIS_ERR_CUDA: return "CUDA error";
        case EVIS_ERR_OOM: return "out of device memory";
        case EVIS_ERR_OVERFLOW: return "event capacity exceeded";
        case EVIS_ERR_MOTION_BOUND: return "motion vector exceeds max_motion_px";
        case EVIS_ERR_BAD_STATE: return "call order violated";
        case EVIS_ERR_TOO_LARGE: return "grid larger than the fixed accumulator of evis_voxelize_static";
        default: return "unknown status";
    }
}

int evis_last_cuda_error(const evis_ctx *ctx) { return ctx ? ctx->last_cuda : 0; }

int evis_create(const evis_config *cfg, evis_ctx **out)
{
    if (!cfg || !out) return EVIS_ERR_INVALID_ARG;
    if (cfg->num_envs <= 0 || cfg->num_envs > 65535 || cfg->height <= 0 || cfg->height > 32767 ||
        cfg->width <= 0 || cfg->width > 32767 || cfg->substeps < 1 || cfg->substeps > 255)
        return EVIS_ERR_INVALID_ARG;
    if (!(cfg->c_pos > 0.0f) || !(cfg->c_neg > 0.0f) || !(cfg->log_eps > 0.0f) || !(cfg->keyframe_dt > 0.0f))
        return EVIS_ERR_INVALID_ARG;
    if (!(cfg->max_motion_px >= 0.0f)) return EVIS_ERR_INVALID_ARG;
    if (cfg->composite_mode != EVIS_COMPOSITE_B_PRIMARY && cfg->composite_mode != EVIS_COMPOSITE_BLEND &&
        cfg->composite_mode != EVIS_COMPOSITE_WEIGHTED)
        return EVIS_ERR_INVALID_ARG;
    if (cfg->path != EVIS_PATH_AUTO && cfg->path != EVIS_PATH_GLOBAL) return EVIS_ERR_INVALID_ARG;
    if (cfg->event_capacity == 0 || cfg->event_capacity > 0x7FFFFFFFull) return EVIS_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess) { cudaGetLastError(); return EVIS_ERR_CUDA; }
    if (cfg->device < 0 || cfg->device >= ndev) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(cfg->device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    evis_ctx *ctx = new (std::nothrow) evis_ctx();     // value-initialised: every POD member is zero
    if (!ctx) return EVIS_ERR_OOM;
    ctx->cfg = *cfg;
    const int rc = create_impl(ctx);
    if (rc != EVIS_OK) { free_all(ctx); delete ctx; return rc; }
    *out = ctx;
    return EVIS_OK;
}

int evis_destroy(evis_ctx *ctx)
{
    if (!ctx) return EVIS_OK;
    DeviceGuard guard(ctx->cfg.device);
    cudaDeviceSynchronize();
    free_all(ctx);
    delete ctx;
    return EVIS_OK;
}

// Everything evis_step enqueues.  capturing: `st` is being captured into a CUDA graph (EVIS_GRAPH=1, a measurement
// hook: ncu can then profile the whole step as ONE workload in its real multi-stream schedule): every stream the
// step forks must join `st` again before the capture ends.
static int step_enqueue(evis_ctx *ctx, const float *rad, const float *mv_bwd, const float *mv_fwd, const float *depth,
                        cudaStream_t st, bool capturing)
{
    const Geom &g = ctx->g;
    const size_t P = (size_t)g.E * g.HW;
    Keyframe &B = ctx->kf[ctx->cur];
    const int ia = (ctx->cur + 2) % 3;
    const Keyframe &A = ctx->kf[ia];

    if (mv_fwd && !B.fwd) {               // forward fields are optional: allocate on first use
        for (int k = 0; k < 3; ++k) CU(dalloc(ctx, &ctx->kf[k].fwd, P));
    }
    B.has_fwd = mv_fwd != nullptr;
    const bool first = ctx->steps == 0;
    if (ctx->prof_on) { ctx->prof_acc.steps += 1; if (ctx->prof_spans.size() > 8192) prof_drain(ctx); }
    // slot of this step's arrival buffer, directory and per-step counters; the order stage that used it last
    // (two steps ago with overlap, the last step without) must be done before it is cleared.  The same wait guards the
    // keyframe buffers, so it comes BEFORE the prep: kf[cur] was keyframe A of the step two steps ago, whose chunk kernels
    // run on the regions' streams and are not joined to `st`; that step's order stage started after them, so once it is
    // done nothing reads kf[cur] (or lin[cur]) any more.  The prep of step k + 1 still runs under step k's chunk kernels.
    const int sl = ctx->overlap ? (int)(ctx->steps & 1) : 0;
    if (ctx->ord_pending[sl]) CU(cudaStreamWaitEvent(st, ctx->ev_order[sl], 0));
    {
        Span sp(ctx, st, EVIS_STAGE_PREP, 1);
        CU(launch_prep(rad, mv_bwd, mv_fwd, depth, (long long)P, ctx->cfg.log_eps, ctx->channel_set ? ctx->channel : -1, B.L, B.mv, B.fwd, B.Z,
                       first ? ctx->l_ref : nullptr, first ? ctx->l_prev : nullptr,
                       ctx->cfg.max_motion_px, ctx->counters + C_MOTION, ctx->defocus ? ctx->lin[ctx->cur] : nullptr, st));
        if (ctx->defocus && first) {
            // the event model's first frame is the blurred keyframe too; the carried unblurred frame is the keyframe
            CU(launch_blur_log(ctx->lin[ctx->cur], g.E, g.H, g.W, ctx->taps, ctx->cfg.log_eps, ctx->l_ref, ctx->l_prev, st));
            CU(cudaMemcpyAsync(ctx->i_prev, ctx->lin[ctx->cur], P * sizeof(float), cudaMemcpyDeviceToDevice, st));
            ctx->launches += 2;
        }
    }
    ctx->last_stream = st;
    if (first) {
        ctx->h_counters[C_EVENTS] = ctx->h_counters[C_HOLES] = ctx->h_counters[C_ALLOC] = 0;
        ctx->steps = 1;
        ctx->cur = (ctx->cur + 1) % 3;
        ctx->have_events = true;
        return EVIS_OK;
    }

    ctx->ep.kf = ctx->kf_next;
    unsigned long long *cnt = ctx->counters_s[sl];
    EventSink sink{ctx->arrival_s[sl], ctx->arrival_cap, cnt + C_ALLOC, cnt + C_EVENTS, ctx->directory_s[sl]};
    const Thresholds th{ctx->th_active ? ctx->th_on : nullptr, ctx->th_active ? ctx->th_off : nullptr};
    // direct mode (the resolve kernel writes events) serves the refractory period and the noise events
    Refractory rf{};
    rf.t_last = (ctx->tau_r > 0.0f || ctx->noise_on) ? ctx->t_last : nullptr;
    rf.tau_r = ctx->tau_r;
    rf.T = ctx->cfg.keyframe_dt;
    if (ctx->noise_on) {
        // P = r dt, binary32 products of the rates and T / S (R29); the per-step part of the generator keys
        volatile float pl = ctx->noise.r_leak * ctx->ep.dt, ps = ctx->noise.r_shot * ctx->ep.dt, ph = ctx->noise.r_hot * ctx->ep.dt;
        rf.noise_on = 1;
        // the kernel keys env e of this context with mix64(noise_key + e): a shard's first env sits at env_offset of the batch
        rf.noise_key = host_mix64(ctx->noise.seed ^ (0x9E3779B97F4A7C15ull * ((unsigned long long)ctx->ep.kf + 1ull))) +
                       (unsigned long long)ctx->env_offset;
        rf.p_leak = pl; rf.p_shot = ps; rf.p_hot = ph;
        rf.i_white = ctx->noise.i_white;
        rf.eps = ctx->cfg.log_eps;
        rf.hot = ctx->hot;
    }
    {
        Span sp(ctx, st, EVIS_STAGE_CLEAR, 2);
        CU(cudaMemsetAsync(cnt, 0, C_STEP_END * sizeof(unsigned long long), st));   // the per-step counters
        CU(cudaMemsetAsync(sink.directory, 0, (size_t)ctx->dir_entries * sizeof(uint2), st));
    }

    // The regions' streams do NOT join `st` again (unless the stage timers are on or EVIS_NO_OVERLAP=1): the order stream
    // waits for them instead, and every call that returns results waits for the order stream.  `st` is then free to run
    // the NEXT step's prep (HBM-bound, into the third keyframe buffer) under this step's chunk kernels; it cannot run
    // further ahead than that, because a step's prep waits for the order stage of two steps before (ev_order, above).
    const bool join_st = !ctx->overlap || ctx->prof_on || capturing;
    {
        // nreg > 1: the env chunks are dealt round-robin to the regions' streams, which fork from `st` here; the
        // substep chunks of one env chunk stay on one stream (L_ref / L_prev carry)
        const bool multi = ctx->nreg > 1;
        const int nchunks_e = (g.E + ctx->chunk_ne - 1) / ctx->chunk_ne, nchunks_i = (g.S + ctx->chunk_ni - 1) / ctx->chunk_ni;
        Span sp_all(ctx, st, EVIS_STAGE_WARP, multi ? 2 * nchunks_e * nchunks_i : 0, multi);
        if (multi) {
            CU(cudaEventRecord(ctx->ev_fork, st));
            for (int r = 0; r < ctx->nreg; ++r) CU(cudaStreamWaitEvent(ctx->reg_stream[r], ctx->ev_fork, 0));
        }
        const size_t planes = (size_t)ctx->nset * ctx->chunk_ni * ctx->chunk_ne;
        for (int e0 = 0, ce = 0; e0 < g.E; e0 += ctx->chunk_ne, ++ce) {
            const int ne = g.E - e0 < ctx->chunk_ne ? g.E - e0 : ctx->chunk_ne;
            const int r = ce % ctx->nreg;
            cudaStream_t cs = multi ? ctx->reg_stream[r] : st;
            unsigned long long *zr = ctx->zmem + (size_t)r * (ctx->zmem_bytes / 8);
            for (int i0 = 1; i0 <= g.S; i0 += ctx->chunk_ni) {
                const int ni = g.S + 1 - i0 < ctx->chunk_ni ? g.S + 1 - i0 : ctx->chunk_ni;
                ZChunk zc;
                zc.e0 = e0; zc.ne = ne; zc.i0 = i0; zc.ni = ni;
                // every chunk uses the plane strides of the full chunk shape, so one pair of tensor maps serves all
                zc.ne_alloc = ctx->chunk_ne; zc.ni_alloc = ctx->chunk_ni;
                zc.zd = zr;
                zc.zc = zr + planes * g.HWp;
                zc.idx_bits = ctx->idx_bits;
                zc.tag = 0;
                zc.tmap_d = ctx->have_tmap ? ctx->tmap_d[r] : nullptr;
                zc.tmap_c = ctx->have_tmap ? ctx->tmap_c[r] : nullptr;
                if (ctx->idx_bits == 32) {
                    Span sp(ctx, cs, EVIS_STAGE_CLEAR, 1, !multi);
                    CU(cudaMemsetAsync(zr, 0xFF, ctx->zmem_bytes, cs));
                } else {
                    // tagged keys: every chunk takes a smaller tag than all before it in its region; stale
                    // entries lose the atomicMin and fail the tag test, so one clear serves 255 chunks
                    if (ctx->ztag[r] <= 0) {
                        Span sp(ctx, cs, EVIS_STAGE_CLEAR, 1, !multi);
                        CU(cudaMemsetAsync(zr, 0xFF, ctx->zmem_bytes, cs));
                        ctx->ztag[r] = 255;
                    }
                    zc.tag = (uint32_t)--ctx->ztag[r];
                }
                { Span sp(ctx, cs, EVIS_STAGE_SPLAT, multi ? 0 : 1, !multi); CU(launch_global_splat(g, zc, A, B, ctx->h_tab, cs)); }
                if (g.mode == EVIS_COMPOSITE_WEIGHTED) {
                    // R32: front depth per target, the weighted sums of its front surface, then Eq. 4 on their quotient
                    Span sp(ctx, cs, EVIS_STAGE_RESOLVE, multi ? 0 : 3, !multi);
                    FrameIO fio{};
                    fio.wacc = ctx->wacc + 2 * (size_t)r * ctx->wchunk_elems;
                    CU(launch_front_wsplat(g, zc, A, B, ctx->h_tab, ctx->zfront + (size_t)r * ctx->wchunk_elems,
                                           ctx->wacc + 2 * (size_t)r * ctx->wchunk_elems, cnt + C_HOLES, ctx->dbg, cs));
                    CU(launch_resolve_weighted(g, zc, ctx->h_tab, ctx->l_ref, ctx->l_prev, ctx->ep, th, rf, sink, cnt + C_HOLES,
                                               ctx->dbg, fio, cs));
                } else if (ctx->defocus) {
                    // two passes (R31): the warped LINEAR frames of the chunk, then blur + log + Eq. 4
                    Span sp(ctx, cs, EVIS_STAGE_RESOLVE, multi ? 0 : 2, !multi);
                    FrameIO fio{ctx->frames + (size_t)r * ctx->frames_elems, ctx->taps, ctx->cfg.log_eps};
                    CU(launch_resolve_frames(g, zc, ctx->lin[ia], ctx->lin[ctx->cur], ctx->h_tab, ctx->i_prev, ctx->ep,
                                             cnt + C_HOLES, ctx->dbg, fio, cs));
                    CU(launch_resolve_blurred(g, zc, ctx->h_tab, ctx->l_ref, ctx->l_prev, ctx->ep, th, rf, sink, cnt + C_HOLES,
                                              ctx->dbg, fio, cs));
                } else {
                    Span sp(ctx, cs, EVIS_STAGE_RESOLVE, multi ? 0 : 1, !multi);
                    CU(launch_global_resolve(g, zc, A, B, ctx->h_tab, ctx->l_ref, ctx->l_prev, ctx->ep, th, rf, sink,
                                             cnt + C_HOLES, ctx->dbg, cs));
                }
            }
        }
        if (multi)
            for (int r = 0; r < ctx->nreg; ++r) {
                CU(cudaEventRecord(ctx->ev_join[r], ctx->reg_stream[r]));
                if (join_st) CU(cudaStreamWaitEvent(st, ctx->ev_join[r], 0));
            }
    }
    // a8, second half, on the order stream: it starts when this step's chunks are done and overlaps the next step
    cudaStream_t os = ctx->ord_stream;
    CU(cudaEventRecord(ctx->ev_chunks[sl], st));
    CU(cudaStreamWaitEvent(os, ctx->ev_chunks[sl], 0));
    if (ctx->nreg > 1 && !join_st)
        for (int r = 0; r < ctx->nreg; ++r) CU(cudaStreamWaitEvent(os, ctx->ev_join[r], 0));
    // this slot's `ordered` (or the voxel image) is still being copied out
    if (ctx->copy_pending && (ctx->copy_slot < 0 || ctx->copy_slot == sl || ctx->ordered_s[0] == ctx->ordered_s[1]))
        CU(cudaStreamWaitEvent(os, ctx->ev_copy, 0));
    VoxelSink vs{};
    vs.store_events = ctx->compact ? 2 : 1;
    vs.dt = ctx->ep.dt;
    if (ctx->vox_on) {
        if (ctx->vox_restart || ctx->vox_j >= (uint32_t)ctx->vox.window_steps) {     // a new window starts with this interval
            CU(cudaMemsetAsync(ctx->vox_v, 0, ctx->vox_cells * sizeof(unsigned long long), os));
            ctx->vox_j = 0;
            ctx->vox_restart = false;
        }
        volatile float tb = (float)ctx->vox_j * ctx->cfg.keyframe_dt;
        volatile float sc = (float)(ctx->vox.bins - 1) / ((float)ctx->vox.window_steps * ctx->cfg.keyframe_dt);
        vs.v = ctx->vox_v;
        vs.bins = (uint32_t)ctx->vox.bins;
        vs.hc = (uint32_t)(g.H - 2 * g.margin); vs.wc = (uint32_t)(g.W - 2 * g.margin);
        vs.t_base = tb; vs.scale = sc;
        if (!ctx->vox.keep_events) vs.store_events = 0;
        ctx->vox_j += 1;
    }
    {
        Span sp(ctx, os, EVIS_STAGE_ORDER, 3);
        unsigned long long *sticky = ctx->counters_s[0];             // C_MOTION, C_TOTAL live in slot 0's array
        if (!rf.t_last) {
            const uint32_t tx = (g.W + G_TILE_W - 1) / G_TILE_W, ty = (g.H + G_TILE_H - 1) / G_TILE_H;
            CU(launch_expand(sink, ctx->dir_entries, ctx->bsum, ctx->ordered_s[sl], ctx->cfg.event_capacity,
                             cnt + C_EVENTS, sticky + C_TOTAL, sticky + C_OVERFLOW, ctx->ep, th, (uint32_t)g.W,
                             (uint32_t)g.HW, (uint32_t)g.margin, tx, tx * ty, (uint32_t)g.S, vs, os));
        } else {
            CU(launch_order(sink, ctx->dir_entries, ctx->bsum, ctx->ordered_s[sl], ctx->cfg.event_capacity,
                            cnt + C_EVENTS, sticky + C_TOTAL, sticky + C_OVERFLOW, vs, os));
        }
        if (ctx->time_sorted && vs.store_events == 1) {
            // the arrival buffer of this slot is free once the stream has been laid out: it is the sort's scratch
            CU(launch_time_sort(sink.directory, ctx->dir_entries, rf.t_last ? 0 : DIR_EV_SHIFT, (uint32_t)g.E,
                                ctx->cfg.event_capacity < ctx->arrival_cap ? ctx->cfg.event_capacity : ctx->arrival_cap,
                                ctx->ordered_s[sl], ctx->arrival_s[sl], ctx->sort_ws, os));
            ctx->launches += 14;
        }
        CU(cudaMemcpyAsync(ctx->h_counters, cnt, C_STEP_END * sizeof(unsigned long long), cudaMemcpyDeviceToHost, os));
        CU(cudaMemcpyAsync(ctx->h_copy + evis_ctx::H_SLOT + sl * evis_ctx::H_SLOT_WORDS, cnt, (C_ALLOC + 1) * sizeof(unsigned long long),
                           cudaMemcpyDeviceToHost, os));
        CU(cudaMemcpyAsync(ctx->h_counters + C_MOTION, sticky + C_MOTION, (NCOUNTERS - C_MOTION) * sizeof(unsigned long long),
                           cudaMemcpyDeviceToHost, os));
    }
    CU(cudaEventRecord(ctx->ev_order[sl], os));
    ctx->ord_pending[sl] = true;
    ctx->last_slot = sl;
    ctx->steps += 1;
    ctx->kf_next += 1;
    ctx->cur = (ctx->cur + 1) % 3;
    ctx->have_events = true;
    if (capturing) CU(cudaStreamWaitEvent(st, ctx->ev_order[sl], 0));       // the order stream joins the captured stream
    return EVIS_OK;
}

int evis_step(evis_ctx *ctx, const float *rad, const float *mv_bwd, const float *mv_fwd, const float *depth,
              void *cuda_stream, uint64_t *n_events)
{
    if (!ctx || !rad || !mv_bwd || !depth) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const bool first = ctx->steps == 0;
    if (ctx->graph_mode && !first && st != nullptr) {
        // measurement hook (EVIS_GRAPH=1): the step as one CUDA graph launch.  Nothing of an earlier step may be pending
        // (a capture cannot wait for work outside it), so the device is drained first: this is not a fast path.
        CU(cudaDeviceSynchronize());
        ctx->ord_pending[0] = ctx->ord_pending[1] = false;
        ctx->copy_pending = false;
        CU(cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed));
        const int rc = step_enqueue(ctx, rad, mv_bwd, mv_fwd, depth, st, true);
        cudaGraph_t gr = nullptr;
        cudaError_t e = cudaStreamEndCapture(st, &gr);
        cudaGraphExec_t ex = nullptr;
        if (rc == EVIS_OK && e == cudaSuccess) e = cudaGraphInstantiate(&ex, gr, 0);
        if (rc == EVIS_OK && e == cudaSuccess) e = cudaGraphLaunch(ex, st);
        if (rc == EVIS_OK && e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (ex) cudaGraphExecDestroy(ex);
        if (gr) cudaGraphDestroy(gr);
        // the events recorded inside the capture belong to the graph: nothing outside may wait for them, and nothing
        // needs to -- the launch has been waited for, order stage included
        ctx->ord_pending[0] = ctx->ord_pending[1] = false;
        if (rc != EVIS_OK) return rc;
        CU(e);
    } else {
        const int rc = step_enqueue(ctx, rad, mv_bwd, mv_fwd, depth, st, false);
        if (rc != EVIS_OK) return rc;
    }
    if (first) {
        if (n_events) { CU(cudaStreamSynchronize(st)); *n_events = 0; }
        return EVIS_OK;
    }
    if (n_events) {
        const int rc = fetch_counters(ctx);
        if (rc != EVIS_OK) return rc;
        *n_events = ctx->last_events;
        if (ctx->last_overflow) return EVIS_ERR_OVERFLOW;
        if (ctx->last_motion) return EVIS_ERR_MOTION_BOUND;
    }
    return EVIS_OK;
}

int evis_set_thresholds(evis_ctx *ctx, const float *theta_on, const float *theta_off, int src_is_device)
{
    if (!ctx || ((theta_on == nullptr) != (theta_off == nullptr))) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    // work already enqueued keeps the thresholds it was launched with
    if (ctx->steps) CU(sync_all(ctx));
    if (!theta_on) { ctx->th_active = false; return EVIS_OK; }
    const size_t P = (size_t)ctx->g.E * ctx->g.HW;
    float *on = nullptr, *off = nullptr;
    unsigned long long *bad = nullptr, h_bad = 0;
    int rc = EVIS_OK;
    cudaError_t e = cudaMalloc((void **)&on, P * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc((void **)&off, P * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc((void **)&bad, sizeof *bad);
    const cudaMemcpyKind kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    cudaStream_t st = ctx->own_stream;
    if (e == cudaSuccess) e = cudaMemsetAsync(bad, 0, sizeof *bad, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(on, theta_on, P * sizeof(float), kind, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(off, theta_off, P * sizeof(float), kind, st);
    if (e == cudaSuccess) e = launch_check_positive(on, (long long)P, bad, st);
    if (e == cudaSuccess) e = launch_check_positive(off, (long long)P, bad, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h_bad, bad, sizeof h_bad, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
        ctx->last_cuda = (int)e;
        cudaGetLastError();
        rc = e == cudaErrorMemoryAllocation ? EVIS_ERR_OOM : EVIS_ERR_CUDA;
    } else if (h_bad) {
        rc = EVIS_ERR_INVALID_ARG;                      // the previous thresholds stay in force
    }
    cudaFree(bad);
    if (rc != EVIS_OK) { cudaFree(on); cudaFree(off); return rc; }
    // the new maps replace the old ones; nothing else the context owns is touched
    if (!ctx->th_on) ctx->device_bytes += 2 * P * sizeof(float);
    cudaFree(ctx->th_on); cudaFree(ctx->th_off);
    ctx->th_on = on; ctx->th_off = off;
    ctx->th_active = true;
    ctx->launches += 2;
    return EVIS_OK;
}

int evis_wait_events(evis_ctx *ctx, void *cuda_stream)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (ctx->steps > 1 && ctx->ord_pending[ctx->last_slot])
        CU(cudaStreamWaitEvent((cudaStream_t)cuda_stream, ctx->ev_order[ctx->last_slot], 0));
    return EVIS_OK;
}

int evis_set_noise(evis_ctx *ctx, const evis_noise *noise, const uint8_t *hot_mask, int mask_is_device)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (ctx->steps) CU(sync_all(ctx));
    if (!noise) { ctx->noise_on = false; return EVIS_OK; }
    const float big = 3.0e38f;
    if (!(noise->r_leak >= 0.0f && noise->r_leak < big) || !(noise->r_shot >= 0.0f && noise->r_shot < big) ||
        !(noise->r_hot >= 0.0f && noise->r_hot < big) || !(noise->i_white > 0.0f && noise->i_white < big))
        return EVIS_ERR_INVALID_ARG;
    const size_t P = (size_t)ctx->g.E * ctx->g.HW;
    if (hot_mask) {
        if (!ctx->hot) CU(dalloc(ctx, &ctx->hot, P));
        CU(cudaMemcpyAsync(ctx->hot, hot_mask, P, mask_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->own_stream));
    } else if (ctx->hot) {
        cudaFree(ctx->hot);
        ctx->hot = nullptr;
        ctx->device_bytes -= P;
    }
    if (!ctx->t_last) {                                   // the direct resolve variant carries t_last
        CU(dalloc(ctx, &ctx->t_last, P));
        CU(launch_fill(ctx->t_last, (long long)P, -INFINITY, ctx->own_stream));
    }
    CU(cudaStreamSynchronize(ctx->own_stream));
    ctx->noise = *noise;
    ctx->noise_on = true;
    return EVIS_OK;
}

int evis_set_voxels(evis_ctx *ctx, const evis_voxel_config *cfg)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    if (cfg && (cfg->bins < 1 || cfg->bins > 65535 || cfg->window_steps < 1)) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (ctx->steps) CU(sync_all(ctx));
    if (ctx->copy_pending) { CU(cudaStreamSynchronize(ctx->copy_stream)); ctx->copy_pending = false; }
    if (ctx->vox_v) {
        ctx->device_bytes -= ctx->vox_cells * (sizeof(unsigned long long) + sizeof(float));
        cudaFree(ctx->vox_v); cudaFree(ctx->vox_out);          // the grid's two buffers, nothing else
        ctx->vox_v = nullptr; ctx->vox_out = nullptr;
    }
    ctx->vox_on = false;
    if (!cfg) return EVIS_OK;
    const Geom &g = ctx->g;
    ctx->vox_cells = (size_t)g.E * 2u * (size_t)cfg->bins * (size_t)(g.H - 2 * g.margin) * (size_t)(g.W - 2 * g.margin);
    CU(dalloc(ctx, &ctx->vox_v, ctx->vox_cells));
    CU(dalloc(ctx, &ctx->vox_out, ctx->vox_cells));
    CU(cudaMemset(ctx->vox_v, 0, ctx->vox_cells * sizeof(unsigned long long)));
    ctx->vox = *cfg;
    ctx->vox_j = 0;
    ctx->vox_restart = false;
    ctx->vox_on = true;
    return EVIS_OK;
}

// enqueue V -> float32 behind the last step's order stage (and behind a copy of the previous image still running)
static int voxel_finish(evis_ctx *ctx, int normalize)
{
    const Geom &g = ctx->g;
    const uint32_t plane = (uint32_t)(g.H - 2 * g.margin) * (uint32_t)(g.W - 2 * g.margin);
    if (ctx->copy_pending) CU(cudaStreamWaitEvent(ctx->ord_stream, ctx->ev_copy, 0));
    // (the order stream already follows every step's chunk phase: nothing else to wait for)
    CU(launch_voxel_finish(ctx->vox_v, ctx->vox_out, (uint32_t)(ctx->vox_cells / plane), plane, normalize, ctx->ord_stream));
    ctx->launches += 1;
    return EVIS_OK;
}

int evis_read_voxels(evis_ctx *ctx, float *dst, int dst_is_device, int normalize, int restart, uint32_t *n_intervals)
{
    if (!ctx || !dst) return EVIS_ERR_INVALID_ARG;
    if (!ctx->vox_on) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (ctx->copy_pending) { CU(cudaStreamSynchronize(ctx->copy_stream)); ctx->copy_pending = false; }
    const int rc = voxel_finish(ctx, normalize);
    if (rc != EVIS_OK) return rc;
    CU(cudaStreamSynchronize(ctx->ord_stream));
    CU(cudaMemcpy(dst, ctx->vox_out, ctx->vox_cells * sizeof(float), dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    if (n_intervals) *n_intervals = ctx->vox_j;
    if (restart) ctx->vox_restart = true;
    return EVIS_OK;
}

int evis_read_voxels_begin(evis_ctx *ctx, float *host_dst, int normalize, int restart)
{
    if (!ctx || !host_dst) return EVIS_ERR_INVALID_ARG;
    if (!ctx->vox_on) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (ctx->copy_pending) { CU(cudaStreamSynchronize(ctx->copy_stream)); ctx->copy_pending = false; }
    const int rc = voxel_finish(ctx, normalize);
    if (rc != EVIS_OK) return rc;
    CU(cudaEventRecord(ctx->ev_copy, ctx->ord_stream));
    CU(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_copy, 0));
    CU(cudaMemcpyAsync(host_dst, ctx->vox_out, ctx->vox_cells * sizeof(float), cudaMemcpyDeviceToHost, ctx->copy_stream));
    CU(cudaEventRecord(ctx->ev_copy, ctx->copy_stream));
    ctx->copy_pending = true;
    ctx->copy_slot = -1;
    if (restart) ctx->vox_restart = true;
    return EVIS_OK;
}

int evis_read_voxels_end(evis_ctx *ctx) { return evis_read_events_end(ctx); }

int evis_set_compact_events(evis_ctx *ctx, int on)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    if (on && (ctx->g.W > 4096 || ctx->g.H > 4096)) return EVIS_ERR_INVALID_ARG;     // 12 bits per coordinate
    if (on && ctx->time_sorted) return EVIS_ERR_BAD_STATE;                            // the sort moves 16-byte events
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (ctx->steps) CU(sync_all(ctx));
    if (ctx->copy_pending) { CU(cudaStreamSynchronize(ctx->copy_stream)); ctx->copy_pending = false; }
    ctx->compact = on != 0;
    ctx->have_events = false;                     // the stored stream of the last step has the other format
    return EVIS_OK;
}

// the 8-byte twin of evis_read_events / _begin: same order, same counts, half the bytes
static int read_events8(evis_ctx *ctx, uint64_t *dst, int dst_is_device, uint64_t max, uint64_t *n_out, bool async)
{
    if (!ctx || (!dst && max > 0)) return EVIS_ERR_INVALID_ARG;
    if (!ctx->have_events || !ctx->compact || (ctx->vox_on && !ctx->vox.keep_events)) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    const int rc = fetch_counters(ctx);
    if (rc != EVIS_OK) return rc;
    if (ctx->copy_pending) { CU(cudaStreamSynchronize(ctx->copy_stream)); ctx->copy_pending = false; }
    uint64_t n = stored_events(ctx);
    if (n > max) n = max;
    if (n && !async)
        CU(cudaMemcpy(dst, ctx->ordered_s[ctx->last_slot], n * sizeof(uint64_t), dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    if (n && async) {
        CU(cudaMemcpyAsync(dst, ctx->ordered_s[ctx->last_slot], n * sizeof(uint64_t), cudaMemcpyDeviceToHost, ctx->copy_stream));
        CU(cudaEventRecord(ctx->ev_copy, ctx->copy_stream));
        ctx->copy_pending = true;
        ctx->copy_slot = ctx->last_slot;
    }
    if (n_out) *n_out = n;
    return ctx->last_overflow ? EVIS_ERR_OVERFLOW : EVIS_OK;
}

int evis_read_events8(evis_ctx *ctx, uint64_t *dst, int dst_is_device, uint64_t max, uint64_t *n_out)
{
    return read_events8(ctx, dst, dst_is_device, max, n_out, false);
}

int evis_read_events8_begin(evis_ctx *ctx, uint64_t *host_dst, uint64_t max, uint64_t *n_out)
{
    return read_events8(ctx, host_dst, 0, max, n_out, true);
}

int evis_set_time_sorted(evis_ctx *ctx, int on)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    if (on && ctx->compact) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (ctx->steps) CU(sync_all(ctx));
    if (on && !ctx->sort_ws) {
        ctx->sort_ws_bytes = sort_workspace_bytes((uint32_t)ctx->g.E, ctx->cfg.event_capacity);
        CU(cudaMalloc(&ctx->sort_ws, ctx->sort_ws_bytes));
        ctx->device_bytes += ctx->sort_ws_bytes;
    }
    ctx->time_sorted = on != 0;
    return EVIS_OK;
}

int evis_set_defocus(evis_ctx *ctx, float sigma)
{
    if (!ctx || !(sigma >= 0.0f) || !(sigma < 3.0e38f)) return EVIS_ERR_INVALID_ARG;
    if (ctx->cfg.composite_mode != EVIS_COMPOSITE_B_PRIMARY) return EVIS_ERR_INVALID_ARG;
    if (ctx->steps) return EVIS_ERR_BAD_STATE;          // the first keyframe already fixed L_ref
    // R = ceil(3 sigma); w_k = exp(-k^2 / (2 sigma^2)) / sum in binary64, rounded to binary32 (R31)
    const double sg = (double)sigma;
    const int R = sigma > 0.0f ? (int)ceil(3.0 * sg) : 0;
    if (R > BLUR_RMAX) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    memset(&ctx->taps, 0, sizeof ctx->taps);
    ctx->taps.R = R;
    double sum = 0.0;
    for (int k = -R; k <= R; ++k) sum += R ? exp(-(double)(k * k) / (2.0 * sg * sg)) : 1.0;
    for (int k = -R; k <= R; ++k) ctx->taps.w[k + R] = (float)((R ? exp(-(double)(k * k) / (2.0 * sg * sg)) : 1.0) / sum);
    if (!ctx->lin[0]) {
        const size_t P = (size_t)ctx->g.E * ctx->g.HW;
        CU(dalloc(ctx, &ctx->lin[0], 3 * P));
        ctx->lin[1] = ctx->lin[0] + P;
        ctx->lin[2] = ctx->lin[0] + 2 * P;
        CU(dalloc(ctx, &ctx->i_prev, P));
        ctx->frames_elems = (size_t)ctx->chunk_ne * ctx->chunk_ni * ctx->g.HW;
        CU(dalloc(ctx, &ctx->frames, ctx->frames_elems * ctx->nreg));
    }
    ctx->defocus = true;
    return EVIS_OK;
}

int evis_set_interval_index(evis_ctx *ctx, uint32_t next_kf)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    ctx->kf_next = next_kf;
    return EVIS_OK;
}

int evis_set_env_offset(evis_ctx *ctx, uint32_t first_env)
{
    if (!ctx || (unsigned long long)first_env + (unsigned long long)ctx->g.E > 0x100000000ull) return EVIS_ERR_INVALID_ARG;
    ctx->env_offset = first_env;
    return EVIS_OK;
}

int evis_set_channel(evis_ctx *ctx, int channel)
{
    if (!ctx || channel < -1 || channel > 2) return EVIS_ERR_INVALID_ARG;
    ctx->channel = channel;
    ctx->channel_set = channel >= 0;
    return EVIS_OK;
}

int evis_set_margin(evis_ctx *ctx, int margin)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    if (margin < 0 || 2 * (long long)margin >= (ctx->g.H < ctx->g.W ? ctx->g.H : ctx->g.W)) return EVIS_ERR_INVALID_ARG;
    if (ctx->vox_on) return EVIS_ERR_BAD_STATE;       // the voxel grid has the cropped frame's shape: set the margin first
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (ctx->steps) CU(sync_all(ctx));
    ctx->g.margin = margin;
    return EVIS_OK;
}

int evis_set_refractory(evis_ctx *ctx, float tau_r)
{
    if (!ctx || !(tau_r >= 0.0f) || !(tau_r < 3.0e38f)) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (ctx->steps) CU(sync_all(ctx));
    if (tau_r > 0.0f) {
        // (re)start with no event emitted yet: t_last = -inf at every pixel
        const size_t P = (size_t)ctx->g.E * ctx->g.HW;
        if (!ctx->t_last) CU(dalloc(ctx, &ctx->t_last, P));
        CU(launch_fill(ctx->t_last, (long long)P, -INFINITY, ctx->own_stream));
        CU(cudaStreamSynchronize(ctx->own_stream));
        ctx->launches += 1;
    }
    ctx->tau_r = tau_r;
    return EVIS_OK;
}

int evis_step_host(evis_ctx *ctx, const float *rad, const float *mv_bwd, const float *mv_fwd,
                   const float *depth, uint64_t *n_events)
{
    if (!ctx || !rad || !mv_bwd || !depth) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    const size_t P = (size_t)ctx->g.E * ctx->g.HW;
    if (!ctx->up_stream) {
        CU(cudaStreamCreateWithFlags(&ctx->up_stream, cudaStreamNonBlocking));
        for (int k = 0; k < 2; ++k) {
            CU(cudaEventCreateWithFlags(&ctx->ev_up[k], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&ctx->ev_used[k], cudaEventDisableTiming));
            CU(dalloc(ctx, &ctx->st_rad[k], 3 * P));
            CU(dalloc(ctx, &ctx->st_mv[k], 2 * P));
            CU(dalloc(ctx, &ctx->st_depth[k], P));
        }
    }
    if (mv_fwd && !ctx->st_fwd[0])
        for (int k = 0; k < 2; ++k) CU(dalloc(ctx, &ctx->st_fwd[k], 2 * P));
    // set k & 1: free once the step that read it two calls ago has run; its upload overlaps the previous step
    const int set = (int)(ctx->host_steps & 1);
    cudaStream_t up = ctx->up_stream, st = ctx->own_stream;
    // the previous call's host buffers are released when this call returns: its upload has to be over
    if (ctx->set_used[set ^ 1]) CU(cudaEventSynchronize(ctx->ev_up[set ^ 1]));
    if (ctx->set_used[set]) CU(cudaStreamWaitEvent(up, ctx->ev_used[set], 0));
    CU(cudaMemcpyAsync(ctx->st_rad[set], rad, 3 * P * sizeof(float), cudaMemcpyHostToDevice, up));
    CU(cudaMemcpyAsync(ctx->st_mv[set], mv_bwd, 2 * P * sizeof(float), cudaMemcpyHostToDevice, up));
    if (mv_fwd) CU(cudaMemcpyAsync(ctx->st_fwd[set], mv_fwd, 2 * P * sizeof(float), cudaMemcpyHostToDevice, up));
    CU(cudaMemcpyAsync(ctx->st_depth[set], depth, P * sizeof(float), cudaMemcpyHostToDevice, up));
    CU(cudaEventRecord(ctx->ev_up[set], up));
    CU(cudaStreamWaitEvent(st, ctx->ev_up[set], 0));
    uint64_t n = 0;
    const int rc = evis_step(ctx, ctx->st_rad[set], ctx->st_mv[set], mv_fwd ? ctx->st_fwd[set] : nullptr, ctx->st_depth[set],
                             (void *)st, n_events ? &n : nullptr);
    cudaEventRecord(ctx->ev_used[set], st);
    ctx->set_used[set] = true;
    ctx->host_steps += 1;
    if (n_events) *n_events = n;
    return rc;
}

int evis_read_events(evis_ctx *ctx, evis_event *dst, int dst_is_device, uint64_t max, uint64_t *n_out)
{
    if (!ctx || (!dst && max > 0)) return EVIS_ERR_INVALID_ARG;
    if (!ctx->have_events || (ctx->vox_on && !ctx->vox.keep_events) || ctx->compact) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    const int rc = fetch_counters(ctx);
    if (rc != EVIS_OK) return rc;
    uint64_t n = stored_events(ctx);
    if (n > max) n = max;
    if (n) CU(cudaMemcpy(dst, ctx->ordered_s[ctx->last_slot], n * sizeof(evis_event),
                         dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost));
    if (n_out) *n_out = n;
    return ctx->last_overflow ? EVIS_ERR_OVERFLOW : EVIS_OK;
}

int evis_read_events_begin(evis_ctx *ctx, evis_event *host_dst, uint64_t max, uint64_t *n_out)
{
    if (!ctx || (!host_dst && max > 0)) return EVIS_ERR_INVALID_ARG;
    if (!ctx->have_events || (ctx->vox_on && !ctx->vox.keep_events) || ctx->compact) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    const int rc = fetch_counters(ctx);
    if (rc != EVIS_OK) return rc;
    if (ctx->copy_pending) CU(cudaStreamSynchronize(ctx->copy_stream));
    uint64_t n = stored_events(ctx);
    if (n > max) n = max;
    if (n) {
        CU(cudaMemcpyAsync(host_dst, ctx->ordered_s[ctx->last_slot], n * sizeof(evis_event), cudaMemcpyDeviceToHost, ctx->copy_stream));
        CU(cudaEventRecord(ctx->ev_copy, ctx->copy_stream));
        ctx->copy_pending = true;
        ctx->copy_slot = ctx->last_slot;
    }
    if (n_out) *n_out = n;
    return ctx->last_overflow ? EVIS_ERR_OVERFLOW : EVIS_OK;
}

int evis_read_events_end(evis_ctx *ctx)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (ctx->copy_pending) CU(cudaStreamSynchronize(ctx->copy_stream));
    ctx->copy_pending = false;
    return EVIS_OK;
}

int evis_read_events_enqueue(evis_ctx *ctx, void *pinned_dst, uint64_t max, int previous_step)
{
    if (!ctx || !pinned_dst) return EVIS_ERR_INVALID_ARG;
    if (!ctx->have_events || (ctx->vox_on && !ctx->vox.keep_events)) return EVIS_ERR_BAD_STATE;
    // the step before the last: its stream lives in the other half of the doubled buffer (needs the overlap: EVIS_NO_OVERLAP
    // keeps one buffer), and there must be such a step
    if (previous_step && (ctx->ordered_s[0] == ctx->ordered_s[1] || ctx->steps < 3 || ctx->graph_mode)) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    cudaPointerAttributes at;                      // page-locked memory only: a pageable destination would make the copy synchronous
    if (cudaPointerGetAttributes(&at, pinned_dst) != cudaSuccess || at.type != cudaMemoryTypeHost) {
        cudaGetLastError();
        return EVIS_ERR_INVALID_ARG;
    }
    if (ctx->copy_pending) { CU(cudaStreamSynchronize(ctx->copy_stream)); ctx->copy_pending = false; }
    const int sl = previous_step ? ctx->last_slot ^ 1 : ctx->last_slot;
    // wait for THAT step's ordering stage only (not for the steps enqueued after it), then its counts are on the host
    if (ctx->ord_pending[sl]) CU(cudaEventSynchronize(ctx->ev_order[sl]));
    const unsigned long long *hc = ctx->h_copy + evis_ctx::H_SLOT + sl * evis_ctx::H_SLOT_WORDS;
    const unsigned long long made = ctx->steps < 2 ? 0ull : hc[C_EVENTS];
    const bool lost = ctx->steps >= 2 && hc[C_ALLOC] > ctx->arrival_cap;
    uint64_t n = lost ? 0ull : (made < ctx->cfg.event_capacity ? made : ctx->cfg.event_capacity);
    if (n > max) n = max;
    if (n) CU(cudaMemcpyAsync(pinned_dst, ctx->ordered_s[sl], n * (ctx->compact ? sizeof(uint64_t) : sizeof(evis_event)),
                              cudaMemcpyDeviceToHost, ctx->copy_stream));
    CU(cudaEventRecord(ctx->ev_copy, ctx->copy_stream));
    ctx->copy_pending = true;
    ctx->copy_slot = sl;
    ctx->deferred = true;
    ctx->h_copy[0] = n;
    ctx->h_copy[1] = lost ? 2ull : (made > ctx->cfg.event_capacity ? 1ull : 0ull);
    return EVIS_OK;
}

int evis_read_events_finish(evis_ctx *ctx, uint64_t *n_out)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (!guard.ok) return EVIS_ERR_CUDA;
    if (!ctx->deferred) return EVIS_ERR_BAD_STATE;      // no _enqueue to finish
    if (ctx->copy_pending) CU(cudaStreamSynchronize(ctx->copy_stream));
    ctx->copy_pending = false;
    ctx->deferred = false;
    if (n_out) *n_out = ctx->h_copy[0];
    return ctx->h_copy[1] ? EVIS_ERR_OVERFLOW : EVIS_OK;
}

int evis_events_device(evis_ctx *ctx, const evis_event **dev_ptr, uint64_t *n_stored)
{
    if (!ctx || !dev_ptr || !n_stored) return EVIS_ERR_INVALID_ARG;
    if (!ctx->have_events || (ctx->vox_on && !ctx->vox.keep_events) || ctx->compact) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    const int rc = fetch_counters(ctx);
    if (rc != EVIS_OK) return rc;
    *dev_ptr = reinterpret_cast<const evis_event *>(ctx->ordered_s[ctx->last_slot]);
    *n_stored = stored_events(ctx);
    return ctx->last_overflow ? EVIS_ERR_OVERFLOW : EVIS_OK;
}

int evis_get_info(evis_ctx *ctx, evis_info *info)
{
    if (!ctx || !info) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (ctx->steps) { const int rc = fetch_counters(ctx); if (rc != EVIS_OK) return rc; }
    memset(info, 0, sizeof *info);
    info->path = EVIS_PATH_GLOBAL;
    info->tile_w = G_TILE_W;
    info->tile_h = G_TILE_H;
    info->steps = ctx->steps;
    info->last_events = ctx->last_events;
    info->last_holes = ctx->last_holes;
    info->kernel_launches = ctx->launches;
    info->last_overflow = ctx->last_overflow;
    info->last_motion_violation = ctx->last_motion;
    info->device_bytes = ctx->device_bytes;
    info->total_events = ctx->h_counters[C_TOTAL];
    info->overflow_steps = ctx->h_counters[C_OVERFLOW];
    return EVIS_OK;
}

int evis_profile_enable(evis_ctx *ctx, int on)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    prof_drain(ctx);
    memset(&ctx->prof_acc, 0, sizeof ctx->prof_acc);
    ctx->prof_on = on != 0;
    return EVIS_OK;
}

int evis_profile_read(evis_ctx *ctx, evis_profile *out)
{
    if (!ctx || !out) return EVIS_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    prof_drain(ctx);
    *out = ctx->prof_acc;
    memset(&ctx->prof_acc, 0, sizeof ctx->prof_acc);
    return EVIS_OK;
}

int evis_get_state(evis_ctx *ctx, float *l_ref, float *l_prev)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    if (!ctx->steps) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    CU(sync_all(ctx));
    const size_t bytes = (size_t)ctx->g.E * ctx->g.HW * sizeof(float);
    if (l_ref) CU(cudaMemcpy(l_ref, ctx->l_ref, bytes, cudaMemcpyDeviceToHost));
    if (l_prev) CU(cudaMemcpy(l_prev, ctx->l_prev, bytes, cudaMemcpyDeviceToHost));
    return EVIS_OK;
}

int evis_refractory_state(evis_ctx *ctx, float *get_t_last, const float *set_t_last)
{
    if (!ctx || (get_t_last && set_t_last)) return EVIS_ERR_INVALID_ARG;
    if (!ctx->t_last) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    CU(sync_all(ctx));
    const size_t bytes = (size_t)ctx->g.E * ctx->g.HW * sizeof(float);
    if (get_t_last) CU(cudaMemcpy(get_t_last, ctx->t_last, bytes, cudaMemcpyDeviceToHost));
    if (set_t_last) CU(cudaMemcpy(ctx->t_last, set_t_last, bytes, cudaMemcpyHostToDevice));
    return EVIS_OK;
}

int evis_set_state(evis_ctx *ctx, const float *l_ref, const float *l_prev)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    if (!ctx->steps) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    CU(sync_all(ctx));
    const size_t bytes = (size_t)ctx->g.E * ctx->g.HW * sizeof(float);
    if (l_ref) CU(cudaMemcpy(ctx->l_ref, l_ref, bytes, cudaMemcpyHostToDevice));
    if (l_prev) CU(cudaMemcpy(ctx->l_prev, l_prev, bytes, cudaMemcpyHostToDevice));
    return EVIS_OK;
}

int evis_debug_read(evis_ctx *ctx, uint32_t *win, uint8_t *dir, float *l_hat)
{
    if (!ctx) return EVIS_ERR_INVALID_ARG;
    if (!ctx->cfg.debug_capture || ctx->steps < 2) return EVIS_ERR_BAD_STATE;
    DeviceGuard guard(ctx->cfg.device);
    CU(sync_all(ctx));
    const size_t n = (size_t)ctx->g.E * ctx->g.HW * ctx->g.S;
    if (win) CU(cudaMemcpy(win, ctx->dbg.win, n * sizeof(uint32_t), cudaMemcpyDeviceToHost));
    if (dir) CU(cudaMemcpy(dir, ctx->dbg.dir, n, cudaMemcpyDeviceToHost));
    if (l_hat) CU(cudaMemcpy(l_hat, ctx->dbg.l_hat, n * sizeof(float), cudaMemcpyDeviceToHost));
    return EVIS_OK;
}

}  // extern "C"
