/*
 * evis.h -- C ABI of the EVIS per-pixel event-synthesis hot path on B200 (sm_100a).
 *
 * What the library computes is defined by the paper (arxiv 2607.08098; /root/reference/PAPER.md):
 *   Sec. 3.2, Eq. 3-4 (lines 92-104): Rec.709 luminance, L = log(I + eps), contrast-threshold
 *            event count n = floor(|dL|/C), polarity, reference update L_ref += p n C;
 *   Sec. 3.3, Eq. 5-7 (lines 106-131): bidirectional motion-vector warping of keyframes A and B
 *            with z-buffered depth splatting, B primary / A fills holes (line 129).
 * Readings of silent or ambiguous points: DESIGN.md Sec. 2 (R1-R33).
 *
 * Conventions.  E environments, H x W pixels, S substeps per keyframe interval (S = the paper's
 * upsampling factor K).  Pixel (x, y) has its centre at integer coordinates, x right, y down.
 * All image tensors are dense, row-major, env-major: index ((e*H + y)*W + x)*C + c.
 * Motion vectors are in pixels: mv_bwd[p] is the displacement from pixel p of this keyframe to
 * the same surface point in the PREVIOUS keyframe.
 *
 * Environment variables read by evis_create (test and measurement hooks; none is needed in production, every default
 * is the measured best):
 *   EVIS_ZBUF_MB=<n>     budget of one z-buffer region in MiB (default 24 when an env's S substeps fit, else 512 / regions)
 *   EVIS_STREAMS=<n>     concurrent z-buffer regions / streams (default 4, or 2 for very large frames; at most 8)
 *   EVIS_CHUNK_NI=<n>, EVIS_CHUNK_NE=<n>   explicit chunk shape in substeps / envs (experiments)
 *   EVIS_NO_ZTAG=1       untagged 64-bit keys, z-buffers cleared before every chunk (the path frames > 2^24 pixels take)
 *   EVIS_NO_TMA=1        the resolve kernel loads keys directly instead of staging them by TMA
 *   EVIS_NO_OVERLAP=1    the ordering stage of a step is not overlapped with the next step (single buffers)
 *   EVIS_GRAPH=1         every evis_step is captured and launched as one CUDA graph (for `ncu --graph-profiling graph`;
 *                        the steps are serialised: no throughput claim)
 * (EVIS_NVCC_EXTRA is read by the build script, not by the library: extra nvcc flags for experiments.)
 *
 * Checkpoint / resume: evis_get_state / evis_set_state carry L_ref and L_prev, evis_refractory_state the refractory stamps,
 * evis_set_interval_index the interval counter.  Two pieces of state are NOT exposed: the carried unblurred frame of the
 * defocus path (a resumed context rebuilds it from keyframe A, so pixels that were holding an older value through a hole
 * or invalid depth can differ until they are reached again) and the position inside a voxel window (resume at a window
 * boundary, or read the grid first).
 *
 * Threading: a context may be used by one host thread at a time.  No function throws or aborts;
 * every function returns an evis_status (0 = OK, negative = error).
 */
#ifndef EVIS_H_
#define EVIS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct evis_ctx evis_ctx;       /* opaque; owned by the library */

typedef enum {
    EVIS_OK               =  0,
    EVIS_ERR_INVALID_ARG  = -1,   /* NULL pointer, non-positive size, threshold <= 0, ... */
    EVIS_ERR_CUDA         = -2,   /* a CUDA call failed; evis_last_cuda_error() has the code */
    EVIS_ERR_OOM          = -3,   /* device allocation failed */
    EVIS_ERR_OVERFLOW     = -4,   /* more events than event_capacity: the count returned is the true count; the
                                     stored stream is the first event_capacity events of the deterministic order,
                                     or EMPTY when the intermediate records did not fit either (evis_info
                                     last_overflow = 2): a read call then reports 0 events */
    EVIS_ERR_MOTION_BOUND = -5,   /* a motion vector exceeded the max_motion_px the caller declared (the results
                                     are exact all the same: the z-buffers take any motion) */
    EVIS_ERR_BAD_STATE    = -6,   /* call order violated (e.g. read before any step) */
    EVIS_ERR_TOO_LARGE    = -7    /* evis_voxelize_static: the grid has more cells than the fixed accumulator */
} evis_status;

/* One path: z-buffers in global memory (L2-resident chunks), any motion.  The per-tile shared-memory path of
 * round 1 (value 2) was measured 3-4x slower on every workload and retired: 2 is INVALID_ARG. */
enum { EVIS_PATH_AUTO = 0, EVIS_PATH_GLOBAL = 1 };
/* 0: Eq. 6 literally, the nearest source's value is copied; B primary, A fills B's holes (R14, R19).
 * 1: nearest of the two directions, time-weighted blend where both see the same surface (R19).
 * 2: weighted front-surface splat ("These target values are then bilinearly interpolated to integer
 *    pixels ... a per-pixel z-buffer that retains only the nearest surface"; R32): per direction, a target takes the
 *    bilinear-weighted mean of the log values of the sources that cover it and lie within 1 % of the z-buffer's depth;
 *    B primary, A fills B's holes.  Integer sums (weights in units of 2^-20, log values in units of 2^-24): the result
 *    does not depend on scheduling. */
enum { EVIS_COMPOSITE_B_PRIMARY = 0, EVIS_COMPOSITE_BLEND = 1, EVIS_COMPOSITE_WEIGHTED = 2 };

typedef struct {
    int32_t  num_envs, height, width;   /* E, H, W  (> 0; H, W <= 32767; E <= 65535)            */
    int32_t  substeps;                  /* S in 1..255 (K)                         */
    float    c_pos, c_neg;              /* contrast thresholds C+, C- (> 0)  (Eq. 4, R4)         */
    float    log_eps;                   /* eps of L = log(I + eps) (> 0)     (R2)   */
    float    keyframe_dt;               /* T = 1/f_k in seconds (> 0)                            */
    float    max_motion_px;             /* bound on |mv| (infinity norm) the caller declares; a violation
                                           is reported (EVIS_ERR_MOTION_BOUND); 0 = none declared   */
    int32_t  composite_mode;            /* EVIS_COMPOSITE_*  (R19)                 */
    int32_t  path;                      /* EVIS_PATH_*                                           */
    int32_t  device;                    /* CUDA device ordinal                                   */
    uint64_t event_capacity;            /* events stored per step (16 B each), > 0               */
    int32_t  debug_capture;             /* 1: keep, for every substep of the last step, the
                                           composite winner and the warped log frame (test hook;
                                           costs 9 B per pixel-substep of device memory)         */
    int32_t  reserved;
} evis_config;

/* One event, 16 bytes.  Absolute time = kf * T + t_off (form it in double).            (a7, R8) */
typedef struct {
    uint16_t x, y;          /* pixel                                                             */
    uint16_t env;           /* environment                                                       */
    int8_t   p;             /* polarity +1 / -1            (Eq. 4)                               */
    uint8_t  substep;       /* i in 1..S: the frame at which the crossing was detected           */
    float    t_off;         /* seconds from the start of the interval, in ((i-1) T/S, i T/S]     */
    uint32_t kf;            /* index of the keyframe interval (0 = between keyframes 0 and 1)    */
} evis_event;

typedef struct {
    int32_t  path;              /* EVIS_PATH_GLOBAL                                              */
    int32_t  tile_w, tile_h;    /* ordering tile of the event stream                             */
    int32_t  halo;              /* reserved (0)                                                  */
    uint64_t steps;             /* evis_step calls so far                                        */
    uint64_t last_events;       /* true event count of the last step                             */
    uint64_t last_holes;        /* pixel-substeps of the last step reached by neither keyframe   */
    uint64_t kernel_launches;   /* kernels + memsets this library launched since creation        */
    int32_t  last_overflow;     /* last step: 0 all events stored; 1 more than event_capacity (a valid prefix
                                   is stored); 2 the intermediate records overflowed too (nothing valid stored) */
    int32_t  last_motion_violation; /* 1 if a motion vector exceeded the declared max_motion_px   */
    uint64_t device_bytes;      /* device memory owned by the context                            */
    uint64_t total_events;      /* true event count summed over every step so far                */
    uint64_t overflow_steps;    /* steps so far whose events did not all fit (sticky)            */
} evis_info;

/* Per-stage device time, measured with CUDA events on the stream evis_step was given (test and
 * bench instrumentation; off by default).  Stages: */
enum { EVIS_STAGE_PREP = 0,     /* a1 + a9: log-luminance, keyframe take-over                     */
       EVIS_STAGE_CLEAR = 1,    /* global path: z-buffer / directory clears                       */
       EVIS_STAGE_SPLAT = 2,    /* global path: a2-a4                                             */
       EVIS_STAGE_RESOLVE = 3,  /* global path: a5-a8 (resolve, event model, compaction)          */
       EVIS_STAGE_ORDER = 4,    /* a8: deterministic ordering                                     */
       EVIS_STAGE_RESERVED5 = 5,
       EVIS_STAGE_WARP = 6,     /* global path with concurrent z-buffer regions: a2-a8 of all chunks, from the
                                   fork of the internal streams to their join (kernels overlap, so splat and
                                   resolve are not timed apart)                                   */
       EVIS_NUM_STAGES = 8 };
typedef struct {
    uint64_t steps;                       /* evis_step calls accumulated since enable / last read */
    uint64_t launches[EVIS_NUM_STAGES];   /* kernels + memsets per stage                          */
    double   ms[EVIS_NUM_STAGES];         /* device milliseconds per stage, summed                 */
} evis_profile;

/* Create a context: validates the configuration, allocates all device state.  *out is set only
 * on success.  Errors: INVALID_ARG, CUDA, OOM. */
int evis_create(const evis_config *cfg, evis_ctx **out);

/* Consume one keyframe (all DEVICE pointers, float32, read-only, caller-owned; they may be
 * freed or overwritten as soon as the work enqueued by this call has run on `cuda_stream`):
 *   rad    [E,H,W,3] scene-linear radiance R,G,B
 *   mv_bwd [E,H,W,2] backward motion vectors of this keyframe, pixels
 *   mv_fwd [E,H,W,2] or NULL: displacement of this keyframe's pixels towards the NEXT keyframe,
 *          used when this keyframe plays the role of A in the next call; NULL = the paper's
 *          default, -mv_bwd (R12)
 *   depth  [E,H,W]   depth, finite and > 0                (R17)
 * The first call only initialises (L_ref = L, R6) and emits no events.  Every later call closes
 * the interval kf = (call index - 1): warps A (previous keyframe) and B (this one) to the S
 * substeps (Eq. 5-7), runs the event model on every substep (Eq. 4), appends the events to the
 * context's device stream in deterministic order, carries L_ref forward and makes B the new A.
 * `cuda_stream` is a cudaStream_t (NULL = default stream).  The call is asynchronous unless
 * `n_events` (HOST pointer, nullable) is given: then it synchronises the stream and stores the
 * true number of events of this step.  Errors: INVALID_ARG, CUDA; with n_events also OVERFLOW
 * and MOTION_BOUND (the state has advanced regardless). */
int evis_step(evis_ctx *ctx, const float *rad, const float *mv_bwd, const float *mv_fwd,
              const float *depth, void *cuda_stream, uint64_t *n_events);

/* The ordered stream of a step is produced on a stream of the library's own, after the step's work on
 * `cuda_stream`, so that it overlaps the next evis_step (the calls that return events or counters wait for it).
 * evis_wait_events makes `cuda_stream` wait for the ordered stream of the last step -- needed only by a caller that
 * consumes evis_events_device()'s buffer, or measures time, on its own stream without one of those calls.
 * Errors: INVALID_ARG, CUDA. */
int evis_wait_events(evis_ctx *ctx, void *cuda_stream);

/* Same step with HOST buffers (pageable or pinned): copies them to device staging owned by the context and runs the
 * step on the context's own streams.  With n_events the call waits for the step and stores its event count.  With
 * n_events = NULL it only enqueues: the host buffers must then stay untouched until the NEXT evis_step_host call (or
 * any call that synchronises, e.g. evis_get_info) has returned.  There are two staging sets, so the upload of the next
 * keyframe starts the moment this one's is over and overlaps this step's kernels; every call that returns results
 * waits for the step as usual. */
int evis_step_host(evis_ctx *ctx, const float *rad, const float *mv_bwd, const float *mv_fwd,
                   const float *depth, uint64_t *n_events);

/* Threshold mismatch (Eq. 8; R25): replace the scalar thresholds C+ / C- of the
 * configuration by per-pixel maps theta_on, theta_off, each [E,H,W] float32, every value finite and > 0 (the
 * caller samples them, e.g. max(N(C, sigma^2), theta_min), once per pixel).  DEVICE pointers if src_is_device != 0,
 * else HOST.  The library copies the maps (the caller may free its buffers when the call returns; the call
 * synchronises) and uses them from the next evis_step on: Eq. 4 at pixel u runs with theta_on(u) for dL > 0 and
 * theta_off(u) for dL < 0.  Both NULL = back to the scalar thresholds.  
 * Errors: INVALID_ARG (exactly one pointer NULL; a value that is not finite and > 0 -- the previous thresholds
 * stay in force), CUDA, OOM. */
int evis_set_thresholds(evis_ctx *ctx, const float *theta_on, const float *theta_off, int src_is_device);

/* Noise events (Eq. 9-10; R29).  In every substep (duration dt = T / S) every pixel
 * draws, from a counter-based generator keyed (seed, interval, env, pixel, substep) -- so the stream does not depend
 * on scheduling --: a leak event (ON) with probability r_leak dt (Eq. 9); a shot event of random polarity with
 * probability r_shot dt (1 - Ibar), Ibar = clamp((exp(L) - eps) / i_white, 0, 1) the normalized intensity of the
 * warped frame (Eq. 10); and, for the pixels of the hot set, an event of random polarity with probability r_hot dt.
 * Their timestamps are uniform inside the substep; they follow the pixel's threshold crossings of that substep in
 * the stream (leak, shot, hot), leave L_ref alone and neither see nor feed the refractory period.  Rates in Hz. */
typedef struct {
    uint64_t seed;
    float    r_leak, r_shot, r_hot;   /* >= 0 */
    float    i_white;                 /* > 0: the linear intensity that normalizes to 1 */
} evis_noise;
/* noise = NULL switches the noise events off.  hot_mask: [E,H,W] bytes, non-zero = the pixel belongs to the hot set
 * (DEVICE pointer if mask_is_device != 0, else HOST; nullable = empty set); the library copies it.  Applies from the
 * next evis_step on; synchronises.  Errors: INVALID_ARG (negative or non-finite rate, i_white
 * <= 0), CUDA, OOM. */
int evis_set_noise(evis_ctx *ctx, const evis_noise *noise, const uint8_t *hot_mask, int mask_is_device);

/* The index `kf` the NEXT closed interval gets (it is stored in every event and keys the noise generator, R29);
 * it starts at 0 and advances by one per interval.  A context resumed from a checkpoint (evis_set_state,
 * evis_refractory_state, keyframe A fed again as its first step) sets it to the interval it continues with, so that
 * events carry the original indices and a noise run draws the same noise events.  Errors: INVALID_ARG. */
int evis_set_interval_index(evis_ctx *ctx, uint32_t next_kf);

/* Env sharding: this context holds the environments [first_env, first_env + num_envs) of a larger
 * batch (0 = the default: it holds the batch's first environments).  The noise generator is keyed by the environment's
 * index in the WHOLE batch (R29), so with the offset set a shard draws exactly the noise events the single context of the
 * whole batch draws for those environments.  Events keep the context's LOCAL env index (add first_env to get the batch's).
 * Applies from the next evis_step on.  Errors: INVALID_ARG (first_env + num_envs > 2^32). */
int evis_set_env_offset(evis_ctx *ctx, uint32_t first_env);

/* Colour events ("Replacing I with individual R, G, B channels and applying the event model to each
 * independently produces color events"; R28): channel = 0, 1 or 2 makes this context take
 * L = log(channel + eps) of the radiance's R, G or B instead of the Rec.709 luminance; -1 = luminance (default).
 * A colour sensor is three contexts fed the same keyframes, one per channel.  Applies to the keyframes given to
 * later evis_step calls: set it before the first one.  Errors: INVALID_ARG. */
int evis_set_channel(evis_ctx *ctx, int channel);

/* Defocus ("Prior to the event generation, the linear intensity is convolved with a separable Gaussian
 * kernel"; 0.1-0.5 px in the paper's sim-to-real data; R31).  With sigma >= 0 (pixels) the
 * frame the event model sees at every substep is log(G_sigma * I_hat + eps): the warped frame in LINEAR intensity
 * (the composite applied to the keyframes' linear luminance or channel; a hole holds its previous unblurred value),
 * convolved with a separable Gaussian -- taps k = -R..R, R = ceil(3 sigma) <= 8, w_k = exp(-k^2 / (2 sigma^2)) / sum,
 * rows then columns, the frame's border replicated -- and only then logged.  With a margin the blur runs on the whole
 * over-rendered frame.  sigma = 0 is a single tap (the plain path up to the rounding of the linear intensity).  Call it
 * before the first evis_step (L_ref starts from the blurred first keyframe); composite mode 0 only.
 * Errors: INVALID_ARG (negative or non-finite sigma, sigma > 8/3, composite mode 1), BAD_STATE (after the first
 * step), CUDA, OOM. */
int evis_set_defocus(evis_ctx *ctx, float sigma);

/* Over-render margin (Supp. B 317-319; R27): the frames handed to evis_step (height x
 * width of the configuration) were rendered with `margin` extra pixels on each side.  The warp uses all of them;
 * the margin is cropped off afterwards: the event model runs and events exist only for the inner
 * (height - 2 margin) x (width - 2 margin) pixels, x and y of an event are relative to that cropped frame, holes are
 * counted inside it.  0 = no margin (default).  Applies from the next evis_step on; synchronises.  
 * Errors: INVALID_ARG (negative, or 2 margin >= min(height, width)), BAD_STATE (a voxel grid is on: its shape is
 * the cropped frame's, so the margin comes first), CUDA. */
int evis_set_margin(evis_ctx *ctx, int margin);

/* Refractory period (R26): with tau_r > 0 (seconds) a threshold crossing of a pixel is
 * emitted only if its timestamp t satisfies t - t_last >= tau_r, t_last being the timestamp of the pixel's last
 * EMITTED event (none before the call: every pixel starts free); suppressed crossings still move L_ref (Eq. 4 is
 * unchanged).  The timestamps then decide which events exist, so they are computed in IEEE binary32 with a fixed
 * operation order.  The state t_last is carried across steps.  tau_r = 0 switches the period off.  Calling it
 * again with tau_r > 0 resets t_last.  Applies from the next evis_step on; synchronises.  
 * Errors: INVALID_ARG (negative or non-finite tau_r), CUDA, OOM. */
int evis_set_refractory(evis_ctx *ctx, float tau_r);

/* Voxel grid / accumulation image ("a per-polarity event voxel grid discretized into 128 temporal bins
 * with linear interpolation applied along the time axis. Each bin is normalized by dividing by its maximum event
 * count"; R30).  The library accumulates, on the device and in the same pass that lays
 * out the event stream, V [E, 2, bins, H', W'] (H' x W' = the frame after the margin crop; channel 0 = ON, 1 = OFF) over
 * a WINDOW of `window_steps` consecutive keyframe intervals: with t the time of an event from the start of the window
 * and D = window_steps * T, tau = (bins - 1) t / D, and the event adds max(0, 1 - |tau - b|) to bin b of its pixel and
 * polarity channel -- the two bins that bracket tau share one unit; bins = 1 is the plain per-polarity event count.
 * The sums are kept in 32.32 fixed point with integer atomics, so they do not depend on scheduling.  The first
 * window starts with the next evis_step that closes an interval; when a window is full the next step clears the grid
 * and starts a new one (read it before).  The grid takes EVERY event of a step, also those beyond event_capacity (only
 * an overflow of the intermediate records, evis_info last_overflow = 2, loses events).  keep_events = 0: the ordered event stream is not stored at all (the read
 * calls for events then return BAD_STATE) -- no 16-byte event ever leaves the GPU.  cfg = NULL switches the grid off.
 * Synchronises.  Errors: INVALID_ARG (bins < 1, window_steps < 1), CUDA, OOM. */
typedef struct {
    int32_t bins;            /* B >= 1 temporal bins per window                                  */
    int32_t window_steps;    /* N >= 1 keyframe intervals per window                             */
    int32_t keep_events;     /* 1: the ordered event stream is produced as well                  */
    int32_t reserved;
} evis_voxel_config;
int evis_set_voxels(evis_ctx *ctx, const evis_voxel_config *cfg);

/* Copy the grid as float32 [E, 2, bins, H', W'] to `dst` (device pointer if dst_is_device != 0, else host).
 * normalize != 0: every (env, channel, bin) plane is divided by its own maximum when that is > 0.
 * restart != 0: the next step starts a new window (clears the grid) even if this one is not full.
 * *n_intervals (nullable) = keyframe intervals accumulated in the window so far.  Synchronises.
 * Errors: INVALID_ARG, BAD_STATE (grid off), CUDA. */
int evis_read_voxels(evis_ctx *ctx, float *dst, int dst_is_device, int normalize, int restart, uint32_t *n_intervals);
/* The same to HOST memory (pinned, for a real overlap) in two halves, like evis_read_events_begin / _end: _begin
 * enqueues the conversion and the copy behind the last step and returns without waiting; _end waits for the copy.
 * The next step's accumulation waits for the copy too. */
int evis_read_voxels_begin(evis_ctx *ctx, float *host_dst, int normalize, int restart);
int evis_read_voxels_end(evis_ctx *ctx);

/* The voxel grid of a FINISHED event stream, for callers that must not allocate device memory.
 *
 * Who that is: evis_set_voxels calls cudaMalloc for its accumulator, and cudaMalloc / cudaFree both can fail and make
 * every stream of the device wait.  A rollout loop in which the simulator, the renderer and the learner have shared out
 * the GPU's memory among their own pools beforehand can afford neither while it runs; nor can a consumer that was handed
 * events (a recording, another process's stream) and owns no evis_ctx at all.  This call gives them the same grid from
 * memory the library already holds: it calls no cudaMalloc, cudaFree or other allocating routine, creates no stream or
 * event and needs no context.  The caller brings the input and the output; the 32.32 fixed-point accumulator between
 * them is ONE array of EVIS_VOXELIZE_STATIC_MAX_CELLS 64-bit words (16 MiB) that is part of the library's device image:
 * every GPU on which this library's kernels are loaded holds it until the process exits, whether or not this function
 * is ever called.
 *
 *   events  [n_events] DEVICE, 16-byte aligned, read-only: evis_event records as evis_read_events / evis_events_device
 *           deliver them (any order).  NULL is allowed when n_events = 0.
 *   grid    [num_envs, 2, bins, height, width] float32 DEVICE, written: the grid evis_read_voxels returns for a window
 *           of `window_steps` intervals of length keyframe_dt that starts with interval first_kf -- an event counts with
 *           t = (kf - first_kf) * keyframe_dt + t_off (binary32, as evis_step forms it); channel 0 = ON, 1 = OFF;
 *           height x width is the frame the events' x, y refer to (the cropped frame when a margin was set).  Events
 *           whose kf lies outside the window, whose x, y lie outside the frame or whose env >= num_envs add nothing.
 *   normalize != 0: every (env, channel, bin) plane is divided by its own maximum when that is > 0.
 *   cuda_stream: a cudaStream_t of the CURRENT device (NULL = default stream).  The call only enqueues (a clear of the
 *           cells it uses, the accumulation, the conversion to float32) and does not wait: `grid` is complete when the
 *           stream has run that work; `events` must stay valid until then.
 *   cuda_error (nullable): receives the cudaError_t behind an EVIS_ERR_CUDA return, else 0.
 *
 * The device that is current when the call is made is the one whose copy of the array is used: events, grid and the
 * stream must belong to it.  The FIRST call on each device also looks up the array's device address
 * (cudaGetSymbolAddress) and may make the CUDA runtime load the library's kernels; make that first call before any
 * stream capture is begun.  Later calls only enqueue the three operations.
 *
 * Sharing: all calls on a device use the same array, and it keeps whatever the last call left in it; each call clears
 * the cells it is about to use first, on its stream.  Calls whose work is ordered on the GPU (same stream, or streams
 * ordered by events) are safe back to back.  Calls whose work may OVERLAP on the GPU -- different unordered streams,
 * from one host thread or several -- race on the array and give wrong grids; so they must be serialised by the caller.
 *
 * Limit: 2 * num_envs * bins * height * width <= EVIS_VOXELIZE_STATIC_MAX_CELLS (2^21, e.g. 346 x 260, 5 bins, 2
 * environments); a larger grid is refused with EVIS_ERR_TOO_LARGE before anything is enqueued and `grid` is left
 * untouched -- call it per group of environments on that group's events, or use evis_set_voxels where allocating is allowed.
 * Errors: INVALID_ARG (NULL grid, NULL events with n_events > 0, a size or bins or window_steps < 1, keyframe_dt not
 * finite and > 0), TOO_LARGE, CUDA.  Argument errors are detected before any CUDA call. */
#define EVIS_VOXELIZE_STATIC_MAX_CELLS (1u << 21)
int evis_voxelize_static(const evis_event *events, uint64_t n_events, int32_t num_envs, int32_t height, int32_t width,
                         int32_t bins, int32_t window_steps, float keyframe_dt, uint32_t first_kf, int normalize,
                         float *grid, void *cuda_stream, int *cuda_error);

/* Time-sorted per-environment stream (the stream E = {(u_k, t_k, p_k)} of PAPER.md:90 in time order): with on != 0 the
 * stored stream of every later step is ordered by (env, t_off); events of one environment with equal timestamps keep
 * the deterministic order described at evis_read_events, so the result does not depend on scheduling.  A stable
 * segmented radix sort on the device, behind the step like the rest of the ordering stage (about 9 extra passes over
 * the stored events).  Needs the event stream (not a voxels-only context).  Synchronises.  Errors: INVALID_ARG, CUDA, OOM. */
int evis_set_time_sorted(evis_ctx *ctx, int on);

/* Compact events: with on != 0 the stored stream of every later step holds 8-byte events instead of 16-byte ones (half
 * the bytes to copy out; the order, the counts and the overflow rules are those of evis_read_events):
 *   bits  0-11 x | 12-23 y | 24-39 env | 40-47 substep i | 48-62 frac | 63 polarity (1 = ON, 0 = OFF)
 * frac = min(32767, floor(fr 2^15)), fr in [0, 1] the position of the timestamp inside its substep (R8), so
 *   t_off = (i - 1 + (frac + 0.5) / 32768) T / S   reproduces the 16-byte event's t_off within T / S * 2^-16
 * (1.6e-8 s at 1 kHz substeps), and the interval index kf is the step's (every event of a step shares it).  The 16-byte
 * read calls then return BAD_STATE; not together with the time-sorted stream.  Needs width, height <= 4096.
 * Synchronises.  Errors: INVALID_ARG, BAD_STATE, CUDA. */
typedef uint64_t evis_event8;
int evis_set_compact_events(evis_ctx *ctx, int on);
int evis_read_events8(evis_ctx *ctx, evis_event8 *dst, int dst_is_device, uint64_t max, uint64_t *n_out);
int evis_read_events8_begin(evis_ctx *ctx, evis_event8 *host_dst, uint64_t max, uint64_t *n_out);   /* ends with evis_read_events_end */

/* Copy the events of the last step, in the deterministic order
 * (env, substep, tile row, tile column, y, x, crossing k), to `dst` (room for `max` events;
 * device pointer if dst_is_device != 0, else host).  Synchronises.  *n_out = events copied
 * (= min(stored, max); stored = min(true count, capacity), see EVIS_ERR_OVERFLOW).
 * Errors: INVALID_ARG, BAD_STATE, CUDA; OVERFLOW when the last step overflowed (the valid prefix, if any, has been
 * copied all the same).  The same holds for evis_read_events_begin and evis_events_device. */
int evis_read_events(evis_ctx *ctx, evis_event *dst, int dst_is_device, uint64_t max, uint64_t *n_out);

/* The same copy to HOST memory (pinned, for a real overlap) in two halves, so that the next evis_step_host can upload
 * its keyframe while the events of this step go down the other direction of the link: _begin waits for the step,
 * stores the number of events that will be copied in *n_out, starts the copy on a stream of the library's own and
 * returns; _end waits for it.  `host_dst` must stay untouched until _end; the next step's ordered stream is not
 * produced before the copy has finished.  A second _begin ends the first.  Errors: INVALID_ARG, BAD_STATE, CUDA. */
int evis_read_events_begin(evis_ctx *ctx, evis_event *host_dst, uint64_t max, uint64_t *n_out);
int evis_read_events_end(evis_ctx *ctx);

/* The same copy for a PIPELINED loop: with previous_step != 0 the call copies the stream of the step BEFORE the last
 * evis_step / evis_step_host call -- still intact, because the ordered stream is double-buffered inside the context -- and
 * waits only for THAT step, not for the one enqueued after it.  So in
 *     evis_step_host(k + 1, n_events = NULL);  evis_read_events_finish(&n) [step k - 1];  evis_read_events_enqueue(buf[k & 1], max, 1) [step k]
 * the upload of keyframe k + 1, the kernels of step k and the download of step k - 1 are in flight together, while the
 * read calls above must wait for the last step before the next one can be enqueued.  _enqueue waits for the chosen step's
 * ordering stage, starts the copy of min(stored, max) events on a stream of the library's own and returns; _finish waits
 * for the copy and returns that number.  previous_step = 0: the last step, like evis_read_events_begin.  `pinned_dst`:
 * page-locked HOST memory (cudaHostAlloc / cudaHostRegister; e.g. a pinned torch tensor) with room for `max` events of
 * the stored format (16-byte evis_event, or 8-byte evis_event8 after evis_set_compact_events), untouched until _finish.
 * One deferred copy at a time: _enqueue first waits for an unfinished earlier copy.  The ordering stage of step k + 2
 * waits for the copy of step k (they share a buffer).
 * Errors: INVALID_ARG (NULL or pageable memory), BAD_STATE (no stored stream; previous_step before two intervals have
 * been closed, or with EVIS_NO_OVERLAP=1 / EVIS_GRAPH=1; _finish without _enqueue), CUDA; _finish returns OVERFLOW when
 * that step overflowed (the valid prefix, if any, has been copied). */
int evis_read_events_enqueue(evis_ctx *ctx, void *pinned_dst, uint64_t max, int previous_step);
int evis_read_events_finish(evis_ctx *ctx, uint64_t *n_out);

/* Device pointer to the ordered stream of the last step and its stored length (no copy);
 * valid until the next evis_step on the same context. */
int evis_events_device(evis_ctx *ctx, const evis_event **dev_ptr, uint64_t *n_stored);

/* Counters and geometry (synchronises the last step's stream). */
int evis_get_info(evis_ctx *ctx, evis_info *info);

/* Stage timing: enable/disable (resets the accumulators), read (synchronises, then resets). */
int evis_profile_enable(evis_ctx *ctx, int on);
int evis_profile_read(evis_ctx *ctx, evis_profile *out);

/* State access for tests and checkpointing: the carried reference level L_ref and the last
 * warped log frame L_prev, each [E,H,W] float32, to/from HOST memory.  Either may be NULL. */
int evis_get_state(evis_ctx *ctx, float *l_ref, float *l_prev);
int evis_set_state(evis_ctx *ctx, const float *l_ref, const float *l_prev);
/* The third piece of carried state, when the refractory period (or the noise events) is on: t_last [E,H,W] float32,
 * the timestamp of each pixel's last emitted event relative to the start of the NEXT interval (-inf: none yet; pixels
 * cropped by the margin keep their initial value).  Exactly one of the HOST pointers is given: get copies it out, set
 * copies it in.  Errors: INVALID_ARG, BAD_STATE (neither feature has been switched on), CUDA. */
int evis_refractory_state(evis_ctx *ctx, float *get_t_last, const float *set_t_last);

/* Test hook (needs debug_capture = 1): for the last step, per substep i-1 in [0,S), per pixel:
 *   win   [S,E,H,W] uint32: source linear index y*W+x of the composite winner, 0xFFFFFFFF = hole
 *   dir   [S,E,H,W] uint8 : 0 = from B, 1 = from A, 2 = blend (mode 1), 3 = hole
 *   l_hat [S,E,H,W] float32: the warped log frame
 * HOST pointers, each nullable. */
int evis_debug_read(evis_ctx *ctx, uint32_t *win, uint8_t *dir, float *l_hat);

/* Release everything.  NULL is accepted. */
int evis_destroy(evis_ctx *ctx);

const char *evis_strerror(int status);
int         evis_last_cuda_error(const evis_ctx *ctx);   /* cudaError_t of the last failure */
const char *evis_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EVIS_H_ */
