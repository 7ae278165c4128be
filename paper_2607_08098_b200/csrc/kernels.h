// kernels.h -- internal launch interface between api.cu and the kernel files (not part of the ABI).
#pragma once
#include "common.cuh"

namespace evis {

// One stored keyframe (device, owned by the context): planar so that the z-test gathers
// (far-endpoint depth, winner's L) touch 4-byte elements.
struct Keyframe {
    float  *L;     // [E*H*W] log-luminance                         (a1)
    float2 *mv;    // [E*H*W] backward motion vector, pixels
    float2 *fwd;   // [E*H*W] explicit forward field, or unused     (R12)
    float  *Z;     // [E*H*W] depth
    bool    has_fwd;
};

struct Geom {
    int E, H, W, S;
    int HW;        // H*W
    int Wp, HWp;   // z-buffer plane: (H+1) rows of pitch Wp = W+1 rounded up to even (TMA needs 16-byte row
                   // pitches), HWp = (H+1) * Wp.  Both kinds of plane use it with the same addressing: a source
                   // whose q has floor (x0, y0), x0 >= -1, y0 >= -1, files itself at (y0+1) * Wp + (x0+1) -- in
                   // the pixel plane zd that is target pixel (x0, y0) (row 0 / column 0 are a guard band for
                   // coordinate -1, never read), in the cell plane zc it is the class-11 cell (x0+1, y0+1)
    int mode;      // EVIS_COMPOSITE_*
    int margin;    // over-render margin (R27): H x W is the over-rendered frame; events exist only for
                   // pixels at least `margin` away from every side and carry coordinates relative to that crop
};

// Eq. 8: per-pixel ON / OFF thresholds [E*H*W], device; both null = the scalar C+ / C- of
// EventParams.
struct Thresholds {
    const float *on, *off;
};

// Refractory period (R26): t_last [E*H*W] = stamp of each pixel's last emitted event relative to
// the start of the current interval (-inf: none yet), device, read and written by the resolve kernel; null = off.
// With it on, the resolve kernel leaves EVENTS (not records) in the arrival buffer and order.cu copies them.
struct Refractory {
    float *t_last;
    float tau_r;    // seconds, >= 0 (0 with t_last set: direct mode for the noise events only)
    float T;        // keyframe period
    // Noise events (Eq. 9-10, R29); they ride on the direct (event-writing) resolve variant
    int noise_on;
    unsigned long long noise_key;    // mix64(seed ^ G (kf + 1)): the per-step part of the pixel keys
    float p_leak, p_shot, p_hot;     // r dt, binary32 products
    float i_white, eps;
    const unsigned char *hot;        // [E*H*W] membership of the hot set, or null
};

struct DebugOut {  // all nullable; [S,E,H,W]
    uint32_t *win;
    uint8_t  *dir;
    float    *l_hat;
};

// a1 + a9 (prep.cu)
// channel: -1 = Rec.709 luminance (Eq. 3), 0 / 1 / 2 = that channel alone (colour events)
cudaError_t launch_prep(const float *rad, const float *mv, const float *fwd, const float *depth, long long n,
                        float eps, int channel, float *L, float2 *mv_out, float2 *fwd_out, float *Z, float *l_ref,
                        float *l_prev, float motion_bound /* 0 = unchecked */, unsigned long long *viol,
                        float *lin_out /* nullable: the linear intensity, binary32 (defocus) */, cudaStream_t st);

// ---- defocus (R31) -----------------------------------------------------------------------------------
constexpr int BLUR_RMAX = 8;                      // R = ceil(3 sigma) <= 8
struct BlurTaps { int R; float w[2 * BLUR_RMAX + 1]; };   // w[k + R], k = -R..R
// the resolve kernel's two passes with defocus on: pass 1 leaves the warped LINEAR frames of the chunk,
// frames [ni_alloc][ne_alloc][HW]; pass 2 blurs them, takes the log and runs Eq. 4
struct FrameIO {
    float *frames;
    BlurTaps taps;
    float eps;
    const long long *wacc;       // weighted splat (R32): [ni_alloc][ne_alloc][HW][2] = (sum W L 2^24, sum W), else null
};
// first keyframe: l_ref = l_prev = log(G * I + eps)
cudaError_t launch_blur_log(const float *I, int E, int H, int W, const BlurTaps &taps, float eps, float *l_ref, float *l_prev,
                            cudaStream_t st);

// ---- global z-buffer path (global_path.cu): any motion -----------------------------------------
// z-buffers of one chunk = envs [e0, e0+ne) x substeps [i0, i0+ni):
//   zd [nset][ni_alloc][ne_alloc][HWp]  direct targets (footprints that are a single pixel or a 2-pixel edge)
//   zc [nset][ni_alloc][ne_alloc][HWp]  class-11 cells: the source covers the 2x2 block whose top-left is the cell
// nset = 1 in composite mode 0 (direction folded into the key's top bit), 2 in mode 1.  ni_alloc x ne_alloc is
// the context's full chunk shape: a smaller last chunk keeps the same plane strides (and tensor maps).
struct ZChunk {
    unsigned long long *zd, *zc;
    int e0, ne, i0, ni;
    int ne_alloc, ni_alloc; // plane strides of the allocation (>= ne, ni)
    uint32_t tag;          // idx_bits == 24: tag of this chunk (254 .. 0, decreasing); else 0
    int idx_bits;          // 32: untagged keys, buffers cleared before every chunk; 24: tagged keys
    const void *tmap_d, *tmap_c;   // HOST pointers to the CUtensorMap of zd / zc (3-D: x, y, plane), or null:
                                   // the resolve kernel then loads the keys directly instead of staging them by TMA
};
constexpr int TMAP_BYTES = 128;    // sizeof(CUtensorMap)
// Encode the tensor maps of a context's z-buffers ([planes][H+1][Wp] of 64-bit keys each, boxes
// of one resolve tile).  Returns false when the driver entry point is unavailable.
bool make_z_tensor_maps(const Geom &g, unsigned long long *zd, unsigned long long *zc, size_t planes, void *tmap_d,
                        void *tmap_c);
#ifndef EVIS_TILE_H
#define EVIS_TILE_H 16
#endif
constexpr int G_TILE_W = 32, G_TILE_H = EVIS_TILE_H;    // ordering tile of the global path
// The global path leaves RECORDS in the arrival buffer, one uint4 per firing pixel-substep:
//   x, y, z = bits of L_ref (before the update), L_prev, L_hat;  w = raster position in the tile | n << 16
// and directory entries (record offset, records | events << DIR_EV_SHIFT); order.cu expands them.
constexpr int DIR_EV_SHIFT = 10;               // a tile has 512 pixels: records <= 512 < 2^10

// tab: HOST copy of the substep table (passed to the kernels as a __grid_constant__ parameter)
cudaError_t launch_global_splat(const Geom &g, const ZChunk &zc, const Keyframe &A, const Keyframe &B,
                                const SubstepTable &tab, cudaStream_t st);
cudaError_t launch_global_resolve(const Geom &g, const ZChunk &zc, const Keyframe &A, const Keyframe &B,
                                  const SubstepTable &tab, float *l_ref, float *l_prev,
                                  const EventParams &ep, const Thresholds &th, const Refractory &rf,
                                  const EventSink &sink, unsigned long long *holes, const DebugOut &dbg, cudaStream_t st);
// the two defocus passes (resolve_defocus.cu)
cudaError_t launch_resolve_frames(const Geom &g, const ZChunk &zc, const float *IA, const float *IB, const SubstepTable &tab,
                                  float *i_prev, const EventParams &ep, unsigned long long *holes, const DebugOut &dbg,
                                  const FrameIO &fio, cudaStream_t st);
cudaError_t launch_resolve_blurred(const Geom &g, const ZChunk &zc, const SubstepTable &tab, float *l_ref, float *l_prev,
                                   const EventParams &ep, const Thresholds &th, const Refractory &rf, const EventSink &sink,
                                   unsigned long long *holes, const DebugOut &dbg, const FrameIO &fio, cudaStream_t st);
// weighted front-surface splat (R32; composite mode 2): front depth per target + the weighted sums
// (global_path.cu), then the event pass (resolve_defocus.cu)
cudaError_t launch_front_wsplat(const Geom &g, const ZChunk &zc, const Keyframe &A, const Keyframe &B, const SubstepTable &tab,
                                uint32_t *zfront, long long *wacc, unsigned long long *holes, const DebugOut &dbg, cudaStream_t st);
cudaError_t launch_resolve_weighted(const Geom &g, const ZChunk &zc, const SubstepTable &tab, float *l_ref, float *l_prev,
                                    const EventParams &ep, const Thresholds &th, const Refractory &rf, const EventSink &sink,
                                    unsigned long long *holes, const DebugOut &dbg, const FrameIO &fio, cudaStream_t st);
// its four instantiation units (resolve_m*.cu): composite mode 0 / 1, without / with the debug capture
#define EVIS_DECL_RESOLVE(name)                                                                                     \
    cudaError_t name(const Geom &g, const ZChunk &zc, const Keyframe &A, const Keyframe &B, const SubstepTable &tab,  \
                     float *l_ref, float *l_prev, const EventParams &ep, const Thresholds &th, const Refractory &rf, \
                     const EventSink &sink, unsigned long long *holes, const DebugOut &dbg, cudaStream_t st)
EVIS_DECL_RESOLVE(launch_resolve_m0);
EVIS_DECL_RESOLVE(launch_resolve_m0d);
EVIS_DECL_RESOLVE(launch_resolve_m1);
EVIS_DECL_RESOLVE(launch_resolve_m1d);
#undef EVIS_DECL_RESOLVE
// fill n floats with v (prep.cu)
cudaError_t launch_fill(float *p, long long n, float v, cudaStream_t st);

// ---- voxel grid / accumulation image (reading R30) ------------------------------------------
// V [E][2][bins][hc][wc] in 32.32 fixed point (integer atomics: the sum does not depend on the order of the adds).
// An event of polarity channel c (ON 0, OFF 1) at window time t adds 1 - w to bin b0 = floor(tau) and w to b0 + 1,
// tau = min((t_base + t_off) * scale, bins - 1), w = tau - b0: linear interpolation along the time axis.
struct VoxelSink {
    unsigned long long *v;      // null = off
    uint32_t bins, hc, wc;
    float t_base;               // start of this interval relative to the start of the window (j * T)
    float scale;                // (bins - 1) / (window_steps * T)
    int store_events;           // 0: the ordered stream is not written (voxels only); 1: 16-byte events; 2: 8-byte
                                // compact events (evis_event8, include/evis.h) at the same positions of the same buffer
    float dt;                   // T / S (compact events: the stamp is stored as a fraction of the substep)
};
// V -> float32 (out, same shape); normalize: every (env, channel, bin) plane divided by its maximum
cudaError_t launch_voxel_finish(const unsigned long long *v, float *out, uint32_t planes, uint32_t cells, int normalize,
                                cudaStream_t st);

// ---- a8 ordering (order.cu) ----------------------------------------------------------------------
// directory entry d = (arrival offset, count); ordered stream = chunks concatenated in d order, cut at
// `capacity` events.  *step_events = events of this step is added to *total_events (running total);
// *overflow_steps counts the steps whose events did not all fit (sticky).
constexpr int ORDER_ENTRIES_PER_BLOCK = 512;     // directory entries scanned and copied by one block
cudaError_t launch_order(const EventSink &sink, uint32_t num_entries, unsigned long long *scan_out /*[n]*/,
                         uint4 *ordered, unsigned long long capacity, const unsigned long long *step_events,
                         unsigned long long *total_events, unsigned long long *overflow_steps, const VoxelSink &vox, cudaStream_t st);
// The same for the global path's records: chunks are expanded to events (a7: timestamps) on the way.
// tiles_x, tiles = tiles per row / per frame of the G_TILE_W x G_TILE_H tiling; S = substeps.
cudaError_t launch_expand(const EventSink &sink, uint32_t num_entries, unsigned long long *scan_out, uint4 *ordered,
                          unsigned long long capacity, const unsigned long long *step_events,
                          unsigned long long *total_events, unsigned long long *overflow_steps, const EventParams &ep, const Thresholds &th, uint32_t W,
                          uint32_t HW, uint32_t margin, uint32_t tiles_x, uint32_t tiles, uint32_t S, const VoxelSink &vox, cudaStream_t st);
// ---- time-sorted per-env stream (sort.cu): stable segmented radix sort of the ordered stream by (env, t_off) -------
size_t sort_workspace_bytes(uint32_t E, unsigned long long capacity);
cudaError_t launch_time_sort(const uint2 *directory, uint32_t num_entries, int dir_shift, uint32_t E, unsigned long long capacity,
                             uint4 *a /* ordered stream, sorted in place */, uint4 *b /* scratch, same size */, void *ws,
                             cudaStream_t st);
// number of values among theta[0..n) that are not (finite and > 0), added to *bad (prep.cu)
cudaError_t launch_check_positive(const float *theta, long long n, unsigned long long *bad, cudaStream_t st);

}  // namespace evis
