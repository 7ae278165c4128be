/*
 * evis_oracle.c -- ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, single-threaded CPU statement of what the EVIS per-pixel event-synthesis hot
 * path computes, written from the paper (/root/reference/PAPER.md, arxiv 2607.08098), Sec. 3.2
 * (HDR event formation, Eq. 3-4, lines 92-104) and Sec. 3.3 (bidirectional motion-vector
 * warping, Eq. 5-7).  It follows the algorithm step by step in the paper's order
 * and notation: no tiling, no fusion, no reordering.  It shares NO code with the CUDA path under
 * paper_2607_08098_b200/csrc and neither includes the other.  Only tests/, the smoke check of
 * __graft_entry__.py and the cpu_baseline / --impl reference legs of bench.py may call it.
 *
 * Precision.  The paper fixes none.  Floating point that DECIDES AN INTEGER (which pixel a
 * source lands on, which source wins the z-test, how many events fire, the carried reference
 * level that feeds the next count) is taken in the kernel's precision, IEEE binary32 with the
 * operation order written below (compile with -ffp-contract=off so that only the fmaf() calls
 * written here are fused).  The log-luminance is evaluated in binary64 and rounded once to
 * binary32.  Timestamps decide nothing and are computed in binary64 -- unless the refractory period
 * is on: then they decide which crossings are emitted and are computed in binary32 [R26].
 *
 * Readings of the paper where it is silent or ambiguous are listed in DESIGN.md ("Readings");
 * the tag [Rn] below names the reading a line depends on.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1 zero motion identity, P2 substep S reproduces
 * keyframe B, P3 integer translation, P4 8x8 gather-form brute force, P5 analytic two-rectangle
 * occlusion, P6-P10 event-count / residual / timestamp closed forms, P11 per-pixel thresholds (Eq. 8), P12 refractory period, P13 margin, P14 colour, P15 noise events,
 * P16 composite mode 1 (every case of the rule by hand; linear time ramp along a translation), P19 defocus (library
 * Gaussian filter, blur-before-log, holes held unblurred), P20 weighted front-surface splat (exact float64 gather form on
 * 8x8, closed forms).  UNPINNED by paper or
 * mathematics (fixed by DESIGN.md readings only): log base R1, epsilon R2, initial reference
 * level R6, nearest-pixel depth lookup R16, hole handling R20, the composite choice R19, and among the
 * non-idealities the choices of R26 (L_ref follows suppressed crossings) and R29 (Ibar's normalisation, stamps,
 * stream order, independence from the refractory period), of R31 (truncation radius ceil(3 sigma), replicated border) and of
 * R32 (the 1 % front-surface band, the mean taken in the log domain, the 2^-20 / 2^-24 grids of its integer sums).
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

#define EVO_EMPTY 0xFFFFFFFFFFFFFFFFull
#define EVO_NONE  0xFFFFFFFFu

typedef struct {
    int32_t env, x, y;      /* pixel */
    int32_t p;              /* polarity +1 / -1 */
    int32_t substep;        /* i in 1..S */
    int32_t k;              /* 1..n: which crossing inside this substep */
    int32_t kf;             /* index of the keyframe interval */
    int32_t pad;
    double  t_off;          /* seconds from the start of the interval */
} evo_event;

static uint32_t f32_bits(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }

/* ---- Eq. 3 + log -----------------------------------------------------------
 * I = 0.2126 R + 0.7152 G + 0.0722 B ;  L = log(I + eps), natural log [R1], I clamped at 0 [R3].
 * binary64, products and sums each rounded (no fma), summed left to right, one rounding to f32. */
/* Colour events: "Replacing I with individual R, G, B channels and applying the event model to each
 * independently produces color events."  channel = 0, 1, 2: I = that channel of the radiance, same clamp, same
 * log; everything downstream is unchanged, one independent run per channel [R28].                              */
void evo_log_channel(const float *rad /* [n][3] */, int64_t n, float eps, int channel, float *L /* [n] */)
{
    for (int64_t i = 0; i < n; ++i) {
        double I = (double)rad[3 * i + channel];
        if (!(I > 0.0)) I = 0.0;
        L[i] = (float)log(I + (double)eps);
    }
}

void evo_log_luminance(const float *rad /* [n][3] */, int64_t n, float eps, float *L /* [n] */)
{
    for (int64_t i = 0; i < n; ++i) {
        double r = (double)rad[3 * i + 0], g = (double)rad[3 * i + 1], b = (double)rad[3 * i + 2];
        double I = (0.2126 * r + 0.7152 * g) + 0.0722 * b;
        if (!(I > 0.0)) I = 0.0;
        L[i] = (float)log(I + (double)eps);
    }
}

/* ---- Eq. 5-7: splat one keyframe in one direction for one substep ---------
 * Source pixel p=(x,y) of keyframe X with displacement field `disp` and time weight w moves to
 *     q = p + w * disp(p)                                                     (Eq. 5)
 * direction B (src_is_B=1): disp = m_B (backward MV of B), w = 1-f   ->  q_B = p + (1-f) m_B
 * direction A (src_is_B=0): disp = -m_A (or the explicit forward field), w = f -> q_A = p - f m_A
 * The other endpoint of the correspondence is p + disp(p); its depth is looked up at the nearest
 * pixel of the other keyframe [R16], falling back to the source's own depth outside the image.
 *     Zt = (1-f) Z_A(p_A) + f Z_B(p_B)                                         (Eq. 7)
 * Every integer pixel with positive bilinear weight is covered [R14]; per target the smallest
 * (Zt bits, source index) is kept [R15] (Eq. 6: nearest surface only).
 * zbuf[H*W] must be EVO_EMPTY-initialised by the caller.                                        */
/* One source pixel (x, y) at substep i in one direction: landing position q (Eq. 5), interpolated depth zt (Eq. 7),
 * floor cell (x0, y0) and whether the +1 neighbours carry positive weight (hx, hy).  Returns 0 when the source is
 * skipped (invalid depth [R17] or a floor cell outside [-1, W-1] x [-1, H-1]).                                   */
static int evo_source(int H, int W, int i, int S, int src_is_B, const float *disp, const float *Zsrc, const float *Zoth,
                      int x, int y, float *qx_, float *qy_, float *zt_, int *x0_, int *y0_, int *hx_, int *hy_)
{
    const float f = (float)i / (float)S;
    const float g = 1.0f - f;
    const float w = src_is_B ? g : f;
    const int p = y * W + x;
    const float dx = disp[2 * p + 0], dy = disp[2 * p + 1];
    const float qx = fmaf(w, dx, (float)x);
    const float qy = fmaf(w, dy, (float)y);
    /* depth at the two endpoints of the correspondence */
    const float ex = (float)x + dx, ey = (float)y + dy;
    const float jx = floorf(ex + 0.5f), jy = floorf(ey + 0.5f);
    const float zs = Zsrc[p];
    float zo = zs;
    if (jx >= 0.0f && jx <= (float)(W - 1) && jy >= 0.0f && jy <= (float)(H - 1))
        zo = Zoth[(int)jy * W + (int)jx];
    const float za = src_is_B ? zo : zs;
    const float zb = src_is_B ? zs : zo;
    const float zt = fmaf(f, zb, g * za);
    if (!(zt > 0.0f) || isinf(zt)) return 0;                    /* [R17] */
    const float x0f = floorf(qx), y0f = floorf(qy);
    if (!(x0f >= -1.0f && x0f <= (float)(W - 1))) return 0;     /* also drops NaN/inf */
    if (!(y0f >= -1.0f && y0f <= (float)(H - 1))) return 0;
    *qx_ = qx; *qy_ = qy; *zt_ = zt;
    *x0_ = (int)x0f; *y0_ = (int)y0f;
    *hx_ = qx > x0f; *hy_ = qy > y0f;                           /* positive weight on the +1 neighbour */
    return 1;
}

void evo_splat(int H, int W, int i, int S, int src_is_B,
               const float *disp /* [H][W][2] */, const float *Zsrc, const float *Zoth,
               uint64_t *zbuf)
{
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            float qx, qy, zt; int x0, y0, hx, hy;
            if (!evo_source(H, W, i, S, src_is_B, disp, Zsrc, Zoth, x, y, &qx, &qy, &zt, &x0, &y0, &hx, &hy)) continue;
            const uint64_t key = ((uint64_t)f32_bits(zt) << 32) | (uint32_t)(y * W + x);
            for (int oy = 0; oy <= hy; ++oy)
                for (int ox = 0; ox <= hx; ++ox) {
                    const int tx = x0 + ox, ty = y0 + oy;
                    if (tx < 0 || tx >= W || ty < 0 || ty >= H) continue;   /* [R18] */
                    if (key < zbuf[ty * W + tx]) zbuf[ty * W + tx] = key;
                }
        }
}

/* ---- Weighted front-surface splat [R32] --------------------------------------------------------------
 * "These target values are then bilinearly interpolated to integer pixels.  When multiple sources land on the same
 * target, we resolve the occlusion with a per-pixel z-buffer that retains only the nearest surface."  Read as weights
 * (the alternative to [R14]'s winner-take-all): per direction and target q, with Z*(q) the z-buffer's depth (evo_splat),
 * the FRONT surface is the sources covering q whose depth is within 1 % of it, zt <= 1.01f * Z*, and the target takes
 * their bilinear-weighted mean
 *     Lhat_X(q) = sum_s W_s L_X(p_s) / sum_s W_s ,   w_s = (1 - |q.x - qs.x|)(1 - |q.y - qs.y|)  (binary32),
 * in the log domain like the blend of [R19]/[R23].  So that the sums do not depend on the order of the sources (the
 * kernel adds them with integer atomics) both are integers: W_s = max(1, rint(w_s 2^20)), L in units of 2^-24
 * (rint(L 2^24)); the quotient is taken in binary64 and rounded once to binary32.  acc[q] = {sum W L, sum W} must be
 * zeroed by the caller; zbuf = this direction's z-buffer of the same substep.                                      */
void evo_wsplat(int H, int W, int i, int S, int src_is_B, const float *disp, const float *Zsrc, const float *Zoth,
                const float *Lsrc, const uint64_t *zbuf, int64_t *acc /* [H*W][2] */)
{
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            float qx, qy, zt; int x0, y0, hx, hy;
            if (!evo_source(H, W, i, S, src_is_B, disp, Zsrc, Zoth, x, y, &qx, &qy, &zt, &x0, &y0, &hx, &hy)) continue;
            const float Lv = Lsrc[y * W + x];
            if (!(fabsf(Lv) < 120.0f)) continue;                /* a non-finite log value carries no weight */
            const int64_t Lq = (int64_t)rint((double)Lv * 16777216.0);
            const float fx = qx - (float)x0, fy = qy - (float)y0;            /* exact */
            for (int oy = 0; oy <= hy; ++oy)
                for (int ox = 0; ox <= hx; ++ox) {
                    const int tx = x0 + ox, ty = y0 + oy;
                    if (tx < 0 || tx >= W || ty < 0 || ty >= H) continue;   /* [R18] */
                    const uint64_t zk = zbuf[ty * W + tx];
                    float zmin; uint32_t zb_ = (uint32_t)(zk >> 32); memcpy(&zmin, &zb_, 4);
                    if (!(zt <= 1.01f * zmin)) continue;                     /* behind the front surface */
                    const float wx = ox ? fx : 1.0f - fx, wy = oy ? fy : 1.0f - fy;
                    const float w = wx * wy;
                    int64_t Wq = (int64_t)rint((double)w * 1048576.0);
                    if (Wq < 1) Wq = 1;
                    acc[2 * (ty * W + tx) + 0] += Wq * Lq;
                    acc[2 * (ty * W + tx) + 1] += Wq;
                }
        }
}

/* composite of the weighted mode: B primary, A fills B's holes, else hold [R19 mode 0, R20] */
void evo_wcomposite(int H, int W, const uint64_t *zA, const uint64_t *zB, const int64_t *accA, const int64_t *accB,
                    const float *Lprev, float *Lhat, uint8_t *win_dir, uint32_t *win_idx)
{
    for (int q = 0; q < H * W; ++q) {
        const int64_t *a = zB[q] != EVO_EMPTY ? accB + 2 * q : (zA[q] != EVO_EMPTY ? accA + 2 * q : 0);
        const uint8_t d = zB[q] != EVO_EMPTY ? 0 : (zA[q] != EVO_EMPTY ? 1 : 3);
        /* the nearest source always belongs to its own front surface, so a reached pixel has weight unless every
         * contributor's log value was non-finite: then it holds, like a hole                                     */
        if (a && a[1] > 0) Lhat[q] = (float)(((double)a[0] / (double)a[1]) / 16777216.0);
        else Lhat[q] = Lprev[q];
        if (win_dir) win_dir[q] = d;
        if (win_idx) win_idx[q] = d == 0 ? (uint32_t)zB[q] : (d == 1 ? (uint32_t)zA[q] : EVO_NONE);
    }
}

/* ---- composite -----------------------------------------------------------------
 * mode 0 [R19]: backward-warped B is primary; forward-warped A fills only B's holes; a pixel
 * reached by neither keeps its previous value [R20].
 * mode 1 [R19]: nearest of the two; where both hit the same surface (depths within 1 %) the two
 * log values are blended with the time weights of Eq. 7: (1-f) L_A* + f L_B*.
 * Out: Lhat[H*W]; win_dir[H*W] (0 = B, 1 = A, 2 = blend, 3 = hole); win_idx[H*W] source index of
 * the chosen (mode 1 blend: the B) winner, EVO_NONE for a hole.                                   */
void evo_composite(int H, int W, int i, int S, int mode,
                   const uint64_t *zA, const uint64_t *zB, const float *LA, const float *LB,
                   const float *Lprev, float *Lhat, uint8_t *win_dir, uint32_t *win_idx)
{
    const float f = (float)i / (float)S;
    const float g = 1.0f - f;
    for (int q = 0; q < H * W; ++q) {
        const int hasA = zA[q] != EVO_EMPTY, hasB = zB[q] != EVO_EMPTY;
        const uint32_t ia = (uint32_t)(zA[q] & 0xFFFFFFFFu), ib = (uint32_t)(zB[q] & 0xFFFFFFFFu);
        float v; uint8_t d; uint32_t idx;
        if (mode == 0) {
            if (hasB)      { v = LB[ib]; d = 0; idx = ib; }
            else if (hasA) { v = LA[ia]; d = 1; idx = ia; }
            else           { v = Lprev[q]; d = 3; idx = EVO_NONE; }
        } else {
            if (hasA && hasB) {
                float da, db;
                uint32_t ua = (uint32_t)(zA[q] >> 32), ub = (uint32_t)(zB[q] >> 32);
                memcpy(&da, &ua, 4); memcpy(&db, &ub, 4);
                const float lo = da < db ? da : db;
                if (fabsf(da - db) <= 0.01f * lo) { v = fmaf(f, LB[ib], g * LA[ia]); d = 2; idx = ib; }
                else if (db < da)                 { v = LB[ib]; d = 0; idx = ib; }
                else                              { v = LA[ia]; d = 1; idx = ia; }
            }
            else if (hasB) { v = LB[ib]; d = 0; idx = ib; }
            else if (hasA) { v = LA[ia]; d = 1; idx = ia; }
            else           { v = Lprev[q]; d = 3; idx = EVO_NONE; }
        }
        Lhat[q] = v;
        if (win_dir) win_dir[q] = d;
        if (win_idx) win_idx[q] = idx;
    }
}

/* ---- Noise events (Eq. 9-10) [R29] --------------------------------------------------
 * "In each synthesis step of duration dt, a pixel leaks with probability P_leak = r_l dt" (spurious ON event);
 * shot noise: random-polarity events with P_shot = r_s dt (1 - Ibar), Ibar in [0,1] the normalized intensity;
 * hot pixels: a fixed subset H fires with P_hot = r_h dt.  The draws come from a counter-based generator that
 * the CUDA path implements too (same integers on both sides):
 *   mix64 = the splitmix64 finalizer;  key(q) = mix64(mix64(mix64(seed ^ G (kf + 1)) + env) + q), q = y W + x;
 *   h_s = mix64(key + 4 i + s) for substep i and stream s = 0, 1, 2;  a 24-bit field u gives uf = u 2^-24.
 *   leak iff uf(h0 >> 40) < r_l dt;  shot iff uf((h0 >> 16) & 0xFFFFFF) < (r_s dt)(1 - Ibar), polarity h0 & 1;
 *   hot (pixels of H only) iff uf(h1 >> 40) < r_h dt, polarity h0 & 2.
 * Stamps: uniform in the substep, t = fma(uf, dt, (i - 1) dt), fields h2 >> 40 (leak), (h2 >> 16) & 0xFFFFFF
 * (shot), (h1 >> 16) & 0xFFFFFF (hot).  Ibar = clamp((exp(L) - eps) / I_white, 0, 1) with L the frame's log
 * value and exp32 below (binary32 with a fixed operation order, so that both sides decide alike).  Noise events
 * follow the pixel's threshold crossings of the substep in the order leak, shot, hot; they leave L_ref alone,
 * and they neither see nor feed the refractory period.                                                       */
typedef struct {
    uint64_t seed;
    float r_leak, r_shot, r_hot;     /* rates in Hz, >= 0 */
    float i_white;                   /* intensity that normalizes to 1 */
    float eps;                       /* the log epsilon */
    const uint8_t *hot;              /* [H*W] membership of H for this env, or NULL */
} evo_noise;

static uint64_t evo_mix64(uint64_t z)
{
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}

uint64_t evo_noise_key(uint64_t seed, int kf, int env, int64_t q)
{
    uint64_t z = evo_mix64(seed ^ (0x9E3779B97F4A7C15ull * (uint64_t)(kf + 1)));
    z = evo_mix64(z + (uint64_t)env);
    return evo_mix64(z + (uint64_t)q);
}

uint64_t evo_noise_hash(uint64_t key, int i, int s) { return evo_mix64(key + 4ull * (uint64_t)i + (uint64_t)s); }

/* exp in binary32, every operation written out: x = k ln2 + r, |r| <= ln2 / 2, Taylor to r^7 by Horner with fma,
 * scaled by 2^k through the exponent field.  Relative error ~2e-7 on [-80, 80]; outside it saturates.          */
float evo_exp32(float x)
{
    if (!(x > -80.0f)) return 0.0f;
    if (x > 80.0f) x = 80.0f;
    const float kf = rintf(x * 1.44269504f);
    float r = fmaf(kf, -0.693145752f, x);          /* ln2 split in two binary32 parts */
    r = fmaf(kf, -1.42860677e-06f, r);
    float p = 1.98412698e-4f;                       /* 1/7! ... 1/2!, 1, 1 */
    p = fmaf(p, r, 1.38888889e-3f);
    p = fmaf(p, r, 8.33333333e-3f);
    p = fmaf(p, r, 4.16666667e-2f);
    p = fmaf(p, r, 1.66666667e-1f);
    p = fmaf(p, r, 0.5f);
    p = fmaf(p, r, 1.0f);
    p = fmaf(p, r, 1.0f);
    uint32_t bits; memcpy(&bits, &p, 4);
    bits += (uint32_t)((int32_t)kf << 23);         /* p in [0.7, 1.5]: the exponent field cannot wrap for |k| <= 116 */
    memcpy(&p, &bits, 4);
    return p;
}

/* ---- Eq. 4 + reference update for one frame of one env ------------------------
 * dL = L - Lref ; n = floor(|dL| / C) ; p = sgn(dL) ; Lref <- Lref + p n C.
 * C = C+ for dL > 0, C- for dL < 0 [R4]; n capped at 255 [R7]; the k-th crossing of the frame is
 * stamped by linear interpolation in log intensity between the previous and the current frame
 * value [R8]: level_k = Lref + p k C, fr = (level_k - Lprev) / (L - Lprev) clamped to [0,1].
 * Frame i covers ((i-1) T/S, i T/S].  Events are appended in (y, x, k) order.
 * Threshold mismatch (Eq. 8): "the scalar threshold C is replaced by per-pixel ON/OFF
 * thresholds ... sampled once per pixel".  The maps are INPUTS (the caller draws them); th_on[q] replaces C+
 * and th_off[q] replaces C- at pixel q, everything else is unchanged [R25].
 * Returns the number of events this frame produced (all are counted; only those that fit are
 * stored).                                                                                        */
int64_t evo_event_frame(int H, int W, int env, int kf, int i, int S, float T,
                        float c_pos, float c_neg,
                        const float *th_on, const float *th_off,   /* [H*W] or NULL (both): Eq. 8 maps */
                        float tau_r, float *t_last,                /* refractory period (<= 0: off) and its state */
                        const evo_noise *noise,                    /* noise events (NULL: off) */
                        const float *Lhat,
                        float *Lref, float *Lprev,
                        evo_event *ev, int64_t cap, int64_t n_have,
                        float *dbg_dL /* [H*W] or NULL: dL = L - Lref before the update */)
{
    int64_t made = 0;
    const double dt = (double)T / (double)S;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            const int q = y * W + x;
            const float L = Lhat[q];
            const float d = L - Lref[q];
            if (dbg_dL) dbg_dL[q] = d;
            float C; int p;
            if (d > 0.0f)      { C = th_on ? th_on[q] : c_pos; p = +1; }     /* theta_ON(u),  Eq. 8 */
            else if (d < 0.0f) { C = th_off ? th_off[q] : c_neg; p = -1; }   /* theta_OFF(u), Eq. 8 */
            else               { C = 1.0f;  p = 0; }
            int n = 0;
            if (p != 0) {
                float r = floorf(fabsf(d) / C);
                n = r >= 255.0f ? 255 : (int)r;
            }
            for (int k = 1; k <= n; ++k) {
                /* the k-th crossing of this frame: level_k = Lref + p k C, placed at the fraction fr of the frame
                 * where the line from Lprev to L reaches it [R8]; fr = 1 when the frame did not move.            */
                const float lev = fmaf((float)(p * k), C, Lref[q]);
                double t;
                if (tau_r > 0.0f) {
                    /* Refractory period [R26]: the stamp now decides an integer (emitted or not), so
                     * it is taken in binary32 with this operation order; the crossing is emitted iff
                     * t - t_last >= tau_r, t_last = stamp of the pixel's last EMITTED event, kept relative to the
                     * start of the current interval.  L_ref follows every crossing, emitted or not (Eq. 4).      */
                    const float dtf = T / (float)S;
                    const float num = lev - Lprev[q], den = L - Lprev[q];
                    float fr = 1.0f;
                    if (den != 0.0f) fr = num / den;
                    if (!(fr >= 0.0f)) fr = 0.0f;
                    if (fr > 1.0f) fr = 1.0f;
                    const float tf = fmaf(fr, dtf, (float)(i - 1) * dtf);
                    if (!(tf - t_last[q] >= tau_r)) continue;         /* suppressed */
                    t_last[q] = tf;
                    t = (double)tf;
                } else {
                    /* the stamp decides nothing: binary64 */
                    const double den = (double)L - (double)Lprev[q];
                    double fr = 1.0;
                    if (den != 0.0) fr = ((double)lev - (double)Lprev[q]) / den;
                    if (!(fr >= 0.0)) fr = 0.0;
                    if (fr > 1.0) fr = 1.0;
                    t = ((double)(i - 1) + fr) * dt;
                }
                if (n_have + made < cap) {
                    evo_event *o = &ev[n_have + made];
                    o->env = env; o->x = x; o->y = y; o->p = p; o->substep = i; o->k = k;
                    o->kf = kf; o->pad = 0;
                    o->t_off = t;
                }
                ++made;
            }
            if (noise) {                                             /* Eq. 9-10 and hot pixels [R29] */
                const float dtf = T / (float)S, t0 = (float)(i - 1) * dtf, U = 5.9604644775390625e-08f; /* 2^-24 */
                const uint64_t key = evo_noise_key(noise->seed, kf, env, q);
                const uint64_t h0 = evo_noise_hash(key, i, 0), h1 = evo_noise_hash(key, i, 1), h2 = evo_noise_hash(key, i, 2);
                int np_[3], nk = 0; float nt[3]; int nkind[3];
                if ((float)(h0 >> 40) * U < noise->r_leak * dtf) {
                    np_[nk] = +1; nt[nk] = fmaf((float)(h2 >> 40) * U, dtf, t0); nkind[nk++] = 1001;
                }
                const float ps = noise->r_shot * dtf, us = (float)((h0 >> 16) & 0xFFFFFFu) * U;
                if (us < ps) {
                    float ibar = (evo_exp32(L) - noise->eps) / noise->i_white;
                    if (!(ibar >= 0.0f)) ibar = 0.0f;
                    if (ibar > 1.0f) ibar = 1.0f;
                    if (us < ps * (1.0f - ibar)) {
                        np_[nk] = (h0 & 1u) ? +1 : -1; nt[nk] = fmaf((float)((h2 >> 16) & 0xFFFFFFu) * U, dtf, t0); nkind[nk++] = 1002;
                    }
                }
                if (noise->hot && noise->hot[q] && (float)(h1 >> 40) * U < noise->r_hot * dtf) {
                    np_[nk] = (h0 & 2u) ? +1 : -1; nt[nk] = fmaf((float)((h1 >> 16) & 0xFFFFFFu) * U, dtf, t0); nkind[nk++] = 1003;
                }
                for (int a = 0; a < nk; ++a) {
                    if (n_have + made < cap) {
                        evo_event *o = &ev[n_have + made];
                        o->env = env; o->x = x; o->y = y; o->p = np_[a]; o->substep = i; o->k = nkind[a];
                        o->kf = kf; o->pad = 0;
                        o->t_off = (double)nt[a];
                    }
                    ++made;
                }
            }
            if (n > 0) Lref[q] = fmaf((float)(p * n), C, Lref[q]);
            Lprev[q] = L;
        }
    return made;
}

/* ---- Defocus [R31] ------------------------------------------------------------------------------
 * "Prior to the event generation, the linear intensity is convolved with a separable Gaussian kernel."
 * The frame the event model sees at every substep is the warped frame in LINEAR intensity, blurred, then logged:
 *   I_X[p]  = (float) max(0, 0.2126 R + 0.7152 G + 0.0722 B)        (binary64 sums as in Eq. 3, rounded once; or the
 *                                                                     chosen channel for colour events)
 *   Ihat_i  = the composite of Sec. 3.3 applied to I_A, I_B (values are copied, so the winners are those of the
 *             log path); a pixel reached by neither keyframe holds its previous UNBLURRED value Ihat_{i-1} [R20]
 *   Iblur_i = G_sigma * Ihat_i, separable: rows first, then columns; taps k = -R..R, R = ceil(3 sigma),
 *             w_k = exp(-k^2 / (2 sigma^2)) / sum (binary64, rounded to binary32); the border replicates the edge
 *             pixel; every pass accumulates in binary32, acc = fmaf(w_k, v_k, acc) for k = -R..R in that order
 *   L_i     = (float) log((double) Iblur_i + eps)                    -> Eq. 4
 * With a margin the blur runs on the whole over-rendered frame and the crop follows.                              */
void evo_linear_luminance(const float *rad /* [n][3] */, int64_t n, int channel /* -1: Rec.709 */, float *I /* [n] */)
{
    for (int64_t i = 0; i < n; ++i) {
        double v;
        if (channel >= 0) v = (double)rad[3 * i + channel];
        else {
            double r = (double)rad[3 * i + 0], g = (double)rad[3 * i + 1], b = (double)rad[3 * i + 2];
            v = (0.2126 * r + 0.7152 * g) + 0.0722 * b;
        }
        if (!(v > 0.0)) v = 0.0;
        I[i] = (float)v;
    }
}

/* taps of the Gaussian: returns R = ceil(3 sigma) (0 for sigma <= 0) and fills w[0 .. 2R] for k = -R .. R */
int evo_gauss_taps(float sigma, float *w, int max_taps)
{
    if (!(sigma > 0.0f)) { w[0] = 1.0f; return 0; }
    int R = (int)ceil(3.0 * (double)sigma);
    if (2 * R + 1 > max_taps) return -1;
    double sum = 0.0;
    for (int k = -R; k <= R; ++k) sum += exp(-(double)(k * k) / (2.0 * (double)sigma * (double)sigma));
    for (int k = -R; k <= R; ++k) w[k + R] = (float)(exp(-(double)(k * k) / (2.0 * (double)sigma * (double)sigma)) / sum);
    return R;
}

void evo_blur(int H, int W, int R, const float *w, const float *src, float *tmp /* [H*W] scratch */, float *dst)
{
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            float acc = 0.0f;
            for (int k = -R; k <= R; ++k) {
                int xx = x + k; if (xx < 0) xx = 0; if (xx > W - 1) xx = W - 1;
                acc = fmaf(w[k + R], src[y * W + xx], acc);
            }
            tmp[y * W + x] = acc;
        }
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            float acc = 0.0f;
            for (int k = -R; k <= R; ++k) {
                int yy = y + k; if (yy < 0) yy = 0; if (yy > H - 1) yy = H - 1;
                acc = fmaf(w[k + R], tmp[yy * W + x], acc);
            }
            dst[y * W + x] = acc;
        }
}

/* ---- one keyframe interval of one env: A -> B, substeps i = 1..S ------------------------------
 * i < S are the paper's K-1 intermediates (f = i/K); i = S is keyframe B itself [R10].
 * fwdA: displacement of A's pixels towards B: -m_A or the explicit forward field.
 * Optional debug outputs, each [S][H*W] or NULL: winners of each direction, composite, Lhat.
 * margin: H x W is the OVER-RENDERED frame (Supp. B 317-319); the warp runs on all of it and the
 * caller crops `margin` pixels off each side afterwards (evis_oracle.py); here it only restricts the hole count. */
int64_t evo_interval(int H, int W, int S, int mode, int env, int kf, int margin, float T, float c_pos, float c_neg,
                     const float *th_on, const float *th_off,              /* [H*W] or NULL: Eq. 8 maps of this env */
                     float tau_r, float *t_last,                           /* refractory period (<= 0: off), state [H*W] */
                     const evo_noise *noise,                               /* noise events of this env (NULL: off) */
                     const float *LA, const float *fwdA, const float *ZA,
                     const float *LB, const float *mB, const float *ZB,
                     float *Lref, float *Lprev,
                     uint64_t *zA, uint64_t *zB, float *Lhat,              /* scratch [H*W] each */
                     evo_event *ev, int64_t cap, int64_t n_have,
                     uint32_t *dbg_winA, uint32_t *dbg_winB, uint8_t *dbg_dir, uint32_t *dbg_idx,
                     float *dbg_Lhat, float *dbg_dL, int64_t *holes,
                     /* defocus [R31]: blur_R < 0 = off (everything below unused).  IA / IB: linear intensity of the keyframes,
                      * Iprev: carried unblurred warped frame, eps: the log epsilon, scratch [H*W] each */
                     int blur_R, const float *blur_w, const float *IA, const float *IB, float *Iprev, float eps,
                     float *blur_tmp, float *blur_out,
                     /* mode 2 (weighted front-surface splat [R32]): scratch [H*W][2] each, else unused */
                     int64_t *waccA, int64_t *waccB)
{
    const int64_t P = (int64_t)H * W;
    int64_t made = 0;
    for (int i = 1; i <= S; ++i) {
        for (int64_t q = 0; q < P; ++q) { zA[q] = EVO_EMPTY; zB[q] = EVO_EMPTY; }
        evo_splat(H, W, i, S, 0, fwdA, ZA, ZB, zA);
        evo_splat(H, W, i, S, 1, mB, ZB, ZA, zB);
        uint8_t *dd = dbg_dir ? dbg_dir + (int64_t)(i - 1) * P : 0;
        uint32_t *di = dbg_idx ? dbg_idx + (int64_t)(i - 1) * P : 0;
        if (mode == 2) {
            /* weighted front-surface splat [R32]: a second walk over the sources against the finished z-buffers */
            for (int64_t q = 0; q < 2 * P; ++q) { waccA[q] = 0; waccB[q] = 0; }
            evo_wsplat(H, W, i, S, 0, fwdA, ZA, ZB, LA, zA, waccA);
            evo_wsplat(H, W, i, S, 1, mB, ZB, ZA, LB, zB, waccB);
            evo_wcomposite(H, W, zA, zB, waccA, waccB, Lprev, Lhat, dd, di);
        } else if (blur_R < 0) {
            evo_composite(H, W, i, S, mode, zA, zB, LA, LB, Lprev, Lhat, dd, di);
        } else {
            /* defocus: composite the LINEAR frame (holes hold the previous unblurred value), blur it, take the log */
            evo_composite(H, W, i, S, mode, zA, zB, IA, IB, Iprev, blur_out, dd, di);
            for (int64_t q = 0; q < P; ++q) Iprev[q] = blur_out[q];
            evo_blur(H, W, blur_R, blur_w, Iprev, blur_tmp, blur_out);
            for (int64_t q = 0; q < P; ++q) Lhat[q] = (float)log((double)blur_out[q] + (double)eps);
        }
        for (int64_t q = 0; q < P; ++q) {
            if (dbg_winA) dbg_winA[(int64_t)(i - 1) * P + q] = zA[q] == EVO_EMPTY ? EVO_NONE : (uint32_t)zA[q];
            if (dbg_winB) dbg_winB[(int64_t)(i - 1) * P + q] = zB[q] == EVO_EMPTY ? EVO_NONE : (uint32_t)zB[q];
            if (dbg_Lhat) dbg_Lhat[(int64_t)(i - 1) * P + q] = Lhat[q];
            if (holes && zA[q] == EVO_EMPTY && zB[q] == EVO_EMPTY) {
                /* over-render margin [R27]: only the pixels kept by the crop count */
                const int qx = (int)(q % W), qy = (int)(q / W);
                if (qx >= margin && qx < W - margin && qy >= margin && qy < H - margin) ++*holes;
            }
        }
        made += evo_event_frame(H, W, env, kf, i, S, T, c_pos, c_neg, th_on, th_off, tau_r, t_last, noise, Lhat, Lref, Lprev,
                                ev, cap, n_have + made, dbg_dL ? dbg_dL + (int64_t)(i - 1) * P : 0);
    }
    /* the next interval starts T later: keep t_last relative to its start (binary32, -inf stays -inf) [R26] */
    if (tau_r > 0.0f)
        for (int64_t q = 0; q < P; ++q) t_last[q] = t_last[q] - T;
    return made;
}
