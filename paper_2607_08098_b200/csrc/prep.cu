// prep.cu -- row a1 of the hot path: radiance -> log-luminance, once per keyframe pixel, fused
// with taking ownership of the keyframe's motion vectors and depth (a9: this keyframe is the next
// step's A, and the caller may free its tensors as soon as this kernel has run).
//
//   I = 0.2126 R + 0.7152 G + 0.0722 B        (Eq. 3)
//   L = log(I + eps), natural log, I clamped at 0   (R1, R3)
//
// Evaluated in binary64 with every product and sum rounded separately (no fma), summed left to
// right, and rounded once to binary32 -- the arithmetic contract of DESIGN.md Sec. 2.
//
// HBM-bound streaming kernel: 24 B read (+8 with mv_fwd) and 16 B written (+8) per pixel, 128-bit
// loads and stores, four pixels per thread.
#include "kernels.h"

namespace evis {

// channel < 0: Rec.709 luminance (Eq. 3); 0 / 1 / 2: that channel alone -- colour events (R28)
// lin: the same intensity in LINEAR form, rounded once to binary32 (defocus, R31)
__device__ __forceinline__ float log_lum(float r, float g, float b, double eps, int channel, float &lin)
{
    double I = __dadd_rn(__dadd_rn(__dmul_rn(0.2126, (double)r), __dmul_rn(0.7152, (double)g)),
                         __dmul_rn(0.0722, (double)b));
    if (channel >= 0) I = (double)(channel == 0 ? r : (channel == 1 ? g : b));
    if (!(I > 0.0)) I = 0.0;
    lin = __double2float_rn(I);
    return __double2float_rn(log(__dadd_rn(I, eps)));
}

// VEC: all pointers 16-byte aligned and n % 4 == 0 -> thread handles 4 consecutive pixels.
template <bool VEC>
__global__ void __launch_bounds__(256)
k_prep(const float *__restrict__ rad, const float *__restrict__ mv, const float *__restrict__ fwd_in,
       const float *__restrict__ depth, long long n, float eps_f, int channel,
       float *__restrict__ L, float2 *__restrict__ mv_out, float2 *__restrict__ fwd_out,
       float *__restrict__ Z, float *__restrict__ l_ref, float *__restrict__ l_prev, float bound,
       unsigned long long *__restrict__ viol, float *__restrict__ lin_out /* nullable: linear intensity (defocus) */)
{
    bool over = false;       // a motion vector beyond the bound the caller declared (max_motion_px)
    const double eps = (double)eps_f;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (VEC) {
        const long long p = t * 4;
        if (p >= n) return;
        const float4 *r4 = reinterpret_cast<const float4 *>(rad + 3 * p);
        const float4 a = __ldcs(r4), b = __ldcs(r4 + 1), c = __ldcs(r4 + 2);
        float4 l, li;
        l.x = log_lum(a.x, a.y, a.z, eps, channel, li.x);
        l.y = log_lum(a.w, b.x, b.y, eps, channel, li.y);
        l.z = log_lum(b.z, b.w, c.x, eps, channel, li.z);
        l.w = log_lum(c.y, c.z, c.w, eps, channel, li.w);
        *reinterpret_cast<float4 *>(L + p) = l;
        if (lin_out) *reinterpret_cast<float4 *>(lin_out + p) = li;
        if (l_ref) {                                  // first keyframe: L_ref = L_prev = L   (R6)
            *reinterpret_cast<float4 *>(l_ref + p) = l;
            *reinterpret_cast<float4 *>(l_prev + p) = l;
        }
        const float4 *m4 = reinterpret_cast<const float4 *>(mv + 2 * p);
        float4 *mo = reinterpret_cast<float4 *>(mv_out + p);
        const float4 m0 = __ldcs(m4), m1 = __ldcs(m4 + 1);
        mo[0] = m0;
        mo[1] = m1;
        over = fmaxf(fmaxf(fmaxf(fabsf(m0.x), fabsf(m0.y)), fmaxf(fabsf(m0.z), fabsf(m0.w))),
                     fmaxf(fmaxf(fabsf(m1.x), fabsf(m1.y)), fmaxf(fabsf(m1.z), fabsf(m1.w)))) > bound;
        if (fwd_in) {
            const float4 *f4 = reinterpret_cast<const float4 *>(fwd_in + 2 * p);
            float4 *fo = reinterpret_cast<float4 *>(fwd_out + p);
            const float4 f0 = __ldcs(f4), f1 = __ldcs(f4 + 1);
            fo[0] = f0;
            fo[1] = f1;
            over |= fmaxf(fmaxf(fmaxf(fabsf(f0.x), fabsf(f0.y)), fmaxf(fabsf(f0.z), fabsf(f0.w))),
                          fmaxf(fmaxf(fabsf(f1.x), fabsf(f1.y)), fmaxf(fabsf(f1.z), fabsf(f1.w)))) > bound;
        }
        *reinterpret_cast<float4 *>(Z + p) = __ldcs(reinterpret_cast<const float4 *>(depth + p));
    } else {
        if (t >= n) return;
        float li;
        const float l = log_lum(rad[3 * t], rad[3 * t + 1], rad[3 * t + 2], eps, channel, li);
        L[t] = l;
        if (lin_out) lin_out[t] = li;
        if (l_ref) { l_ref[t] = l; l_prev[t] = l; }
        mv_out[t] = make_float2(mv[2 * t], mv[2 * t + 1]);
        over = fmaxf(fabsf(mv[2 * t]), fabsf(mv[2 * t + 1])) > bound;
        if (fwd_in) {
            fwd_out[t] = make_float2(fwd_in[2 * t], fwd_in[2 * t + 1]);
            over |= fmaxf(fabsf(fwd_in[2 * t]), fabsf(fwd_in[2 * t + 1])) > bound;
        }
        Z[t] = depth[t];
    }
    if (over) atomicAdd(viol, 1ull);        // rare by contract; reported as EVIS_ERR_MOTION_BOUND
}

static bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

cudaError_t launch_prep(const float *rad, const float *mv, const float *fwd, const float *depth, long long n,
                        float eps, int channel, float *L, float2 *mv_out, float2 *fwd_out, float *Z, float *l_ref,
                        float *l_prev, float bound, unsigned long long *viol, float *lin_out, cudaStream_t st)
{
    if (!(bound > 0.0f)) bound = __builtin_inff();      // no bound declared: nothing to check
    const bool vec = (n % 4 == 0) && aligned16(rad) && aligned16(mv) && aligned16(depth) && (!fwd || aligned16(fwd)) && (!lin_out || aligned16(lin_out));
    if (vec) {
        const long long threads = n / 4;
        k_prep<true><<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(rad, mv, fwd, depth, n, eps, channel, L, mv_out,
                                                                         fwd_out, Z, l_ref, l_prev, bound, viol, lin_out);
    } else {
        k_prep<false><<<(unsigned)((n + 255) / 256), 256, 0, st>>>(rad, mv, fwd, depth, n, eps, channel, L, mv_out,
                                                                    fwd_out, Z, l_ref, l_prev, bound, viol, lin_out);
    }
    return cudaGetLastError();
}

// Defocus (R31): the event model's first frame is the blurred keyframe as well: L_ref = L_prev =
// log(G * I + eps).  One thread per pixel; the row sums it needs are recomputed with the pass order of the reading
// (rows first, each rounded to binary32, then the column sum; replicated border; acc = fmaf(w_k, v_k, acc), k = -R..R).
__global__ void __launch_bounds__(256)
k_blur_log(const float *__restrict__ I, int E, int H, int W, const BlurTaps taps, float eps_f, float *__restrict__ l_ref,
           float *__restrict__ l_prev)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long HW = (long long)H * W;
    if (t >= (long long)E * HW) return;
    const int e = (int)(t / HW), p = (int)(t - (long long)e * HW), y = p / W, x = p - y * W;
    const float *src = I + (size_t)e * HW;
    const int R = taps.R;
    float acc = 0.0f;
    for (int ky = -R; ky <= R; ++ky) {
        const int yy = min(max(y + ky, 0), H - 1);
        float row = 0.0f;
        for (int kx = -R; kx <= R; ++kx) row = __fmaf_rn(taps.w[kx + R], __ldg(src + yy * W + min(max(x + kx, 0), W - 1)), row);
        acc = __fmaf_rn(taps.w[ky + R], row, acc);
    }
    const float l = __double2float_rn(log(__dadd_rn((double)acc, (double)eps_f)));
    l_ref[t] = l;
    l_prev[t] = l;
}

cudaError_t launch_blur_log(const float *I, int E, int H, int W, const BlurTaps &taps, float eps, float *l_ref, float *l_prev,
                            cudaStream_t st)
{
    const long long n = (long long)E * H * W;
    k_blur_log<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(I, E, H, W, taps, eps, l_ref, l_prev);
    return cudaGetLastError();
}

// Eq. 8 precondition: thresholds must be finite and > 0 (a zero threshold would fire without end)
__global__ void __launch_bounds__(256) k_check_positive(const float *__restrict__ theta, long long n, unsigned long long *bad)
{
    unsigned int mine = 0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float v = theta[i];
        if (!(v > 0.0f && v < __int_as_float(0x7f800000))) ++mine;
    }
    mine = __reduce_add_sync(0xFFFFFFFFu, mine);
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(bad, (unsigned long long)mine);
}

cudaError_t launch_check_positive(const float *theta, long long n, unsigned long long *bad, cudaStream_t st)
{
    const long long blocks = (n + 255) / 256;
    k_check_positive<<<(unsigned)(blocks < 4096 ? (blocks < 1 ? 1 : blocks) : 4096), 256, 0, st>>>(theta, n, bad);
    return cudaGetLastError();
}

__global__ void __launch_bounds__(256) k_fill(float *__restrict__ p, long long n, float v)
{
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) p[i] = v;
}

cudaError_t launch_fill(float *p, long long n, float v, cudaStream_t st)
{
    const long long blocks = (n + 255) / 256;
    k_fill<<<(unsigned)(blocks < 4096 ? (blocks < 1 ? 1 : blocks) : 4096), 256, 0, st>>>(p, n, v);
    return cudaGetLastError();
}

}  // namespace evis
