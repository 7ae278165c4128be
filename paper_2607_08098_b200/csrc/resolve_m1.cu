// resolve_m1.cu -- k_resolve_global, composite mode 1: 16 variants (key layout, TMA, thresholds, direct mode).
#include "resolve_kernel.cuh"

namespace evis {

cudaError_t launch_resolve_m1(const Geom &g, const ZChunk &zc, const Keyframe &A, const Keyframe &B,
                              const SubstepTable &tab, float *l_ref, float *l_prev, const EventParams &ep,
                              const Thresholds &th, const Refractory &rf, const EventSink &sink,
                              unsigned long long *holes, const DebugOut &dbg, cudaStream_t st)
{
    return launch_resolve_md<1, false>(g, zc, A, B, tab, l_ref, l_prev, ep, th, rf, sink, holes, dbg, st);
}

}  // namespace evis
