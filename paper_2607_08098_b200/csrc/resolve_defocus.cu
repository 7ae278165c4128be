// resolve_defocus.cu -- k_resolve_global's two defocus passes (R31) and the event pass of the weighted
// front-surface splat (R32): 8 + 8 + 8 variants.
#include "resolve_kernel.cuh"

namespace evis {

cudaError_t launch_resolve_frames(const Geom &g, const ZChunk &zc, const float *IA, const float *IB, const SubstepTable &tab,
                                  float *i_prev, const EventParams &ep, unsigned long long *holes, const DebugOut &dbg,
                                  const FrameIO &fio, cudaStream_t st)
{
    return dbg.win ? launch_resolve_frames_d<true>(g, zc, IA, IB, tab, i_prev, ep, holes, dbg, fio, st)
                   : launch_resolve_frames_d<false>(g, zc, IA, IB, tab, i_prev, ep, holes, dbg, fio, st);
}

cudaError_t launch_resolve_blurred(const Geom &g, const ZChunk &zc, const SubstepTable &tab, float *l_ref, float *l_prev,
                                   const EventParams &ep, const Thresholds &th, const Refractory &rf, const EventSink &sink,
                                   unsigned long long *holes, const DebugOut &dbg, const FrameIO &fio, cudaStream_t st)
{
    return dbg.win ? launch_resolve_blurred_d<true, 2>(g, zc, tab, l_ref, l_prev, ep, th, rf, sink, holes, dbg, fio, st)
                   : launch_resolve_blurred_d<false, 2>(g, zc, tab, l_ref, l_prev, ep, th, rf, sink, holes, dbg, fio, st);
}

// the weighted front-surface splat's event pass (R32): fio.wacc holds the sums
cudaError_t launch_resolve_weighted(const Geom &g, const ZChunk &zc, const SubstepTable &tab, float *l_ref, float *l_prev,
                                    const EventParams &ep, const Thresholds &th, const Refractory &rf, const EventSink &sink,
                                    unsigned long long *holes, const DebugOut &dbg, const FrameIO &fio, cudaStream_t st)
{
    return dbg.win ? launch_resolve_blurred_d<true, 3>(g, zc, tab, l_ref, l_prev, ep, th, rf, sink, holes, dbg, fio, st)
                   : launch_resolve_blurred_d<false, 3>(g, zc, tab, l_ref, l_prev, ep, th, rf, sink, holes, dbg, fio, st);
}

}  // namespace evis
