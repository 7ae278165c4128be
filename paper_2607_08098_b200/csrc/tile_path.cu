// tile_path.cu -- rows a2-a8 fused per target tile with z-buffers in shared memory (bounded motion).
// Not built yet: plan_tile() declines, so every configuration runs the global z-buffer path.
#include "kernels.h"

namespace evis {

bool plan_tile(const Geom &, float, TilePlan *) { return false; }
cudaError_t tile_setup(const Geom &, const TilePlan &) { return cudaSuccess; }
cudaError_t launch_tile(const Geom &, const TilePlan &, const Keyframe &, const Keyframe &, const SubstepTable *,
                        float *, float *, const EventParams &, const EventSink &, unsigned long long *,
                        unsigned long long *, const DebugOut &, cudaStream_t)
{
    return cudaErrorNotSupported;
}

}  // namespace evis
