// Fused single-pass Gaussian smoothing (placeholder until the tiled kernel lands).
#include "kernels.h"

namespace demons {
int launch_smooth_fused(const SmoothArgs&, cudaStream_t) { return 0; }
}  // namespace demons
