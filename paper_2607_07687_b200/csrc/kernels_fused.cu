// kernels_fused.cu -- tiled fast path (placeholder: nothing supported yet).
#include "stencil.cuh"
namespace gmgf {
bool sweep_supported(const LevelGeom&) { return false; }
void rb_sweep(const LevelGeom&, const float*, const float*, float*, const float*, const float*, int,
              const float*, cudaStream_t) {}
bool resrestrict_supported(const LevelGeom&) { return false; }
void residual_restrict(const LevelGeom&, const float*, const float*, const float*, float*, float*,
                       cudaStream_t) {}
int configure() { return 0; }
}  // namespace gmgf
