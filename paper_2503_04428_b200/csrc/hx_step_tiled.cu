// hx_step_tiled.cu -- fused tile kernel (placeholder until the TMA z-marching kernel lands).
#include "hx_common.cuh"

namespace hx {
struct TiledPlan { int unused; };
int tiled_supported(const Layout&, const Phys&) { return 0; }
cudaError_t tiled_plan_create(const Layout&, const Phys&, double* const*, TiledPlan** out) { *out = nullptr; return cudaErrorNotSupported; }
void tiled_plan_destroy(TiledPlan* p) { delete p; }
cudaError_t launch_step_tiled(TiledPlan*, const StepArgs&, int, cudaStream_t) { return cudaErrorNotSupported; }
const char* tiled_kernel_name(const TiledPlan*) { return "tiled"; }
}  // namespace hx
