// NV = 6 (3-D, one passive scalar): runtime-switch build only.
#include "hx_step_tile2_launch.cuh"
namespace hx {
namespace t2 {
template <>
cudaError_t launch_nv<6>(Plan& plan, const Args& a, int cur, cudaStream_t st) {
  return launch_generic<6>(plan, a, cur, st);
}
}  // namespace t2
}  // namespace hx
