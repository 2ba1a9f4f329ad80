// placeholder: filled in by the quad kernel
#include "bg_internal.h"
namespace bg {
bool cdbg_quad_supported(int) { return false; }
size_t cdbg_quad_current_bytes(int) { return 0; }
cudaError_t cdbg_quad_launch(cudaStream_t, int, int, long long, const double*, const signed char*, const signed char*,
                             double*) { return cudaErrorNotSupported; }
}  // namespace bg
