// fused row-step kernel, scalar = float
#define TTSH_BUILD_ROWSTEP
#include "engine_fft.cuh"
namespace ttsh {
template cudaError_t launch_row_step<float>(const Geom&, const Model&, const void*, const void*, const void*, const void*, void*, void*, const void*, const double*, cudaStream_t, int);
template cudaError_t prepare_row_step<float>(const Geom&, int*, int*, int*);
template cudaError_t launch_row_step_tan<float>(const Geom&, const Model&, const void*, const void*, const void*, const void*, void*, void*, const void*, const double*, cudaStream_t, int, size_t, int, const void*, const void*, const void*);
template cudaError_t launch_row_step_ens<float>(const Geom&, const Model&, const void*, const void*, const void*, const void*, void*, void*, const void*, const double*, cudaStream_t, int, size_t, int);
template bool row_step_supported<float>(const Geom&);
template bool row_step_is_real<float>(const Geom&);
template int row_step_real_tabr<float>(const Geom&);
}
