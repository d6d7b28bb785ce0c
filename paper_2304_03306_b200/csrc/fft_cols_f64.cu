// column-pass kernels, scalar = double
#define TTSH_BUILD_COLS
#include "engine_fft.cuh"
namespace ttsh {
template cudaError_t launch_inv_col<double>(const Geom&, const Batch&, int, const void*, const void*, const double*, cudaStream_t, int, size_t);
template cudaError_t launch_fwd_col<double>(const Geom&, const Batch&, int, const void*, const void*, cudaStream_t, int, size_t);
template cudaError_t prepare_cols<double>(const Geom&);
template bool col_step_supported<double>(const Geom&);
template cudaError_t launch_col_step<double>(const Geom&, const Model&, const void*, const void*, void*, void*, double*, void*, void*, void*, const void*, const void*, cudaStream_t, int, size_t);
}
