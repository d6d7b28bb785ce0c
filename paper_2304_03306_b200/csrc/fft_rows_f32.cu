// row-pass kernels, scalar = float
#define TTSH_BUILD_ROWS
#include "engine_fft.cuh"
namespace ttsh {
template cudaError_t launch_inv_row<float>(const Geom&, const Batch&, int, const void*, const void*, const double*, cudaStream_t, int, size_t);
template cudaError_t launch_fwd_row<float>(const Geom&, const Batch&, int, const void*, const void*, cudaStream_t, int, size_t);
template cudaError_t prepare_rows<float>(const Geom&);
template cudaError_t launch_fwd_row_fused<float>(const Geom&, const Model&, const void*, const void*, const void*, const void*, void*, void*, const void*, cudaStream_t);
}
