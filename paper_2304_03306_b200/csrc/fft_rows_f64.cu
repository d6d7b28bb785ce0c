// row-pass kernels, scalar = double
#define TTSH_BUILD_ROWS
#include "engine_fft.cuh"
namespace ttsh {
template cudaError_t launch_inv_row<double>(const Geom&, const Batch&, int, const void*, const void*, const double*, cudaStream_t, int, size_t);
template cudaError_t launch_fwd_row<double>(const Geom&, const Batch&, int, const void*, const void*, cudaStream_t, int, size_t);
template cudaError_t prepare_rows<double>(const Geom&);
template cudaError_t launch_fwd_row_fused<double>(const Geom&, const Model&, const void*, const void*, const void*, const void*, void*, void*, const void*, cudaStream_t);
}
