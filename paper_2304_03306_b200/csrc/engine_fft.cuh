// engine_fft.cuh — size dispatch for the FFT pass kernels (included by the per-dtype translation units).
#pragma once
#include "engine.h"
#include "fft_passes.cuh"

namespace ttsh {

#define TTSH_FOR_SIZES(X) X(64) X(128) X(256) X(512) X(1024) X(2048) X(4096) X(8192)
// Ny = 16384 (Fig. 6(f)): half-length column transforms of 8192 points, one column per CTA.
// Nx = 16384: one real row per half-length complex transform (fft_rows_real.cuh) instead of packed row pairs.
#define TTSH_FOR_COL_SIZES(X) TTSH_FOR_SIZES(X) X(16384)
#define TTSH_REAL_ROW_NX 16384

template <typename K> static cudaError_t set_smem(K kernel, size_t bytes) {
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

#ifdef TTSH_BUILD_COLS
// the grouped variant is used when it still leaves at least one 128-thread CTA per SM
static int col_fill_ctas() {
  static int n = 0;
  if (n == 0) {
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    n = sms > 0 ? sms : 148;
  }
  return n;
}
template <typename T, int NY> static cudaError_t go_inv_col(const Geom& g, const Batch& b, int nf, const void* tab, const void* tabS, const double* v0, cudaStream_t s,
                                                            int members, size_t mstride) {
  using C = ColCfg<T, NY>;
  const long long items = (long long)g.NT * nf * members;
  constexpr int G = C::GMAX;
  if (G > 1 && 2 * items >= (long long)G * col_fill_ctas()) {          // several items per CTA once that still fills the GPU
    const long long ctas = (items + G - 1) / G;
    if (ctas > 65535) return cudaErrorInvalidValue;
    return launch_pdl(k_inv_col<T, NY, G>, dim3(2, (unsigned)ctas), dim3(G * C::THREADS), G * C::SMEM, s, g, b, static_cast<const cplx<T>*>(tab),
                      static_cast<const cplx<T>*>(tabS), v0, nf, members, mstride);
  }
  if (items > 65535) return cudaErrorInvalidValue;
  return launch_pdl(k_inv_col<T, NY, 1>, dim3(2, (unsigned)items), dim3(C::THREADS), C::SMEM, s, g, b, static_cast<const cplx<T>*>(tab),
                    static_cast<const cplx<T>*>(tabS), v0, nf, members, mstride);
}
template <typename T, int NY> static cudaError_t go_fwd_col(const Geom& g, const Batch& b, int nf, const void* tab, const void* tabS, cudaStream_t s,
                                                            int members, size_t mstride) {
  using C = ColCfg<T, NY>;
  const long long items = (long long)g.NT * nf * members;
  constexpr int G = C::GMAX;
  if (items > 0x3fffffffLL) return cudaErrorInvalidValue;
  if (G > 1 && items >= (long long)G * col_fill_ctas()) {
    return launch_pdl(k_fwd_col<T, NY, G>, dim3((unsigned)((items + G - 1) / G)), dim3(G * C::THREADS), G * C::SMEM, s, g, b,
                      static_cast<const cplx<T>*>(tab), static_cast<const cplx<T>*>(tabS), nf, members, mstride);
  }
  return launch_pdl(k_fwd_col<T, NY, 1>, dim3((unsigned)items), dim3(C::THREADS), C::SMEM, s, g, b, static_cast<const cplx<T>*>(tab),
                    static_cast<const cplx<T>*>(tabS), nf, members, mstride);
}
template <typename T> cudaError_t launch_inv_col(const Geom& g, const Batch& b, int nf, const void* tab, const void* tabS, const double* v0, cudaStream_t s,
                                                 int members, size_t mstride) {
  switch (g.Ny) {
#define X(N) case N: return go_inv_col<T, N>(g, b, nf, tab, tabS, v0, s, members, mstride);
    TTSH_FOR_COL_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
template <typename T> cudaError_t launch_fwd_col(const Geom& g, const Batch& b, int nf, const void* tab, const void* tabS, cudaStream_t s,
                                                 int members, size_t mstride) {
  switch (g.Ny) {
#define X(N) case N: return go_fwd_col<T, N>(g, b, nf, tab, tabS, s, members, mstride);
    TTSH_FOR_COL_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
}  // namespace ttsh
#include "col_step.cuh"
namespace ttsh {
template <typename T> bool col_step_supported(const Geom& g) {
  if (2 * g.My != g.Ny / 2 || g.Hy != g.Ny / 2 + 1) return false;      // 1/2 rule only
  switch (g.Ny) {
#define X(N) case N: return ColStepCfg<T, N>::OK;
    TTSH_FOR_SIZES(X)
#undef X
  }
  return false;
}
template <typename T, int NY> static cudaError_t go_col_step(const Geom& g, const Model& m, const void* srcA, const void* srcB, void* w, void* psi,
                                                            double* v0, void* dstW, void* dstPsi, void* dstVx, const void* tab, const void* tabS,
                                                            cudaStream_t s, int members, size_t mstride) {
  using S = ColStepCfg<T, NY>;
  if constexpr (!S::OK) return cudaErrorInvalidConfiguration;
  else {
    if (members < 1 || members > 65535) return cudaErrorInvalidValue;
    return launch_pdl(k_col_step<T, NY>, dim3(g.NT, members), dim3(S::THREADS), S::SMEM, s, g, m, (const cplx<T>*)srcA, (const cplx<T>*)srcB,
                      (cplx<T>*)w, (cplx<T>*)psi, v0, (cplx<T>*)dstW, (cplx<T>*)dstPsi, (cplx<T>*)dstVx, static_cast<const cplx<T>*>(tab),
                      static_cast<const cplx<T>*>(tabS), mstride);
  }
}
template <typename T> cudaError_t launch_col_step(const Geom& g, const Model& m, const void* srcA, const void* srcB, void* w, void* psi, double* v0,
                                                  void* dstW, void* dstPsi, void* dstVx, const void* tab, const void* tabS, cudaStream_t s,
                                                  int members, size_t mstride) {
  switch (g.Ny) {
#define X(N) case N: return go_col_step<T, N>(g, m, srcA, srcB, w, psi, v0, dstW, dstPsi, dstVx, tab, tabS, s, members, mstride);
    TTSH_FOR_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
template <typename T, int NY> static cudaError_t prep_col_step() {
  if constexpr (ColStepCfg<T, NY>::OK) return set_smem(k_col_step<T, NY>, ColStepCfg<T, NY>::SMEM);
  else return cudaSuccess;
}
template <typename T> cudaError_t prepare_cols(const Geom& g) {
  switch (g.Ny) {
#define X(N) case N: { using C = ColCfg<T, N>; \
                       cudaError_t e = prep_col_step<T, N>(); if (e != cudaSuccess) return e; \
                       e = set_smem(k_inv_col<T, N, 1>, C::SMEM); if (e != cudaSuccess) return e; \
                       e = set_smem(k_inv_col<T, N, C::GMAX>, C::GMAX * C::SMEM); if (e != cudaSuccess) return e; \
                       e = set_smem(k_fwd_col<T, N, C::GMAX>, C::GMAX * C::SMEM); if (e != cudaSuccess) return e; \
                       return set_smem(k_fwd_col<T, N, 1>, C::SMEM); }
    TTSH_FOR_COL_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
#endif

#ifdef TTSH_BUILD_ROWS
}  // namespace ttsh
#include "fft_rows_real.cuh"
namespace ttsh {
template <typename T, int NX> static cudaError_t go_inv_row_real(const Geom& g, const Batch& b, int nf, const void* tab, const void* tabR, const double* v0,
                                                                 cudaStream_t s, int members, size_t mstride) {
  using C = RealRowCfg<T, NX>;
  return launch_pdl(k_inv_row_real<T, NX>, dim3(g.Ny, nf, members), dim3(C::TPL), C::SMEM, s, g, b, static_cast<const cplx<T>*>(tab),
                    static_cast<const cplx<T>*>(tabR), v0, mstride);
}
template <typename T, int NX> static cudaError_t go_fwd_row_real(const Geom& g, const Batch& b, int nf, const void* tab, const void* tabR, cudaStream_t s,
                                                                 int members, size_t mstride) {
  using C = RealRowCfg<T, NX>;
  return launch_pdl(k_fwd_row_real<T, NX>, dim3(g.Ny, nf, members), dim3(C::TPL), C::SMEM, s, g, b, static_cast<const cplx<T>*>(tab),
                    static_cast<const cplx<T>*>(tabR), mstride);
}
template <typename T, int NX> static cudaError_t go_inv_row(const Geom& g, const Batch& b, int nf, const void* tab, const double* v0, cudaStream_t s,
                                                            int members, size_t mstride) {
  using C = RowCfg<T, NX>;
  dim3 grid((g.Ny / 2) / C::L, nf, members);
  return launch_pdl(k_inv_row<T, NX>, grid, dim3(C::THREADS), C::SMEM, s, g, b, static_cast<const cplx<T>*>(tab), v0, mstride);
}
template <typename T, int NX> static cudaError_t go_fwd_row(const Geom& g, const Batch& b, int nf, const void* tab, cudaStream_t s,
                                                            int members, size_t mstride) {
  using C = RowCfg<T, NX>;
  dim3 grid((g.Ny / 2) / C::L, nf, members);
  return launch_pdl(k_fwd_row<T, NX>, grid, dim3(C::THREADS), C::SMEM, s, g, b, static_cast<const cplx<T>*>(tab), mstride);
}
template <typename T, int NX> static size_t fused_smem(const Geom& g) {
  return RowCfg<T, NX>::SMEM + (size_t)RowCfg<T, NX>::L * 2 * ((g.Wx + 3) & ~3) * sizeof(cplx<T>);
}
template <typename T, int NX> static cudaError_t go_fwd_row_fused(const Geom& g, const Model& m, const void* vx, const void* vy,
                                                                  const void* w, const void* K, void* oA, void* oB,
                                                                  const void* tab, cudaStream_t s) {
  using C = RowCfg<T, NX>;
  return launch_pdl(k_fwd_row_fused<T, NX>, dim3((g.Ny / 2) / C::L), dim3(C::THREADS), fused_smem<T, NX>(g), s, g, m, (const T*)vx, (const T*)vy,
                    (const T*)w, (const T*)K, (cplx<T>*)oA, (cplx<T>*)oB, static_cast<const cplx<T>*>(tab));
}
template <typename T> cudaError_t launch_fwd_row_fused(const Geom& g, const Model& m, const void* vx, const void* vy, const void* w,
                                                       const void* K, void* oA, void* oB, const void* tab, cudaStream_t s) {
  switch (g.Nx) {       // pair kernels only (Nx <= 8192)
#define X(N) case N: return go_fwd_row_fused<T, N>(g, m, vx, vy, w, K, oA, oB, tab, s);
    TTSH_FOR_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
template <typename T> cudaError_t launch_inv_row(const Geom& g, const Batch& b, int nf, const void* tab, const void* tabR, const double* v0,
                                                 cudaStream_t s, int members, size_t mstride) {
  if (members < 1 || members > 65535) return cudaErrorInvalidValue;
  if (g.Nx == TTSH_REAL_ROW_NX) return go_inv_row_real<T, TTSH_REAL_ROW_NX>(g, b, nf, tab, tabR, v0, s, members, mstride);
  switch (g.Nx) {
#define X(N) case N: return go_inv_row<T, N>(g, b, nf, tab, v0, s, members, mstride);
    TTSH_FOR_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
template <typename T> cudaError_t launch_fwd_row(const Geom& g, const Batch& b, int nf, const void* tab, const void* tabR, cudaStream_t s,
                                                 int members, size_t mstride) {
  if (members < 1 || members > 65535) return cudaErrorInvalidValue;
  if (g.Nx == TTSH_REAL_ROW_NX) return go_fwd_row_real<T, TTSH_REAL_ROW_NX>(g, b, nf, tab, tabR, s, members, mstride);
  switch (g.Nx) {
#define X(N) case N: return go_fwd_row<T, N>(g, b, nf, tab, s, members, mstride);
    TTSH_FOR_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
template <typename T> cudaError_t prepare_rows(const Geom& g) {
  if (g.Nx == TTSH_REAL_ROW_NX) {
    using C = RealRowCfg<T, TTSH_REAL_ROW_NX>;
    cudaError_t e = set_smem(k_inv_row_real<T, TTSH_REAL_ROW_NX>, C::SMEM);
    if (e != cudaSuccess) return e;
    return set_smem(k_fwd_row_real<T, TTSH_REAL_ROW_NX>, C::SMEM);
  }
  switch (g.Nx) {
#define X(N) case N: { cudaError_t e = set_smem(k_inv_row<T, N>, RowCfg<T, N>::SMEM); if (e != cudaSuccess) return e; \
                       e = set_smem(k_fwd_row_fused<T, N>, fused_smem<T, N>(g)); if (e != cudaSuccess) return e; \
                       return set_smem(k_fwd_row<T, N>, RowCfg<T, N>::SMEM); }
    TTSH_FOR_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
#endif

#ifdef TTSH_BUILD_ROWSTEP
}  // namespace ttsh
#include "row_step.cuh"
#include "row_step_real.cuh"
namespace ttsh {
// Nx = 8192 (fp64: a packed row pair does not fit in shared memory; fp32: faster): one real row per half-length transform (row_step_real.cuh);
// K in the thread order of that kernel (launch_reperm_real), table = fill_stage_tables_real
template <typename T, int NX> constexpr bool row_step_real_enabled() { return NX == 8192 || (NX == 16384 && sizeof(T) == 4); }
__host__ __device__ constexpr int row_step_real_tabr_offset(int M) { return ((M == 4096 ? fft_wl_tw_elems_rt(M) : fft_tw_elems_rt(M) + 1) + 15) / 16 * 16; }
// Single systems and ensembles run the SAME instantiation (the member loop of the ensemble variant with one member), so that an
// ensemble member is bit-identical to the system stepped alone whatever the compiler does with the two variants.
template <typename T, int NX, bool ENS_> static cudaError_t prep_row_step_real(int* slots) {
  constexpr bool ENS = true;
  using C = RowStepRealCfg<T, NX>;
  static_assert(C::FITS, "row_step_real: line, stash, table and the K slot must fit in shared memory");
  cudaError_t e = set_smem(k_row_step_real<T, NX, ENS>, C::SMEM);
  if (e != cudaSuccess) return e;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  *slots = sms > 0 ? sms : 148;                                   // one CTA per SM
  return cudaSuccess;
}
template <typename T, int NX, bool ENS_>
static cudaError_t go_row_step_real(const Geom& g, const Model& m, const void* inW, const void* inVx, const void* inPsi, const void* K2,
                                    void* oA, void* oB, const void* tab, const double* v0, cudaStream_t s, int members, size_t mstride, int slots) {
  constexpr bool ENS = true;
  using C = RowStepRealCfg<T, NX>;
  if (slots <= 0) return cudaErrorInvalidConfiguration;
  const int rpm = g.Ny / 2;
  const long long nblk_ll = (long long)rpm * members;
  if (nblk_ll > 0x3fffffff) return cudaErrorInvalidValue;
  const int nblk = (int)nblk_ll;
  const int grid = nblk < slots ? nblk : slots;
  const cplx<T>* tabW = static_cast<const cplx<T>*>(tab);
  return launch_pdl(k_row_step_real<T, NX, ENS>, dim3(grid), dim3(C::THREADS), C::SMEM, s, g, m, (const cplx<T>*)inW, (const cplx<T>*)inVx,
                    (const cplx<T>*)inPsi, (const T*)K2, (cplx<T>*)oA, (cplx<T>*)oB, tabW, tabW + row_step_real_tabr_offset(C::M), v0, nblk, rpm, mstride);
}
// persistent grid: one CTA per resident slot (SMs x occupancy), looping over the row-pair blocks.  The opt-in to > 48 KB of
// dynamic shared memory and the occupancy are per DEVICE: prepare_row_step runs in ttsh_create on the handle's device and the
// slot counts live in the handle.
template <typename T, int NX, int LL, bool ENS, bool TAN = false>
static cudaError_t prep_row_step(int* slots) {
  using C = RowStepCfg<T, NX, LL, TAN>;
  *slots = 0;
  if constexpr (!C::FITS) return cudaSuccess;
  else {
    cudaError_t e = set_smem(k_row_step<T, NX, LL, ENS, TAN>, C::SMEM);
    if (e != cudaSuccess) return e;
    int dev = 0, sms = 0, occ = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_row_step<T, NX, LL, ENS, TAN>, C::THREADS, C::SMEM);
    if (e != cudaSuccess) return e;
    *slots = sms * (occ > 0 ? occ : 1);
    return cudaSuccess;
  }
}
template <typename T, int NX, int LL, bool ENS, bool TAN = false>
static cudaError_t go_row_step(const Geom& g, const Model& m, const void* inW, const void* inVx, const void* inPsi, const void* K,
                               void* oA, void* oB, const void* tab, const double* v0, cudaStream_t s, int members, size_t mstride, int slots,
                               const void* bw = nullptr, const void* bvx = nullptr, const void* bvy = nullptr) {
  using C = RowStepCfg<T, NX, LL, TAN>;
  if constexpr (!C::FITS) return cudaErrorInvalidConfiguration;
  else {
    if (slots <= 0) return cudaErrorInvalidConfiguration;
    const int rpm = g.Ny / 2;                                  // row pairs per member
    const long long nblk_ll = (long long)rpm * members / C::L;
    if (nblk_ll > 0x3fffffff) return cudaErrorInvalidValue;
    const int nblk = (int)nblk_ll;
    const int grid = nblk < slots ? nblk : slots;
    return launch_pdl(k_row_step<T, NX, LL, ENS, TAN>, dim3(grid), dim3(C::THREADS), C::SMEM, s, g, m, (const cplx<T>*)inW, (const cplx<T>*)inVx,
                      (const cplx<T>*)inPsi, (const T*)K, (cplx<T>*)oA, (cplx<T>*)oB, static_cast<const cplx<T>*>(tab), v0, nblk, rpm, mstride,
                      (const T*)bw, (const T*)bvx, (const T*)bvy);
  }
}
template <typename T> cudaError_t prepare_row_step(const Geom& g, int* slots, int* slots_ens, int* slots_tan) {
  *slots = *slots_ens = *slots_tan = 0;
  if constexpr (row_step_real_enabled<T, TTSH_REAL_ROW_NX>()) {
    if (g.Nx == TTSH_REAL_ROW_NX) {
      cudaError_t e = prep_row_step_real<T, TTSH_REAL_ROW_NX, false>(slots); if (e != cudaSuccess) return e;
      return prep_row_step_real<T, TTSH_REAL_ROW_NX, true>(slots_ens);
    }
  }
  switch (g.Nx) {
#define X(N) case N: { cudaError_t e = prep_row_step<T, N, row_step_ens_lines<N>(), true, true>(slots_tan); if (e != cudaSuccess) return e; \
                       if constexpr (row_step_real_enabled<T, N>()) { \
                         e = prep_row_step_real<T, N, false>(slots); if (e != cudaSuccess) return e; \
                         return prep_row_step_real<T, N, true>(slots_ens); \
                       } else { \
                         e = prep_row_step<T, N, 1, false>(slots); if (e != cudaSuccess) return e; \
                         return prep_row_step<T, N, row_step_ens_lines<N>(), true>(slots_ens); } }
    TTSH_FOR_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
template <typename T> cudaError_t launch_row_step(const Geom& g, const Model& m, const void* inW, const void* inVx, const void* inPsi,
                                                  const void* K, void* oA, void* oB, const void* tab, const double* v0, cudaStream_t s, int slots) {
  if constexpr (row_step_real_enabled<T, TTSH_REAL_ROW_NX>()) {
    if (g.Nx == TTSH_REAL_ROW_NX) return go_row_step_real<T, TTSH_REAL_ROW_NX, false>(g, m, inW, inVx, inPsi, K, oA, oB, tab, v0, s, 1, 0, slots);
  }
  switch (g.Nx) {
#define X(N) case N: if constexpr (row_step_real_enabled<T, N>()) return go_row_step_real<T, N, false>(g, m, inW, inVx, inPsi, K, oA, oB, tab, v0, s, 1, 0, slots); \
                     else return go_row_step<T, N, 1, false>(g, m, inW, inVx, inPsi, K, oA, oB, tab, v0, s, 1, 0, slots);
    TTSH_FOR_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
template <typename T> cudaError_t launch_row_step_ens(const Geom& g, const Model& m, const void* inW, const void* inVx, const void* inPsi,
                                                      const void* K, void* oA, void* oB, const void* tab, const double* v0, cudaStream_t s,
                                                      int members, size_t mstride, int slots) {
  if constexpr (row_step_real_enabled<T, TTSH_REAL_ROW_NX>()) {
    if (g.Nx == TTSH_REAL_ROW_NX) return go_row_step_real<T, TTSH_REAL_ROW_NX, true>(g, m, inW, inVx, inPsi, K, oA, oB, tab, v0, s, members, mstride, slots);
  }
  switch (g.Nx) {
#define X(N) case N: if constexpr (row_step_real_enabled<T, N>()) return go_row_step_real<T, N, true>(g, m, inW, inVx, inPsi, K, oA, oB, tab, v0, s, members, mstride, slots); \
                     else return go_row_step<T, N, row_step_ens_lines<N>(), true>(g, m, inW, inVx, inPsi, K, oA, oB, tab, v0, s, members, mstride, slots);
    TTSH_FOR_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
// tangent-linear variant: members = tangent vectors (in / out / v0 at mstride), K and the base fields bw, bvx, bvy shared
template <typename T> cudaError_t launch_row_step_tan(const Geom& g, const Model& m, const void* inW, const void* inVx, const void* inPsi,
                                                      const void* K, void* oA, void* oB, const void* tab, const double* v0, cudaStream_t s,
                                                      int members, size_t mstride, int slots, const void* bw, const void* bvx, const void* bvy) {
  switch (g.Nx) {
#define X(N) case N: return go_row_step<T, N, row_step_ens_lines<N>(), true, true>(g, m, inW, inVx, inPsi, K, oA, oB, tab, v0, s, members, mstride, slots, bw, bvx, bvy);
    TTSH_FOR_SIZES(X)
#undef X
  }
  return cudaErrorInvalidValue;
}
template <typename T> bool row_step_is_real(const Geom& g) {
  return row_step_supported<T>(g) && (g.Nx == 8192 || g.Nx == TTSH_REAL_ROW_NX);
}
template <typename T> int row_step_real_tabr(const Geom& g) { return row_step_real_tabr_offset(g.Nx / 2); }
template <typename T> bool row_step_supported(const Geom& g) {
  if (4 * (g.Wx - 1) != g.Nx) return false;          // 1/2 rule only
  if (g.Nx == TTSH_REAL_ROW_NX) return row_step_real_enabled<T, TTSH_REAL_ROW_NX>();
  switch (g.Nx) {
#define X(N) case N: return RowStepCfg<T, N>::FITS || row_step_real_enabled<T, N>();
    TTSH_FOR_SIZES(X)
#undef X
  }
  return false;
}
#endif

}  // namespace ttsh
