// element-wise kernels and reductions, both scalar types
#include "engine.h"
#include "pointwise.cuh"

namespace ttsh {

static inline int blocks_for(size_t n, int threads, int cap) {
  size_t b = (n + threads - 1) / threads;
  return (int)(b < (size_t)cap ? (b ? b : 1) : cap);
}
constexpr int GRID_CAP = 148 * 16;

template <typename T> cudaError_t launch_realspace(const Geom& g, const Model& m, const void* vx, const void* vy, const void* K,
                                                   void* w_s, void* gx_fx, void* gy_fy, cudaStream_t s) {
  const size_t nvec = (size_t)g.Nx * g.Ny / Vec<T>::n;
  k_realspace<T><<<blocks_for(nvec, 256, GRID_CAP), 256, 0, s>>>(nvec, m, (const T*)vx, (const T*)vy, (const T*)K,
                                                                  (T*)w_s, (T*)gx_fx, (T*)gy_fy);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_realspace_cons(const Geom& g, const Model& m, const void* vx, const void* vy, const void* K,
                                                        void* w_s, void* gx_out, void* gy_out, cudaStream_t s) {
  const size_t nvec = (size_t)g.Nx * g.Ny / Vec<T>::n;
  k_realspace_cons<T><<<blocks_for(nvec, 256, GRID_CAP), 256, 0, s>>>(nvec, m, (const T*)vx, (const T*)vy, (const T*)K,
                                                                       (T*)w_s, (T*)gx_out, (T*)gy_out);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_spectral(const Geom& g, const Model& m, const void* Fx, const void* Fy, const void* S,
                                                  void* w, void* psi, double* v0, cudaStream_t s, int members, size_t mstride) {
  if (members < 1 || members > 65535) return cudaErrorInvalidValue;
  const dim3 grid((unsigned)(((size_t)g.NT * g.Hy * g.CW + 255) / 256), (unsigned)members);
  return launch_pdl(k_spectral<T>, grid, dim3(256), 0, s, g, m, (const cplx<T>*)Fx, (const cplx<T>*)Fy, (const cplx<T>*)S, (cplx<T>*)w, (cplx<T>*)psi, v0, mstride);
}
template <typename T> cudaError_t launch_spectral_p2(const Geom& g, const Model& m, const void* A, const void* B, void* w, void* psi,
                                                     double* v0, cudaStream_t s, int members, size_t mstride) {
  if (members > 65535) return cudaErrorInvalidValue;
  const dim3 grid((unsigned)(((size_t)g.NT * g.Hy * g.CW + 255) / 256), (unsigned)members);
  return launch_pdl(k_spectral_p2<T>, grid, dim3(256), 0, s, g, m, (const cplx<T>*)A, (const cplx<T>*)B, (cplx<T>*)w, (cplx<T>*)psi, v0, mstride);
}
template <typename T> cudaError_t launch_spectral_init(const Geom& g, const void* Vx, const void* Vy, void* w, void* psi, double* v0, cudaStream_t s) {
  const unsigned grid = (unsigned)(((size_t)g.NT * g.Hy * g.CW + 255) / 256);
  k_spectral_init<T><<<grid, 256, 0, s>>>(g, (const cplx<T>*)Vx, (const cplx<T>*)Vy, (cplx<T>*)w, (cplx<T>*)psi, v0);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_psi_from_w(const Geom& g, const void* w, void* psi, cudaStream_t s) {
  const unsigned grid = (unsigned)(((size_t)g.NT * g.Hy * g.CW + 255) / 256);
  k_psi_from_w<T><<<grid, 256, 0, s>>>(g, (const cplx<T>*)w, (cplx<T>*)psi);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_state_pack(const Geom& g, const void* w, void* nat, cudaStream_t s) {
  const unsigned grid = (unsigned)(((size_t)g.Hy * g.Wx + 255) / 256);
  k_state_pack<T><<<grid, 256, 0, s>>>(g, (const cplx<T>*)w, (cplx<T>*)nat);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_state_unpack(const Geom& g, const void* nat, void* w, cudaStream_t s) {
  const unsigned grid = (unsigned)(((size_t)g.NT * g.Hy * g.CW + 255) / 256);
  k_state_unpack<T><<<grid, 256, 0, s>>>(g, (const cplx<T>*)nat, (cplx<T>*)w);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_mask_to_real(size_t n, const unsigned char* mask, void* out, cudaStream_t s) {
  k_mask_to_real<T><<<blocks_for(n, 256, GRID_CAP), 256, 0, s>>>(n, mask, (T*)out);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_square(size_t n, const void* in, void* out, cudaStream_t s) {
  k_square<T><<<blocks_for(n, 256, GRID_CAP), 256, 0, s>>>(n, (const T*)in, (T*)out);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_permute(int Nx, size_t n, const void* in, void* out, int to_perm, cudaStream_t s) {
  k_permute_rows<T><<<blocks_for(n, 256, GRID_CAP), 256, 0, s>>>(Nx, n, (const T*)in, (T*)out, to_perm);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_reperm_real(int Nx, size_t n, const void* in, void* out, cudaStream_t s) {
  if (Nx < 512) return cudaErrorInvalidValue;
  k_reperm_real<T><<<blocks_for(n, 256, GRID_CAP), 256, 0, s>>>(Nx, n, (const T*)in, (T*)out, Nx == 8192 ? 1 : 0, Nx == 16384 ? 1 : 0);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_reperm_wl(int Nx, size_t n, const void* in, void* out, cudaStream_t s) {
  k_reperm_wl<T><<<blocks_for(n, 256, GRID_CAP), 256, 0, s>>>(Nx, n, (const T*)in, (T*)out);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_fill(size_t n, void* out, double val, cudaStream_t s) {
  k_fill<T><<<blocks_for(n, 256, GRID_CAP), 256, 0, s>>>(n, (T*)out, (T)val);
  return cudaGetLastError();
}
template <typename T> cudaError_t launch_diag(const Geom& g, double dx, double cx, double cy, const void* vx, const void* vy,
                                              const void* w, double* partial, double* out, cudaStream_t s) {
  k_diag_partial<T><<<DIAG_BLOCKS, 256, 0, s>>>(g.Nx, g.Ny, dx, cx, cy, (const T*)vx, (const T*)vy, (const T*)w, partial);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_diag_final<<<1, 256, 0, s>>>(DIAG_BLOCKS, partial, out);
  return cudaGetLastError();
}

template <typename T> cudaError_t launch_region_argmax(const Geom& g, double dx, double cxl, double cyl, double cxr, double cyr, double radius,
                                                       const void* w, double* partial, double* out, cudaStream_t s) {
  k_region_argmax_partial<T><<<DIAG_BLOCKS, 256, 0, s>>>(g.Nx, g.Ny, dx, cxl, cyl, cxr, cyr, radius, (const T*)w, partial);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_region_argmax_final<<<1, 256, 0, s>>>(DIAG_BLOCKS, partial, out);
  return cudaGetLastError();
}

template <typename T> cudaError_t launch_psd_accumulate(size_t n, int nf, const double* cs, const double* sn, const void* w, void* acc, cudaStream_t s) {
  for (int m0 = 0; m0 < nf; m0 += PSD_CHUNK) {
    const int cnt = nf - m0 < PSD_CHUNK ? nf - m0 : PSD_CHUNK;
    PsdPhases ph;
    for (int m = 0; m < PSD_CHUNK; ++m) { ph.c[m] = m < cnt ? cs[m0 + m] : 0.0; ph.s[m] = m < cnt ? sn[m0 + m] : 0.0; }
    k_psd_accumulate<T><<<blocks_for(n, 256, GRID_CAP), 256, 0, s>>>(n, cnt, ph, (const T*)w, (cplx<T>*)acc + (size_t)m0 * n);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}
template <typename T> cudaError_t launch_psd_power(size_t n, int nf, const void* acc, double* partial, double* out, cudaStream_t s) {
  k_psd_power_partial<T><<<dim3(PSD_BLOCKS, nf), 256, 0, s>>>(n, (const cplx<T>*)acc, partial);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_psd_power_final<<<nf, 32, 0, s>>>(PSD_BLOCKS, partial, out);
  return cudaGetLastError();
}
int psd_blocks() { return PSD_BLOCKS; }

template <typename T> cudaError_t launch_realspace_tangent(const Geom& g, const Model& m, const void* vx, const void* vy, const void* w,
                                                           const void* K, void* dvx, void* dvy, void* dw, cudaStream_t s,
                                                           int members, size_t mstride) {
  if (members < 1 || members > 65535) return cudaErrorInvalidValue;
  const size_t nvec = (size_t)g.Nx * g.Ny / Vec<T>::n;
  const dim3 grid((unsigned)blocks_for(nvec, 256, GRID_CAP), (unsigned)members);
  return launch_pdl(k_realspace_tangent<T>, grid, dim3(256), 0, s, nvec, m, (const T*)vx, (const T*)vy, (const T*)w, (const T*)K, (T*)dvx, (T*)dvy, (T*)dw, mstride);
}
// count = 1, norm_slot >= 0:  rdiag[norm_slot] <- |a|, coef[0] <- 1/|a|   (b = a)
// norm_slot < 0:              coef[j] <- <a, b_j>, b_j = b + j * bstride bytes, j < count;  partial: DIAG_BLOCKS * count doubles
template <typename T> cudaError_t launch_spec_dot(const Geom& g, const void* a, const void* b, const double* a0, const double* b0,
                                                  int count, size_t bstride, int norm_slot, double* partial, double* rdiag,
                                                  double* coef, cudaStream_t s) {
  cudaError_t e = launch_pdl(k_spec_dot_partial<T>, dim3(DIAG_BLOCKS, count), dim3(256), 0, s, g, (const cplx<T>*)a, (const cplx<T>*)b, partial, bstride);
  if (e != cudaSuccess) return e;
  return launch_pdl(k_spec_dot_final, dim3(count), dim3(32), 0, s, (int)DIAG_BLOCKS, (const double*)partial, a0, b0, bstride, norm_slot, rdiag, coef);
}
// y_j <- coef[j] y_j (x == NULL) or y_j <- y_j - coef[j] x, j < count, on the spectrum and the mean flow
template <typename T> cudaError_t launch_spec_scale_axpy(const Geom& g, const double* coef, const void* x, void* y, const double* x0,
                                                         double* y0, int count, size_t ystride, cudaStream_t s) {
  const size_t n = (size_t)g.NT * g.Hy * g.CW;
  return launch_pdl(k_spec_scale_axpy<T>, dim3(blocks_for(n, 256, GRID_CAP), count), dim3(256), 0, s, n, coef, (const cplx<T>*)x, (cplx<T>*)y, x0, y0, ystride);
}

// Gram matrix of nvec tangent vectors (spectra v + j vstride bytes, mean flows v0 + j vstride bytes) into G[nvec][nvec] (device);
// partial: nvec * nvec * DIAG_BLOCKS doubles
template <typename T> cudaError_t launch_gram(const Geom& g, const void* v, const double* v0, size_t vstride, int nvec, double* partial, double* G,
                                              cudaStream_t s) {
  const int tiles = (nvec + GRAM_TILE - 1) / GRAM_TILE;
  const size_t n = (size_t)g.NT * g.Hy * g.CW;
  const int nb = blocks_for(n, 256, DIAG_BLOCKS);      // small spectra: no more blocks than there is work (nvec * tiles of them each)
  cudaError_t e = launch_pdl(k_gram_partial<T>, dim3(nb, nvec, tiles), dim3(256), 0, s, g, (const cplx<T>*)v, vstride, nvec, partial);
  if (e != cudaSuccess) return e;
  return launch_pdl(k_gram_final, dim3(nvec, nvec), dim3(32), 0, s, nb, nvec, (const double*)partial, v0, vstride, G);
}
// Cholesky factor of G and its inverse on the device (nvec <= 64); logr[i] += log R_ii; *flag set on a breakdown
cudaError_t launch_chol_inv(int nvec, const double* G, double* S, double* logr, int* flag, cudaStream_t s) {
  if (nvec < 1 || nvec > 64) return cudaErrorInvalidValue;
  return launch_pdl(k_chol_inv, dim3(1), dim3(64), 0, s, nvec, G, S, logr, flag);
}
// A <- A S (S upper triangular, device, row-major), psi^ = w^/k^2 and the mean flows alongside
template <typename T> cudaError_t launch_tri_apply(const Geom& g, int nvec, const double* S, void* v, void* psi, double* v0, size_t vstride, cudaStream_t s) {
  const size_t n = (size_t)g.NT * g.Hy * g.CW;
  return launch_pdl(k_tri_apply<T>, dim3(blocks_for(n, 256, GRID_CAP)), dim3(256), 0, s, g, nvec, S, (cplx<T>*)v, (cplx<T>*)psi, v0, vstride);
}

#define INST(T) \
  template cudaError_t launch_gram<T>(const Geom&, const void*, const double*, size_t, int, double*, double*, cudaStream_t); \
  template cudaError_t launch_tri_apply<T>(const Geom&, int, const double*, void*, void*, double*, size_t, cudaStream_t); \
  template cudaError_t launch_realspace_tangent<T>(const Geom&, const Model&, const void*, const void*, const void*, const void*, void*, void*, void*, cudaStream_t, int, size_t); \
  template cudaError_t launch_spec_dot<T>(const Geom&, const void*, const void*, const double*, const double*, int, size_t, int, double*, double*, double*, cudaStream_t); \
  template cudaError_t launch_spec_scale_axpy<T>(const Geom&, const double*, const void*, void*, const double*, double*, int, size_t, cudaStream_t); \
  template cudaError_t launch_psd_accumulate<T>(size_t, int, const double*, const double*, const void*, void*, cudaStream_t); \
  template cudaError_t launch_psd_power<T>(size_t, int, const void*, double*, double*, cudaStream_t); \
  template cudaError_t launch_region_argmax<T>(const Geom&, double, double, double, double, double, double, const void*, double*, double*, cudaStream_t); \
  template cudaError_t launch_realspace<T>(const Geom&, const Model&, const void*, const void*, const void*, void*, void*, void*, cudaStream_t); \
  template cudaError_t launch_realspace_cons<T>(const Geom&, const Model&, const void*, const void*, const void*, void*, void*, void*, cudaStream_t); \
  template cudaError_t launch_spectral<T>(const Geom&, const Model&, const void*, const void*, const void*, void*, void*, double*, cudaStream_t, int, size_t); \
  template cudaError_t launch_spectral_init<T>(const Geom&, const void*, const void*, void*, void*, double*, cudaStream_t); \
  template cudaError_t launch_psi_from_w<T>(const Geom&, const void*, void*, cudaStream_t); \
  template cudaError_t launch_state_pack<T>(const Geom&, const void*, void*, cudaStream_t); \
  template cudaError_t launch_state_unpack<T>(const Geom&, const void*, void*, cudaStream_t); \
  template cudaError_t launch_spectral_p2<T>(const Geom&, const Model&, const void*, const void*, void*, void*, double*, cudaStream_t, int, size_t); \
  template cudaError_t launch_mask_to_real<T>(size_t, const unsigned char*, void*, cudaStream_t); \
  template cudaError_t launch_square<T>(size_t, const void*, void*, cudaStream_t); \
  template cudaError_t launch_fill<T>(size_t, void*, double, cudaStream_t); \
  template cudaError_t launch_permute<T>(int, size_t, const void*, void*, int, cudaStream_t); \
  template cudaError_t launch_reperm_wl<T>(int, size_t, const void*, void*, cudaStream_t); \
  template cudaError_t launch_reperm_real<T>(int, size_t, const void*, void*, cudaStream_t); \
  template cudaError_t launch_diag<T>(const Geom&, double, double, double, const void*, const void*, const void*, double*, double*, cudaStream_t);
INST(double)
INST(float)

}  // namespace ttsh
