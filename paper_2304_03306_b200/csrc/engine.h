// engine.h — host-side launchers of the CUDA kernels, one explicit instantiation per scalar type.
#pragma once
#include <cuda_runtime.h>
#include "ttsh_common.cuh"

namespace ttsh {

// launch with programmatic dependent launch allowed (ttsh_common.cuh: pdl_wait / pdl_trigger); captured into CUDA graphs as a
// programmatic dependency edge
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = TTSH_PDL;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// FFT passes (fft_passes.cuh).  nfields <= 5 fields per launch (grid.y).  Return cudaErrorInvalidValue for an
// unsupported transform length.
// Ensembles (ttsh_ensemble_step): `members` independent systems whose workspaces lie `mstride` bytes apart are advanced by
// ONE launch of each hot kernel: member b uses every pointer argument (field sources / destinations, K, v0) + b * mstride;
// the twiddle tables are member 0's.
template <typename T> cudaError_t launch_inv_col(const Geom& g, const Batch& b, int nfields, const void* tabY, const void* tabS, const double* v0, cudaStream_t s,
                                                 int members = 1, size_t mstride = 0);
template <typename T> cudaError_t launch_fwd_col(const Geom& g, const Batch& b, int nfields, const void* tabY, const void* tabS, cudaStream_t s,
                                                 int members = 1, size_t mstride = 0);
// tabR: W_Nx^j, j < Nx/32, used by the real-row kernels of Nx = 16384 (fft_rows_real.cuh); ignored on the other grids
template <typename T> cudaError_t launch_inv_row(const Geom& g, const Batch& b, int nfields, const void* tabX, const void* tabR, const double* v0,
                                                 cudaStream_t s, int members = 1, size_t mstride = 0);
template <typename T> cudaError_t launch_fwd_row(const Geom& g, const Batch& b, int nfields, const void* tabX, const void* tabR, cudaStream_t s,
                                                 int members = 1, size_t mstride = 0);
// fused real-space + forward row pass (conservative form): reads v_x, v_y, w, K; writes A~ = i kx Gy~ + S'~ and B~ = Gx~
template <typename T> cudaError_t launch_fwd_row_fused(const Geom& g, const Model& m, const void* vx, const void* vy, const void* w,
                                                       const void* K, void* oA, void* oB, const void* tabX, cudaStream_t s);
// a5 for the two-spectrum form: rhs^ = A^ - i ky B^ (column mx = 0: A^ = S'^ + i Gy^ separated by Hermitian symmetry)
template <typename T> cudaError_t launch_spectral_p2(const Geom& g, const Model& m, const void* A, const void* B, void* w, void* psi,
                                                     double* v0, cudaStream_t s, int members = 1, size_t mstride = 0);
// the whole row half of a step in one kernel (row_step.cuh): reads the inverse intermediates of w, v_x (= i k_y psi^ with the mean
// flow) and psi, and K; writes A~ and B~.  Supported for the 1/2 rule when one packed row pair fits in shared memory.
template <typename T> cudaError_t launch_row_step(const Geom& g, const Model& m, const void* inW, const void* inVx, const void* inPsi,
                                                  const void* K, void* oA, void* oB, const void* tabX, const double* v0, cudaStream_t s, int slots);
template <typename T> bool row_step_supported(const Geom& g);
// ... and it is the real-row variant (row_step_real.cuh: Nx = 8192): K in its thread order (launch_reperm_real); table = the warp-local
// table of length Nx/2 followed, at element row_step_real_tabr(g), by W_Nx^j, j < Nx/32
template <typename T> bool row_step_is_real(const Geom& g);
template <typename T> int row_step_real_tabr(const Geom& g);
// per-device set-up of k_row_step (shared-memory opt-in, resident CTAs): call on the handle's device; slots = CTAs of the
// persistent grid of the single-system / ensemble variant (0: not supported for this grid)
template <typename T> cudaError_t prepare_row_step(const Geom& g, int* slots, int* slots_ens, int* slots_tan);
// tangent-linear variant of the row-step kernel (row_step.cuh, TAN): members = tangent vectors whose intermediates / outputs / mean
// flows lie mstride bytes apart; K and the base fields bw, bvx, bvy (internal real fields, layout perm_index) are shared.  tabX: the
// plain per-stage tables (this variant never runs the warp-local plan)
template <typename T> cudaError_t launch_row_step_tan(const Geom& g, const Model& m, const void* inW, const void* inVx, const void* inPsi,
                                                      const void* K, void* oA, void* oB, const void* tabX, const double* v0, cudaStream_t s,
                                                      int members, size_t mstride, int slots, const void* bw, const void* bvx, const void* bvy);
// the same kernel over an ensemble: several row pairs per CTA on small grids (a line of Nx = 64 has 4 threads), row pairs
// of all members in one persistent grid
template <typename T> cudaError_t launch_row_step_ens(const Geom& g, const Model& m, const void* inW, const void* inVx, const void* inPsi,
                                                      const void* K, void* oA, void* oB, const void* tabX, const double* v0, cudaStream_t s,
                                                      int members, size_t mstride, int slots);
// set the dynamic shared-memory attribute of the pass kernels for this grid (no launch)
template <typename T> cudaError_t prepare_rows(const Geom& g);
template <typename T> cudaError_t prepare_cols(const Geom& g);
// the column half of the time loop in one kernel (col_step.cuh; Ny <= 1024, 1/2 rule): forward column pass of A~, B~, lines 3-13 of
// Algorithm 1 on the state (w, psi, v0), inverse column pass of w^, psi^, i k_y psi^ for the next row kernel
template <typename T> bool col_step_supported(const Geom& g);
template <typename T> cudaError_t launch_col_step(const Geom& g, const Model& m, const void* srcA, const void* srcB, void* w, void* psi, double* v0,
                                                  void* dstW, void* dstPsi, void* dstVx, const void* tabY, const void* tabS, cudaStream_t s,
                                                  int members = 1, size_t mstride = 0);

// element-wise kernels and reductions (pointwise.cuh)
template <typename T> cudaError_t launch_realspace(const Geom& g, const Model& m, const void* vx, const void* vy, const void* K,
                                                   void* w_s, void* gx_fx, void* gy_fy, cudaStream_t s);
template <typename T> cudaError_t launch_realspace_cons(const Geom& g, const Model& m, const void* vx, const void* vy, const void* K,
                                                        void* w_s, void* gx_out, void* gy_out, cudaStream_t s);
template <typename T> cudaError_t launch_spectral(const Geom& g, const Model& m, const void* Fx, const void* Fy, const void* S,
                                                  void* w, void* psi, double* v0, cudaStream_t s, int members = 1, size_t mstride = 0);
template <typename T> cudaError_t launch_spectral_init(const Geom& g, const void* Vx, const void* Vy, void* w, void* psi, double* v0, cudaStream_t s);
template <typename T> cudaError_t launch_psi_from_w(const Geom& g, const void* w, void* psi, cudaStream_t s);
// checkpoint layout: the tile-major pruned spectrum <-> natural order complex[Hy][Wx] (independent of the tile width CW)
template <typename T> cudaError_t launch_state_pack(const Geom& g, const void* w, void* nat, cudaStream_t s);
template <typename T> cudaError_t launch_state_unpack(const Geom& g, const void* nat, void* w, cudaStream_t s);
template <typename T> cudaError_t launch_mask_to_real(size_t n, const unsigned char* mask, void* out, cudaStream_t s);
template <typename T> cudaError_t launch_square(size_t n, const void* in, void* out, cudaStream_t s);
template <typename T> cudaError_t launch_fill(size_t n, void* out, double val, cudaStream_t s);
// natural <-> permuted row layout of an internal real field (to_perm = 1: natural -> permuted)
template <typename T> cudaError_t launch_permute(int Nx, size_t n, const void* in, void* out, int to_perm, cudaStream_t s);
// permuted internal row layout (perm_index) -> thread-order layout of the warp-local plan (perm_index_wl)
template <typename T> cudaError_t launch_reperm_wl(int Nx, size_t n, const void* in, void* out, cudaStream_t s);
// permuted internal row layout -> thread order of row_step_real.cuh: (K(y, 2n), K(y, 2n+1)), n = wl_j(t) + (Nx/32) k, at y Nx + (k Nx/32 + t) 2
template <typename T> cudaError_t launch_reperm_real(int Nx, size_t n, const void* in, void* out, cudaStream_t s);
constexpr int DIAG_BLOCKS = 592;   // 4 x 148 SMs
template <typename T> cudaError_t launch_diag(const Geom& g, double dx, double cx, double cy, const void* vx, const void* vy,
                                              const void* w, double* partial, double* out, cudaStream_t s);

// Psi_2: per side (|w|, w, linear index) of the argmax of |w| within `radius` of (cx, cy); out[6]
template <typename T> cudaError_t launch_region_argmax(const Geom& g, double dx, double cxl, double cyl, double cxr, double cyr, double radius,
                                                       const void* w, double* partial, double* out, cudaStream_t s);

// streaming temporal PSD, Eq. (5): acc[nf][n] += w exp(-i Omega t) with host-computed phases cs = cos(Omega t),
// sn = -sin(Omega t) (HOST arrays);  out[m] = sum_x |acc[m][x]|^2 through partial[nf][psd_blocks()]
template <typename T> cudaError_t launch_psd_accumulate(size_t n, int nf, const double* cs, const double* sn, const void* w, void* acc, cudaStream_t s);
template <typename T> cudaError_t launch_psd_power(size_t n, int nf, const void* acc, double* partial, double* out, cudaStream_t s);
int psd_blocks();

// tangent-linear step and Gram-Schmidt on tangent vectors (pointwise.cuh)
// members: tangent vectors whose (dvx, dvy, dw) lie mstride bytes apart; the base fields and K are shared
template <typename T> cudaError_t launch_realspace_tangent(const Geom& g, const Model& m, const void* vx, const void* vy, const void* w,
                                                           const void* K, void* dvx, void* dvy, void* dw, cudaStream_t s,
                                                           int members = 1, size_t mstride = 0);
// batched over count vectors b_j / y_j at a uniform byte stride (one launch per Gram-Schmidt row)
template <typename T> cudaError_t launch_spec_dot(const Geom& g, const void* a, const void* b, const double* a0, const double* b0,
                                                  int count, size_t bstride, int norm_slot, double* partial, double* rdiag,
                                                  double* coef, cudaStream_t s);
template <typename T> cudaError_t launch_spec_scale_axpy(const Geom& g, const double* coef, const void* x, void* y, const double* x0,
                                                         double* y0, int count, size_t ystride, cudaStream_t s);

// blocked QR (CholeskyQR2) of tangent vectors at a uniform byte stride: Gram matrix G[nvec][nvec] (device; partial: nvec^2 *
// DIAG_BLOCKS doubles) and the in-place product A <- A S with an upper-triangular S (device), which also refreshes psi^ = w^/k^2
template <typename T> cudaError_t launch_gram(const Geom& g, const void* v, const double* v0, size_t vstride, int nvec, double* partial, double* G,
                                              cudaStream_t s);
cudaError_t launch_chol_inv(int nvec, const double* G, double* S, double* logr, int* flag, cudaStream_t s);
template <typename T> cudaError_t launch_tri_apply(const Geom& g, int nvec, const double* S, void* v, void* psi, double* v0, size_t vstride, cudaStream_t s);

}  // namespace ttsh
