// pointwise.cuh — element-wise kernels of Algorithm 1 and the diagnostics reduction.
//   k_realspace      lines 1-2: rhs1 = -beta |v|^2 v - gamma_v K v ;  rhs2 = -lambda0 v.grad(w) - gamma_w K w
//   k_spectral       lines 3-12: curl + sum, integrating-factor Euler, k = 0 / cutoff / Hermitian cases
//   k_spectral_init  state from a velocity field (ttsh_set_velocity)
//   k_diag_*         warp-shuffle reductions for E, Z, Psi (Eq. 11), polar order
// "any if statement should be purged": the k = 0 / cutoff cases are predicated selects on an
// integer predicate; the only divergent branch is the mx = 0 column of the Hermitian symmetrisation.
#pragma once
#include "ttsh_common.cuh"
#include "spectral_point.cuh"

namespace ttsh {

// ---------------------------------------------------------------------------------------
// a3: fused real-space kernel.  In place: (w, gx, gy) -> (rhs2, rhs1x, rhs1y); v and K are read-only.
// 16-byte vector accesses; Nx*Ny is a multiple of 4.
// ---------------------------------------------------------------------------------------
template <typename T> struct Vec;   // 16-byte vector of T
template <> struct Vec<double> { using type = double2; static constexpr int n = 2; };
template <> struct Vec<float> { using type = float4; static constexpr int n = 4; };

template <typename T>
__global__ void __launch_bounds__(256)
k_realspace(size_t nvec, Model m, const T* __restrict__ vx, const T* __restrict__ vy, const T* __restrict__ K,
            T* __restrict__ w_s, T* __restrict__ gx_fx, T* __restrict__ gy_fy) {
  using V = typename Vec<T>::type;
  constexpr int n = Vec<T>::n;
  const T beta = (T)m.beta, gv = (T)m.gamma_v, gw = (T)m.gamma_w, lam = (T)m.lambda0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    V a = reinterpret_cast<const V*>(vx)[i], b = reinterpret_cast<const V*>(vy)[i];
    V k = reinterpret_cast<const V*>(K)[i];
    V w = reinterpret_cast<V*>(w_s)[i], gx = reinterpret_cast<V*>(gx_fx)[i], gy = reinterpret_cast<V*>(gy_fy)[i];
    T* pa = reinterpret_cast<T*>(&a); T* pb = reinterpret_cast<T*>(&b); T* pk = reinterpret_cast<T*>(&k);
    T* pw = reinterpret_cast<T*>(&w); T* pgx = reinterpret_cast<T*>(&gx); T* pgy = reinterpret_cast<T*>(&gy);
#pragma unroll
    for (int e = 0; e < n; ++e) {
      const T u = pa[e], v = pb[e], kk = pk[e];
      const T c = -beta * (u * u + v * v) - gv * kk;                 // rhs1 = c * v           (line 1)
      const T s = -lam * (u * pgx[e] + v * pgy[e]) - gw * kk * pw[e];  // rhs2                   (line 2)
      pgx[e] = c * u;
      pgy[e] = c * v;
      pw[e] = s;
    }
    reinterpret_cast<V*>(w_s)[i] = w;
    reinterpret_cast<V*>(gx_fx)[i] = gx;
    reinterpret_cast<V*>(gy_fy)[i] = gy;
  }
}

// conservative form of the advection term (include/ttsh.h, ttsh_advection_form): with div v = 0,
//   -lambda0 v.grad(w) = -lambda0 (d_x (v_x w) + d_y (v_y w)), so the spectral curl+sum of line 3 absorbs it:
//   rhs^ = i kx (rhs1_y - lambda0 v_x w)^ - i ky (rhs1_x + lambda0 v_y w)^ + (-gamma_w K w)^.
// Reads v, w, K (4 fields), writes 3: w -> -gamma_w K w in place, gx_out, gy_out.
template <typename T>
__global__ void __launch_bounds__(256)
k_realspace_cons(size_t nvec, Model m, const T* __restrict__ vx, const T* __restrict__ vy, const T* __restrict__ K,
                 T* __restrict__ w_s, T* __restrict__ gx_out, T* __restrict__ gy_out) {
  using V = typename Vec<T>::type;
  constexpr int n = Vec<T>::n;
  const T beta = (T)m.beta, gv = (T)m.gamma_v, gw = (T)m.gamma_w, lam = (T)m.lambda0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    V a = reinterpret_cast<const V*>(vx)[i], b = reinterpret_cast<const V*>(vy)[i];
    V k = reinterpret_cast<const V*>(K)[i];
    V w = reinterpret_cast<V*>(w_s)[i], ox, oy;
    T* pa = reinterpret_cast<T*>(&a); T* pb = reinterpret_cast<T*>(&b); T* pk = reinterpret_cast<T*>(&k);
    T* pw = reinterpret_cast<T*>(&w); T* pox = reinterpret_cast<T*>(&ox); T* poy = reinterpret_cast<T*>(&oy);
#pragma unroll
    for (int e = 0; e < n; ++e) {
      const T u = pa[e], v = pb[e], kk = pk[e], ww = pw[e];
      const T c = -beta * (u * u + v * v) - gv * kk;      // rhs1 = c * v   (line 1)
      pox[e] = c * u + lam * (v * ww);                    // rhs1_x + lambda0 v_y w
      poy[e] = c * v - lam * (u * ww);                    // rhs1_y - lambda0 v_x w
      pw[e] = -gw * kk * ww;                              // damping part of rhs2   (line 2)
    }
    reinterpret_cast<V*>(w_s)[i] = w;
    reinterpret_cast<V*>(gx_out)[i] = ox;
    reinterpret_cast<V*>(gy_out)[i] = oy;
  }
}

// ---------------------------------------------------------------------------------------
// a5: fused spectral kernel on the tile-major pruned spectrum (spec_index).
//   w^_naive = exp(sigma dt) (w^ + dt (i kx F^y - i ky F^x + S^))                       (lines 3-4)
//   k = 0:   w^ = 0,  v^(0) <- exp(-alpha dt) (v^(0) + dt F^(0))                         (lines 6-8, Eq. C1)
//   cut:     w^ = 0                                                                       (lines 9-11)
//   else:    w^ = (w^_naive(k) + conj w^_naive(-k)) / 2 — the identity off the mx = 0 column in half-spectrum
//            storage; on that column the thread of (0, my > 0) computes both +-my and writes both   (line 12, R6)
// In place on w^ (every element is read and written by exactly one thread).
// ---------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ cplx<T> naive_update(const Geom& g, const Model& m, int mx, int my, size_t idx,
                                                const cplx<T>* __restrict__ Fx, const cplx<T>* __restrict__ Fy,
                                                const cplx<T>* __restrict__ S, const cplx<T>* w) {
  const T kx = (T)(g.dkx * mx), ky = (T)(g.dky * my);
  const T k2 = kx * kx + ky * ky;
  const T sigma = -(T)m.alpha - (T)m.Gamma0 * k2 - (T)m.Gamma2 * k2 * k2;
  const T dt = (T)m.dt;
  const cplx<T> r = kx * mul_i(Fy[idx]) - ky * mul_i(Fx[idx]) + S[idx];      // line 3
  const T e = sizeof(T) == 8 ? (T)exp((double)(sigma * dt)) : (T)expf((float)(sigma * dt));
  return e * (w[idx] + dt * r);                                               // line 4
}


template <typename T>
__global__ void __launch_bounds__(256)
k_spectral(Geom g, Model m, const cplx<T>* __restrict__ Fx_, const cplx<T>* __restrict__ Fy_,
           const cplx<T>* __restrict__ S_, cplx<T>* w_, cplx<T>* __restrict__ psi_, double* v0_, size_t mstride) {
  pdl_wait();
  // threads enumerate the tile-major array in memory order: idx = (t Hy + q) CW + c
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)g.NT * g.Hy * g.CW) return;
  const size_t moff = (size_t)blockIdx.y * mstride;      // member (tangent vectors at a uniform byte stride); 0 otherwise
  const cplx<T>* __restrict__ Fx = reinterpret_cast<const cplx<T>*>(reinterpret_cast<const char*>(Fx_) + moff);
  const cplx<T>* __restrict__ Fy = reinterpret_cast<const cplx<T>*>(reinterpret_cast<const char*>(Fy_) + moff);
  const cplx<T>* __restrict__ S = reinterpret_cast<const cplx<T>*>(reinterpret_cast<const char*>(S_) + moff);
  cplx<T>* w = reinterpret_cast<cplx<T>*>(reinterpret_cast<char*>(w_) + moff);
  cplx<T>* __restrict__ psi = reinterpret_cast<cplx<T>*>(reinterpret_cast<char*>(psi_) + moff);
  double* v0 = reinterpret_cast<double*>(reinterpret_cast<char*>(v0_) + moff);
  const int t = (int)(idx / ((size_t)g.Hy * g.CW));
  const int rem = (int)(idx - (size_t)t * g.Hy * g.CW);
  const int q = rem >> g.cw_shift;
  const int mx = t * g.CW + (rem & (g.CW - 1));
  if (mx >= g.Wx) return;
  const int my = q <= g.My ? q : q - g.Hy;
  const bool zero = (mx == 0 && my == 0);
  const bool cut = is_cut(g, mx, my, g.num, g.den);
  if (mx == 0) {
    if (my < 0) return;                                   // written by the thread of (0, -my)
    if (zero) {
      // mean flow, Eq. (C1): only rhs1 contributes
      const double e = exp(-m.alpha * m.dt);
      v0[0] = e * (v0[0] + m.dt * (double)Fx[idx].x);
      v0[1] = e * (v0[1] + m.dt * (double)Fy[idx].x);
      w[idx] = mk<T>(0, 0);
      psi[idx] = mk<T>(0, 0);
      return;
    }
    const size_t idn = spec_index(g, g.Hy - my, 0);       // row of -my, mx = 0
    cplx<T> out = mk<T>(0, 0);
    if (!cut) {
      const cplx<T> a = naive_update<T>(g, m, 0, my, idx, Fx, Fy, S, w);
      const cplx<T> b = naive_update<T>(g, m, 0, -my, idn, Fx, Fy, S, w);
      out = (T)0.5 * (a + conj(b));
    }
    const T ik2 = inv_k2<T>(g, 0, my);                          // psi^ = w^/k^2 (line 13)
    w[idx] = out;
    w[idn] = conj(out);
    psi[idx] = ik2 * out;
    psi[idn] = ik2 * conj(out);
    return;
  }
  cplx<T> out = naive_update<T>(g, m, mx, my, idx, Fx, Fy, S, w);
  out = cut ? mk<T>(0, 0) : out;
  w[idx] = out;
  psi[idx] = inv_k2<T>(g, mx, my) * out;                       // line 13
}

// a5 for the two-spectrum form produced by k_fwd_row_fused:  rhs^ = A^ - i ky B^  with  A = i kx Gy + S',  B = Gx.
// Column mx = 0 carries A^(0,my) = S'^(0,my) + i Gy^(0,my); S'(0,.) and Gy(0,.) are transforms of real sequences, so
//   S'^(0,my) = (A^(0,my) + conj A^(0,-my)) / 2,   i Gy^(0,my) = (A^(0,my) - conj A^(0,-my)) / 2,
// and i kx Gy^ = 0 there.  Gy^(0,0) = Im A^(0,0) and Gx^(0,0) = Re B^(0,0) feed the mean-flow update (line 8, Eq. C1).
template <typename T>
__global__ void __launch_bounds__(256)
k_spectral_p2(Geom g, Model m, const cplx<T>* __restrict__ A_, const cplx<T>* __restrict__ B_, cplx<T>* w_,
              cplx<T>* __restrict__ psi_, double* v0_, size_t mstride) {
  pdl_wait();
  pdl_trigger();
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)g.NT * g.Hy * g.CW) return;
  const size_t moff = (size_t)blockIdx.y * mstride;      // ensemble member (bytes); 0 outside ensembles
  const cplx<T>* __restrict__ A = reinterpret_cast<const cplx<T>*>(reinterpret_cast<const char*>(A_) + moff);
  const cplx<T>* __restrict__ B = reinterpret_cast<const cplx<T>*>(reinterpret_cast<const char*>(B_) + moff);
  cplx<T>* w = reinterpret_cast<cplx<T>*>(reinterpret_cast<char*>(w_) + moff);
  cplx<T>* __restrict__ psi = reinterpret_cast<cplx<T>*>(reinterpret_cast<char*>(psi_) + moff);
  double* v0 = reinterpret_cast<double*>(reinterpret_cast<char*>(v0_) + moff);
  spectral_p2_point<T>(g, m, idx, A, B, w, psi, v0, [](size_t, cplx<T>, cplx<T>) {});
}

// ttsh_set_velocity: w^ = i kx v^y - i ky v^x, v^(0) kept, then the same post-processing
template <typename T>
__global__ void __launch_bounds__(256)
k_spectral_init(Geom g, const cplx<T>* __restrict__ Vx, const cplx<T>* __restrict__ Vy, cplx<T>* w,
                cplx<T>* __restrict__ psi, double* v0) {
  // threads enumerate the tile-major array in memory order: idx = (t Hy + q) CW + c
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)g.NT * g.Hy * g.CW) return;
  const int t = (int)(idx / ((size_t)g.Hy * g.CW));
  const int rem = (int)(idx - (size_t)t * g.Hy * g.CW);
  const int q = rem >> g.cw_shift;
  const int mx = t * g.CW + (rem & (g.CW - 1));
  if (mx >= g.Wx) return;
  const int my = q <= g.My ? q : q - g.Hy;
  const bool cut = is_cut(g, mx, my, g.num, g.den);
  auto curl = [&](int my_, size_t id) -> cplx<T> {
    const T kx = (T)(g.dkx * mx), ky = (T)(g.dky * my_);
    return kx * mul_i(Vy[id]) - ky * mul_i(Vx[id]);
  };
  if (mx == 0) {
    if (my < 0) return;
    if (my == 0) {
      v0[0] = (double)Vx[idx].x;
      v0[1] = (double)Vy[idx].x;
      w[idx] = mk<T>(0, 0);
      psi[idx] = mk<T>(0, 0);
      return;
    }
    const size_t idn = spec_index(g, g.Hy - my, 0);
    cplx<T> out = mk<T>(0, 0);
    if (!cut) out = (T)0.5 * (curl(my, idx) + conj(curl(-my, idn)));
    const T ik2 = inv_k2<T>(g, 0, my);
    w[idx] = out;
    w[idn] = conj(out);
    psi[idx] = ik2 * out;
    psi[idn] = ik2 * conj(out);
    return;
  }
  const cplx<T> out = cut ? mk<T>(0, 0) : curl(my, idx);
  w[idx] = out;
  psi[idx] = inv_k2<T>(g, mx, my) * out;
}

// psi^ = w^/k^2 from a restored w^ (ttsh_set_state)
template <typename T>
__global__ void __launch_bounds__(256)
k_psi_from_w(Geom g, const cplx<T>* __restrict__ w, cplx<T>* __restrict__ psi) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)g.NT * g.Hy * g.CW) return;
  const int t = (int)(idx / ((size_t)g.Hy * g.CW));
  const int rem = (int)(idx - (size_t)t * g.Hy * g.CW);
  const int q = rem >> g.cw_shift;
  const int mx = t * g.CW + (rem & (g.CW - 1));
  const int my = q <= g.My ? q : q - g.Hy;
  psi[idx] = (mx >= g.Wx || (mx == 0 && my == 0)) ? mk<T>(0, 0) : inv_k2<T>(g, mx, my) * w[idx];
}

// Checkpoints (ttsh_get_state / ttsh_set_state) cross the C ABI in NATURAL order, complex[Hy][Wx]: element (q, mx) at q Wx + mx,
// so that their size and layout do not depend on the tile width CW of this build (col_tile_width and the TTSH_COL_* macros).
// pack: tile-major -> natural.  unpack: natural -> tile-major, padding columns mx >= Wx set to zero (they never hold anything else).
template <typename T>
__global__ void __launch_bounds__(256) k_state_pack(Geom g, const cplx<T>* __restrict__ w, cplx<T>* __restrict__ nat) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)g.Hy * g.Wx) return;
  const int q = (int)(idx / g.Wx), mx = (int)(idx - (size_t)q * g.Wx);
  nat[idx] = w[spec_index(g, q, mx)];
}
template <typename T>
__global__ void __launch_bounds__(256) k_state_unpack(Geom g, const cplx<T>* __restrict__ nat, cplx<T>* __restrict__ w) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)g.NT * g.Hy * g.CW) return;
  const int t = (int)(idx / ((size_t)g.Hy * g.CW));
  const int rem = (int)(idx - (size_t)t * g.Hy * g.CW);
  const int q = rem >> g.cw_shift;
  const int mx = t * g.CW + (rem & (g.CW - 1));
  w[idx] = mx < g.Wx ? nat[(size_t)q * g.Wx + mx] : mk<T>(0, 0);
}

// natural <-> permuted row layout of the internal real fields (perm_index: x = j + k TPL -> ((k>>2) TPL + j) 4 + (k&3)).
// Only for buffers that cross the C ABI in natural order (a processed mask, debug copies).
template <typename T>
__global__ void k_permute_rows(int Nx, size_t n, const T* __restrict__ in, T* __restrict__ out, int to_perm) {
  const int tpl = Nx / 16;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t row = i / Nx;
    const int x = (int)(i - row * Nx);
    const int j = x % tpl, k = x / tpl;
    const size_t pi = row * Nx + (size_t)(((k >> 2) * tpl + j) * 4 + (k & 3));
    if (to_perm) out[pi] = in[i]; else out[i] = in[pi];
  }
}

template <typename T>
__global__ void k_reperm_wl(int Nx, size_t n, const T* __restrict__ in, T* __restrict__ out) {
  const int tpl = Nx / 16;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t row = i / Nx;
    const int x = (int)(i - row * Nx);
    out[row * Nx + perm_index_wl(x, tpl)] = in[row * Nx + perm_index(x, tpl)];
  }
}

// K for row_step_real.cuh: slot n = own(t) + TPL k of thread t (TPL = Nx/32 threads; own(t) = wl_j(t) = (t >> 4) + (TPL/16) (t & 15) for the
// warp-local plan, t for the plain plan) holds the points x = 2n, 2n+1 of the row;  out[y Nx + (k TPL + t) 2 + par] = K(y, 2n + par).
// natural: the source rows are in natural order (Nx = 16384), else in the permuted internal layout (perm_index).
template <typename T>
__global__ void k_reperm_real(int Nx, size_t n, const T* __restrict__ in, T* __restrict__ out, int wl, int natural) {
  const int tpl_in = Nx / 16, TPL = Nx / 32, r1 = TPL / 16;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t row = i / (size_t)Nx;
    const int e = (int)(i - row * (size_t)Nx), par = e & 1, t = (e >> 1) % TPL, k = (e >> 1) / TPL;
    const int own = wl ? (t >> 4) + r1 * (t & 15) : t;     // warp-local plan: wl_j(t); plain plan: t
    const int x = 2 * (own + TPL * k) + par;
    out[i] = in[row * Nx + (natural ? x : perm_index(x, tpl_in))];
  }
}

// ---------------------------------------------------------------------------------------
// small helpers for Algorithm 2
// ---------------------------------------------------------------------------------------
template <typename T>
__global__ void k_mask_to_real(size_t n, const unsigned char* __restrict__ mask, T* __restrict__ out) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    out[i] = mask[i] ? (T)1 : (T)0;
}
template <typename T>
__global__ void k_square(size_t n, const T* __restrict__ in, T* __restrict__ out) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const T s = in[i];
    out[i] = s * s;                                                           // line 9
  }
}
template <typename T>
__global__ void k_fill(size_t n, T* __restrict__ out, T val) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    out[i] = val;
}

// ---------------------------------------------------------------------------------------
// a7: diagnostics.  Stage 1: grid-stride accumulation in fp64, warp-shuffle + smem block reduction, one
// partial record per block.  Stage 2: one block reduces the partials (fixed order => deterministic).
// record: [0] sum|v|^2  [1] sum w^2  [2] sum|v|  [3] sum|e_theta.v|  [4] sum vx  [5] sum vy  [6] max|v|  [7] #nonfinite
// ---------------------------------------------------------------------------------------
constexpr int DIAG_REC = 8;

__device__ __forceinline__ void diag_warp_reduce(double* a) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
    for (int k = 0; k < DIAG_REC; ++k) {
      const double o = __shfl_down_sync(0xffffffffu, a[k], off);
      if (k == 6) a[k] = fmax(a[k], o); else a[k] += o;
    }
  }
}

__device__ __forceinline__ void diag_block_reduce(double* a, double* out) {
  __shared__ double sh[32][DIAG_REC];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  diag_warp_reduce(a);
  if (lane == 0)
    for (int k = 0; k < DIAG_REC; ++k) sh[wid][k] = a[k];
  __syncthreads();
  if (wid == 0) {
    for (int k = 0; k < DIAG_REC; ++k) a[k] = lane < nw ? sh[lane][k] : 0.0;
    diag_warp_reduce(a);
    if (lane == 0)
      for (int k = 0; k < DIAG_REC; ++k) out[k] = a[k];
  }
}

template <typename T>
__global__ void __launch_bounds__(256)
k_diag_partial(int Nx, int Ny, double dx, double cx, double cy, const T* __restrict__ vx, const T* __restrict__ vy,
               const T* __restrict__ w, double* __restrict__ partial) {
  double a[DIAG_REC];
#pragma unroll
  for (int k = 0; k < DIAG_REC; ++k) a[k] = 0.0;
  const size_t n = (size_t)Nx * Ny;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const double u = (double)vx[i], v = (double)vy[i], ww = (double)w[i];
    const int ix = (int)(i % Nx), iy = (int)(i / Nx);
    const double x = ix * dx - cx, y = iy * dx - cy;
    const double r = sqrt(x * x + y * y);
    const double s2 = u * u + v * v;
    const double vth = r == 0.0 ? 0.0 : (-y * u + x * v) / r;       // e_theta . v  (Eq. 11)
    a[0] += s2;
    a[1] += ww * ww;
    a[2] += sqrt(s2);
    a[3] += fabs(vth);
    a[4] += u;
    a[5] += v;
    a[6] = fmax(a[6], sqrt(s2));
    a[7] += (isfinite(u) ? 0.0 : 1.0) + (isfinite(v) ? 0.0 : 1.0) + (isfinite(ww) ? 0.0 : 1.0);
  }
  diag_block_reduce(a, partial + (size_t)blockIdx.x * DIAG_REC);
}

__global__ void __launch_bounds__(256) k_diag_final(int nblocks, const double* __restrict__ partial, double* __restrict__ out) {
  double a[DIAG_REC];
#pragma unroll
  for (int k = 0; k < DIAG_REC; ++k) a[k] = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += blockDim.x)
#pragma unroll
    for (int k = 0; k < DIAG_REC; ++k) {
      const double o = partial[(size_t)b * DIAG_REC + k];
      if (k == 6) a[k] = fmax(a[k], o); else a[k] += o;
    }
  diag_block_reduce(a, out);
}

// ---------------------------------------------------------------------------------------
// Psi_2 of the dumbbell geometry: per side, argmax of |w| over the grid points within `radius` of the cavity
// centre, (i dx - cx)^2 + (j dx - cy)^2 <= radius^2 evaluated in fp64 without contraction (the same IEEE operations as the
// definition), ties to the lowest linear index.  Record per side: (|w|, w, index); index -1 = no point.
// ---------------------------------------------------------------------------------------
struct ArgBest { double a, v, i; };
__device__ __forceinline__ void arg_merge(ArgBest& x, double a, double v, double i) {
  if (a > x.a || (a == x.a && i < x.i)) { x.a = a; x.v = v; x.i = i; }
}
__device__ __forceinline__ void arg_warp_reduce(ArgBest& x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const double a = __shfl_down_sync(0xffffffffu, x.a, o), v = __shfl_down_sync(0xffffffffu, x.v, o), i = __shfl_down_sync(0xffffffffu, x.i, o);
    arg_merge(x, a, v, i);
  }
}
__device__ __forceinline__ void arg_block_reduce(ArgBest* x, double* out) {     // x[2] -> out[6], thread 0 writes
  __shared__ double sh[32][6];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  for (int s = 0; s < 2; ++s) {
    arg_warp_reduce(x[s]);
    if (lane == 0) { sh[wid][3 * s] = x[s].a; sh[wid][3 * s + 1] = x[s].v; sh[wid][3 * s + 2] = x[s].i; }
  }
  __syncthreads();
  if (wid == 0) {
    for (int s = 0; s < 2; ++s) {
      ArgBest y;
      y.a = lane < nw ? sh[lane][3 * s] : -1.0; y.v = lane < nw ? sh[lane][3 * s + 1] : 0.0; y.i = lane < nw ? sh[lane][3 * s + 2] : -1.0;
      arg_warp_reduce(y);
      if (lane == 0) { out[3 * s] = y.a; out[3 * s + 1] = y.v; out[3 * s + 2] = y.i; }
    }
  }
}
template <typename T>
__global__ void __launch_bounds__(256)
k_region_argmax_partial(int Nx, int Ny, double dx, double cxl, double cyl, double cxr, double cyr, double radius,
                        const T* __restrict__ w, double* __restrict__ partial) {
  ArgBest x[2];
  x[0].a = x[1].a = -1.0; x[0].v = x[1].v = 0.0; x[0].i = x[1].i = -1.0;
  const double r2 = __dmul_rn(radius, radius);
  const size_t n = (size_t)Nx * Ny;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const double px = __dmul_rn((double)(int)(i % Nx), dx), py = __dmul_rn((double)(int)(i / Nx), dx);
    const double ww = (double)w[i];
    const double xl = __dsub_rn(px, cxl), yl = __dsub_rn(py, cyl), xr = __dsub_rn(px, cxr), yr = __dsub_rn(py, cyr);
    if (__dadd_rn(__dmul_rn(xl, xl), __dmul_rn(yl, yl)) <= r2) arg_merge(x[0], fabs(ww), ww, (double)i);
    if (__dadd_rn(__dmul_rn(xr, xr), __dmul_rn(yr, yr)) <= r2) arg_merge(x[1], fabs(ww), ww, (double)i);
  }
  arg_block_reduce(x, partial + (size_t)blockIdx.x * DIAG_REC);
}
__global__ void __launch_bounds__(256) k_region_argmax_final(int nblocks, const double* __restrict__ partial, double* __restrict__ out) {
  ArgBest x[2];
  x[0].a = x[1].a = -1.0; x[0].v = x[1].v = 0.0; x[0].i = x[1].i = -1.0;
  for (int b = threadIdx.x; b < nblocks; b += blockDim.x)
    for (int s = 0; s < 2; ++s) {
      const double* r = partial + (size_t)b * DIAG_REC + 3 * s;
      arg_merge(x[s], r[0], r[1], r[2]);
    }
  arg_block_reduce(x, out);
}

// ---------------------------------------------------------------------------------------
// streaming temporal PSD, Eq. (5): per point and frequency one complex accumulator
//   A_m(x) += w(x, t) exp(-i Omega_m t);     S(Omega_m) = (1/P) sum_x |A_m(x)|^2
// acc is frequency-major [nf][n]: every access is unit-stride.  The phases of one sample (host-computed, <= 64 per launch)
// travel as a kernel argument.  Pure streaming: 2 x sizeof(cplx<T>) bytes per point and frequency -> HBM-bound.
// ---------------------------------------------------------------------------------------
constexpr int PSD_CHUNK = 64;
constexpr int PSD_BLOCKS = 296;
struct PsdPhases { double c[PSD_CHUNK], s[PSD_CHUNK]; };      // cos(Omega t), -sin(Omega t)

template <typename T>
__global__ void __launch_bounds__(256)
k_psd_accumulate(size_t n, int nf, const __grid_constant__ PsdPhases ph, const T* __restrict__ w, cplx<T>* __restrict__ acc) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const T ww = w[i];
    int m = 0;
    for (; m + 4 <= nf; m += 4) {                 // four independent read-modify-write streams in flight per thread
      cplx<T> v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) v[u] = acc[(size_t)(m + u) * n + i];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        v[u].x += ww * (T)ph.c[m + u];
        v[u].y += ww * (T)ph.s[m + u];
        acc[(size_t)(m + u) * n + i] = v[u];
      }
    }
    for (; m < nf; ++m) {
      cplx<T> v = acc[(size_t)m * n + i];
      v.x += ww * (T)ph.c[m];
      v.y += ww * (T)ph.s[m];
      acc[(size_t)m * n + i] = v;
    }
  }
}
// partial[m][b] = sum over the block's points of |A_m|^2 (fp64);  grid (PSD_BLOCKS, nf)
template <typename T>
__global__ void __launch_bounds__(256) k_psd_power_partial(size_t n, const cplx<T>* __restrict__ acc, double* __restrict__ partial) {
  const cplx<T>* a = acc + (size_t)blockIdx.y * n;
  double sum = 0.0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const double x = (double)a[i].x, y = (double)a[i].y;
    sum += x * x + y * y;
  }
  __shared__ double sh[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
  if (lane == 0) sh[wid] = sum;
  __syncthreads();
  if (wid == 0) {
    sum = lane < (int)(blockDim.x >> 5) ? sh[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
    if (lane == 0) partial[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = sum;
  }
}
// out[m] = sum_b partial[m][b];  grid nf, one warp each
__global__ void __launch_bounds__(32) k_psd_power_final(int nblocks, const double* __restrict__ partial, double* __restrict__ out) {
  double sum = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += 32) sum += partial[(size_t)blockIdx.x * nblocks + b];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
  if (threadIdx.x == 0) out[blockIdx.x] = sum;
}

// ---------------------------------------------------------------------------------------
// tangent-linear step (Lyapunov exponents): derivative of lines 1-2 of Algorithm 1 in the conservative
// form of k_realspace_cons at the base state (u, v, w), applied to a perturbation (du, dv, dw); in place:
//   c = -beta (u^2 + v^2) - gamma_v K,   dc = -2 beta (u du + v dv)
//   du <- dGx = dc u + c du + lambda0 (dv w + v dw),   dv <- dGy = dc v + c dv - lambda0 (du w + u dw),   dw <- -gamma_w K dw
// ---------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256)
k_realspace_tangent(size_t nvec, Model m, const T* __restrict__ vx, const T* __restrict__ vy, const T* __restrict__ w,
                    const T* __restrict__ K, T* __restrict__ dvx_, T* __restrict__ dvy_, T* __restrict__ dw_, size_t mstride) {
  pdl_wait();
  const size_t moff = (size_t)blockIdx.y * mstride;      // tangent vector (bytes); the base fields and K are shared
  T* __restrict__ dvx = reinterpret_cast<T*>(reinterpret_cast<char*>(dvx_) + moff);
  T* __restrict__ dvy = reinterpret_cast<T*>(reinterpret_cast<char*>(dvy_) + moff);
  T* __restrict__ dw = reinterpret_cast<T*>(reinterpret_cast<char*>(dw_) + moff);
  using V = typename Vec<T>::type;
  constexpr int n = Vec<T>::n;
  const T beta = (T)m.beta, gv = (T)m.gamma_v, gw = (T)m.gamma_w, lam = (T)m.lambda0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    V a = reinterpret_cast<const V*>(vx)[i], b = reinterpret_cast<const V*>(vy)[i], ww = reinterpret_cast<const V*>(w)[i];
    V k = reinterpret_cast<const V*>(K)[i];
    V da = reinterpret_cast<V*>(dvx)[i], db = reinterpret_cast<V*>(dvy)[i], dww = reinterpret_cast<V*>(dw)[i];
    T* pa = reinterpret_cast<T*>(&a); T* pb = reinterpret_cast<T*>(&b); T* pw = reinterpret_cast<T*>(&ww); T* pk = reinterpret_cast<T*>(&k);
    T* pda = reinterpret_cast<T*>(&da); T* pdb = reinterpret_cast<T*>(&db); T* pdw = reinterpret_cast<T*>(&dww);
#pragma unroll
    for (int e = 0; e < n; ++e) {
      const T u = pa[e], v = pb[e], om = pw[e], kk = pk[e], du = pda[e], dv = pdb[e], dom = pdw[e];
      const T c = -beta * (u * u + v * v) - gv * kk;
      const T dc = (T)-2 * beta * (u * du + v * dv);
      pda[e] = dc * u + c * du + lam * (dv * om + v * dom);
      pdb[e] = dc * v + c * dv - lam * (du * om + u * dom);
      pdw[e] = -gw * kk * dom;
    }
    reinterpret_cast<V*>(dvx)[i] = da;
    reinterpret_cast<V*>(dvy)[i] = db;
    reinterpret_cast<V*>(dw)[i] = dww;
  }
}

// Gram-Schmidt on tangent vectors (a^, a0) = (pruned tile-major half spectrum, mean flow[2]).  Inner product = the Euclidean
// one of the real vectors [a(x) ; a0] = sum over the FULL spectrum of Re(a^ conj b^) + a0 . b0 (unitary DFT): stored entries
// of the column mx = 0 count once (both +-my are stored), mx > 0 twice (their conjugates are implicit).
template <typename T>
__global__ void __launch_bounds__(256)
k_spec_dot_partial(Geom g, const cplx<T>* __restrict__ a, const cplx<T>* __restrict__ b_, double* __restrict__ partial, size_t bstride) {
  pdl_wait();
  // grid.y = vector j of a batch <a, b_j>, b_j = b_ + j * bstride bytes;  partial[j][gridDim.x]
  const cplx<T>* __restrict__ b = reinterpret_cast<const cplx<T>*>(reinterpret_cast<const char*>(b_) + (size_t)blockIdx.y * bstride);
  const size_t n = (size_t)g.NT * g.Hy * g.CW;
  double sum = 0.0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int t = (int)(i / ((size_t)g.Hy * g.CW));
    const int mx = t * g.CW + (int)(i & (size_t)(g.CW - 1));
    if (mx >= g.Wx) continue;
    const double re = (double)a[i].x * (double)b[i].x + (double)a[i].y * (double)b[i].y;
    sum += mx == 0 ? re : 2.0 * re;
  }
  __shared__ double sh[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
  if (lane == 0) sh[wid] = sum;
  __syncthreads();
  if (wid == 0) {
    sum = lane < (int)(blockDim.x >> 5) ? sh[lane] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
    if (lane == 0) partial[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = sum;
  }
}
// one warp per vector j (blockIdx.x): total = sum partial + a0 . b0.  norm_slot >= 0: rdiag[norm_slot] = sqrt(total), coef[0] = 1 / sqrt(total)
// (0 if total == 0); else coef[0] = total.
__global__ void __launch_bounds__(32)
k_spec_dot_final(int nblocks, const double* __restrict__ partial, const double* __restrict__ a0, const double* __restrict__ b0_,
                 size_t bstride, int norm_slot, double* __restrict__ rdiag, double* __restrict__ coef_) {
  pdl_wait();
  const double* __restrict__ b0 = reinterpret_cast<const double*>(reinterpret_cast<const char*>(b0_) + (size_t)blockIdx.x * bstride);
  double* __restrict__ coef = coef_ + blockIdx.x;
  double sum = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += 32) sum += partial[(size_t)blockIdx.x * nblocks + b];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
  if (threadIdx.x == 0) {
    sum += a0[0] * b0[0] + a0[1] * b0[1];
    if (norm_slot >= 0) {
      const double r = sqrt(sum);
      rdiag[norm_slot] = r;
      coef[0] = r > 0.0 ? 1.0 / r : 0.0;
    } else coef[0] = sum;
  }
}
// scale: y <- coef y (x == nullptr);  axpy: y <- y - coef x.  coef is read from device memory (no host round trip in the QR).
template <typename T>
__global__ void __launch_bounds__(256)
k_spec_scale_axpy(size_t n, const double* __restrict__ coef_, const cplx<T>* __restrict__ x, cplx<T>* __restrict__ y_,
                  const double* __restrict__ x0, double* __restrict__ y0_, size_t ystride) {
  pdl_wait();
  // grid.y = vector j of a batch: y_j = y_ + j * ystride bytes, coefficient coef_[j]
  const double* __restrict__ coef = coef_ + blockIdx.y;
  cplx<T>* __restrict__ y = reinterpret_cast<cplx<T>*>(reinterpret_cast<char*>(y_) + (size_t)blockIdx.y * ystride);
  double* __restrict__ y0 = reinterpret_cast<double*>(reinterpret_cast<char*>(y0_) + (size_t)blockIdx.y * ystride);
  const T c = (T)coef[0];
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    cplx<T> v = y[i];
    if (x) { const cplx<T> u = x[i]; v.x -= c * u.x; v.y -= c * u.y; }
    else { v.x *= c; v.y *= c; }
    y[i] = v;
  }
  if (blockIdx.x == 0 && threadIdx.x < 2) {
    const double cd = coef[0];
    y0[threadIdx.x] = x0 ? y0[threadIdx.x] - cd * x0[threadIdx.x] : cd * y0[threadIdx.x];
  }
}


// ---------------------------------------------------------------------------------------
// Blocked QR of the tangent vectors (CholeskyQR2) in the same inner product as above: G = A^T A in one launch, R = chol(G) on
// the host (nvec <= 64), A <- A R^-1 in one launch, twice; R = R2 R1.  Against Gram-Schmidt row by row (6 launches per vector)
// this is 3 launches per pass whatever nvec.
// k_gram_partial: grid (blocks, nvec, ceil(nvec / 8)); block (b, i, jt) accumulates <v_i, v_j> for the 8 vectors j of tile jt with
// j >= i over its share of the spectrum.  partial[(i nvec + j) nblocks + b].
// ---------------------------------------------------------------------------------------
constexpr int GRAM_TILE = 8;
template <typename T>
__global__ void __launch_bounds__(256)
k_gram_partial(Geom g, const cplx<T>* __restrict__ v_, size_t vstride, int nvec, double* __restrict__ partial) {
  pdl_wait();
  const int i = blockIdx.y, j0 = blockIdx.z * GRAM_TILE;
  if (j0 + GRAM_TILE <= i) return;                      // nothing of this tile lies on or above the diagonal
  const cplx<T>* __restrict__ a = reinterpret_cast<const cplx<T>*>(reinterpret_cast<const char*>(v_) + (size_t)i * vstride);
  const size_t n = (size_t)g.NT * g.Hy * g.CW;
  double acc[GRAM_TILE];
#pragma unroll
  for (int u = 0; u < GRAM_TILE; ++u) acc[u] = 0.0;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
    const int t = (int)(e / ((size_t)g.Hy * g.CW));
    const int mx = t * g.CW + (int)(e & (size_t)(g.CW - 1));
    if (mx >= g.Wx) continue;
    const double wgt = mx == 0 ? 1.0 : 2.0;
    const double ax = wgt * (double)a[e].x, ay = wgt * (double)a[e].y;
#pragma unroll
    for (int u = 0; u < GRAM_TILE; ++u) {
      const int j = j0 + u;
      if (j < i || j >= nvec) continue;
      const cplx<T> b = reinterpret_cast<const cplx<T>*>(reinterpret_cast<const char*>(v_) + (size_t)j * vstride)[e];
      acc[u] += ax * (double)b.x + ay * (double)b.y;
    }
  }
  __shared__ double sh[8][GRAM_TILE];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int u = 0; u < GRAM_TILE; ++u) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc[u] += __shfl_down_sync(0xffffffffu, acc[u], o);
    if (lane == 0) sh[wid][u] = acc[u];
  }
  __syncthreads();
  if (threadIdx.x < GRAM_TILE) {
    const int j = j0 + threadIdx.x;
    if (j >= i && j < nvec) {
      double s = 0.0;
      for (int w = 0; w < 8; ++w) s += sh[w][threadIdx.x];
      partial[((size_t)i * nvec + j) * gridDim.x + blockIdx.x] = s;
    }
  }
}
// one warp per entry (i, j >= i): G[i][j] = G[j][i] = sum of the partials + the mean-flow part
__global__ void __launch_bounds__(32)
k_gram_final(int nblocks, int nvec, const double* __restrict__ partial, const double* __restrict__ v0_, size_t vstride, double* __restrict__ G) {
  pdl_wait();
  const int i = blockIdx.y, j = blockIdx.x;
  if (j < i) return;
  double s = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += 32) s += partial[((size_t)i * nvec + j) * nblocks + b];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
  if (threadIdx.x == 0) {
    const double* a0 = reinterpret_cast<const double*>(reinterpret_cast<const char*>(v0_) + (size_t)i * vstride);
    const double* b0 = reinterpret_cast<const double*>(reinterpret_cast<const char*>(v0_) + (size_t)j * vstride);
    s += a0[0] * b0[0] + a0[1] * b0[1];
    G[i * nvec + j] = s;
    G[j * nvec + i] = s;
  }
}
// G = R^T R (R upper triangular, positive diagonal) and S = R^-1 for nvec <= 64, one block of 64 threads (thread j owns column
// j); logr[i] += log R_ii.  A pivot at or below 1e-13 of its diagonal entry (numerically dependent vectors) sets *flag and leaves
// S = identity, so that the following k_tri_apply changes nothing and the host can fall back to Gram-Schmidt.
__global__ void __launch_bounds__(64) k_chol_inv(int M, const double* __restrict__ G, double* __restrict__ S, double* __restrict__ logr, int* flag) {
  pdl_wait();
  __shared__ double R[64][65];
  __shared__ int bad;
  const int j = threadIdx.x;
  if (j == 0) bad = *flag;
  for (int i = 0; i < M; ++i) R[i][j] = (j < M) ? G[i * M + j] : 0.0;
  __syncthreads();
  for (int k = 0; k < M && !bad; ++k) {
    if (j == k) {
      const double d = R[k][k];
      if (!(d > 1e-13 * G[k * M + k]) || !isfinite(d)) bad = 1; else R[k][k] = sqrt(d);
    }
    __syncthreads();
    if (bad) break;
    if (j > k && j < M) R[k][j] /= R[k][k];
    __syncthreads();
    if (j > k && j < M)
      for (int i = k + 1; i <= j; ++i) R[i][j] -= R[k][i] * R[k][j];
    __syncthreads();
  }
  __syncthreads();
  if (j < M) {
    if (bad) {
      for (int i = 0; i < M; ++i) S[i * M + j] = (i == j) ? 1.0 : 0.0;
    } else {
      // column j of S = R^-1 by back substitution (entries below the diagonal are zero)
      double col[64];
      col[j] = 1.0 / R[j][j];
      for (int i = j - 1; i >= 0; --i) {
        double v = 0.0;
        for (int k = i + 1; k <= j; ++k) v -= R[i][k] * col[k];
        col[i] = v / R[i][i];
      }
      for (int i = 0; i < M; ++i) S[i * M + j] = i <= j ? col[i] : 0.0;
      logr[j] += log(R[j][j]);
    }
  }
  if (j == 0 && bad) *flag = 1;
}

// A <- A S with S upper triangular (S = R^-1, row-major S[i nvec + j]): q_j = sum_{i <= j} S[i][j] a_i, computed in place from the
// last column to the first (q_j needs only a_i, i <= j).  Also psi^_j = q_j / k^2 (line 13) and the mean-flow part (block 0).
template <typename T>
__global__ void __launch_bounds__(256)
k_tri_apply(Geom g, int nvec, const double* __restrict__ S, cplx<T>* v_, cplx<T>* __restrict__ psi_, double* v0_, size_t vstride) {
  pdl_wait();
  const size_t n = (size_t)g.NT * g.Hy * g.CW;
  auto vec = [&](cplx<T>* p, int j) { return reinterpret_cast<cplx<T>*>(reinterpret_cast<char*>(p) + (size_t)j * vstride); };
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
    const int t = (int)(e / ((size_t)g.Hy * g.CW));
    const int rem = (int)(e - (size_t)t * g.Hy * g.CW);
    const int q = rem >> g.cw_shift;
    const int mx = t * g.CW + (rem & (g.CW - 1));
    const int my = q <= g.My ? q : q - g.Hy;
    const bool dead = mx >= g.Wx || (mx == 0 && my == 0);
    const T ik2 = dead ? (T)0 : inv_k2<T>(g, mx, my);
    for (int j = nvec - 1; j >= 0; --j) {
      double sx = 0.0, sy = 0.0;
      for (int i = 0; i <= j; ++i) {
        const double c = S[i * nvec + j];
        const cplx<T> a = vec(v_, i)[e];
        sx += c * (double)a.x; sy += c * (double)a.y;
      }
      const cplx<T> out = dead ? mk<T>(0, 0) : mk<T>((T)sx, (T)sy);
      vec(v_, j)[e] = out;
      vec(psi_, j)[e] = ik2 * out;
    }
  }
  if (blockIdx.x == 0 && threadIdx.x < 2) {
    for (int j = nvec - 1; j >= 0; --j) {
      double s = 0.0;
      for (int i = 0; i <= j; ++i)
        s += S[i * nvec + j] * reinterpret_cast<double*>(reinterpret_cast<char*>(v0_) + (size_t)i * vstride)[threadIdx.x];
      reinterpret_cast<double*>(reinterpret_cast<char*>(v0_) + (size_t)j * vstride)[threadIdx.x] = s;
    }
  }
}

}  // namespace ttsh
