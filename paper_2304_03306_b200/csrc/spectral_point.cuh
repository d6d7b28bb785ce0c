// spectral_point.cuh — lines 3-13 of Algorithm 1 for ONE retained mode of the two-spectrum form, shared by
// k_spectral_p2 (pointwise.cuh) and the fused column kernel (col_step.cuh) so that both evaluate the same expressions.
#pragma once
#include "ttsh_common.cuh"

namespace ttsh {

template <typename T> __device__ __forceinline__ T inv_k2(const Geom& g, int mx, int my) {
  const T kx = (T)(g.dkx * mx), ky = (T)(g.dky * my);
  return (T)1 / (kx * kx + ky * ky);
}

// idx: position in the tile-major spectrum, (t Hy + q) CW + c.  A, B: the two forward spectra (rhs^ = A^ - i ky B^; column mx = 0 of A
// carries S'^ + i Gy^, see k_spectral_p2); w: the state w^ (read at t, written at t + dt); psi: psi^ = w^/k^2; v0: the mean flow.
// A, B may point into shared memory shifted so that A[idx] is the mode's entry.  emit(i, w_new, psi_new) is called for every entry
// this thread writes (the thread of (0, my > 0) also writes (0, -my)).  A thread whose mode is written by another returns at once.
template <typename T, class Emit>
__device__ __forceinline__ void spectral_p2_point(const Geom& g, const Model& m, size_t idx, const cplx<T>* A, const cplx<T>* B,
                                                  cplx<T>* w, cplx<T>* psi, double* v0, Emit emit) {
  const int t = (int)(idx / ((size_t)g.Hy * g.CW));
  const int rem = (int)(idx - (size_t)t * g.Hy * g.CW);
  const int q = rem >> g.cw_shift;
  const int mx = t * g.CW + (rem & (g.CW - 1));
  if (mx >= g.Wx) return;
  const int my = q <= g.My ? q : q - g.Hy;
  const bool cut = is_cut(g, mx, my, g.num, g.den);
  const T dt = (T)m.dt;
  auto factor = [&](int my_) -> T {          // exp(sigma(k) dt), line 4
    const T kx = (T)(g.dkx * mx), ky = (T)(g.dky * my_);
    const T k2 = kx * kx + ky * ky;
    const T sigma = -(T)m.alpha - (T)m.Gamma0 * k2 - (T)m.Gamma2 * k2 * k2;
    return sizeof(T) == 8 ? (T)exp((double)(sigma * dt)) : (T)expf((float)(sigma * dt));
  };
  if (mx == 0) {
    if (my < 0) return;                                   // written by the thread of (0, -my)
    if (my == 0) {
      const double e = exp(-m.alpha * m.dt);
      v0[0] = e * (v0[0] + m.dt * (double)B[idx].x);      // Gx^(0,0)
      v0[1] = e * (v0[1] + m.dt * (double)A[idx].y);      // Gy^(0,0)
      w[idx] = mk<T>(0, 0);
      psi[idx] = mk<T>(0, 0);
      emit(idx, mk<T>(0, 0), mk<T>(0, 0));
      return;
    }
    const size_t idn = spec_index(g, g.Hy - my, 0);       // row of -my, mx = 0
    cplx<T> out = mk<T>(0, 0);
    if (!cut) {
      const T ky = (T)(g.dky * my);
      const cplx<T> sp = (T)0.5 * (A[idx] + conj(A[idn]));                   // S'^(0, my); S'^(0,-my) = conj
      const cplx<T> rp = sp - ky * mul_i(B[idx]);                            // rhs^(0, my)
      const cplx<T> rn = conj(sp) + ky * mul_i(B[idn]);                      // rhs^(0,-my)
      const T e = factor(my);
      const cplx<T> np_ = e * (w[idx] + dt * rp), nn = e * (w[idn] + dt * rn);
      out = (T)0.5 * (np_ + conj(nn));                                       // line 12
    }
    const T ik2 = inv_k2<T>(g, 0, my);
    w[idx] = out;
    w[idn] = conj(out);
    psi[idx] = ik2 * out;
    psi[idn] = ik2 * conj(out);
    emit(idx, out, ik2 * out);
    emit(idn, conj(out), ik2 * conj(out));
    return;
  }
  const T ky = (T)(g.dky * my);
  cplx<T> out = factor(my) * (w[idx] + dt * (A[idx] - ky * mul_i(B[idx])));  // lines 3-4
  out = cut ? mk<T>(0, 0) : out;
  const cplx<T> ps = inv_k2<T>(g, mx, my) * out;                             // line 13
  w[idx] = out;
  psi[idx] = ps;
  emit(idx, out, ps);
}

}  // namespace ttsh
