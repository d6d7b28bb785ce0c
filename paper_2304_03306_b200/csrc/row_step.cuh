// row_step.cuh — the whole row half of one Euler step in ONE kernel (conservative advection form, 1/2 rule):
//
//   inverse row pass of w~, v_x~, psi~ (C2R, a2 + a6)  ->  rhs of Algorithm 1 lines 1-2 (a3)  ->  forward row pass (R2C, a4)
//
// All three operate on whole rows, and a thread of the Stockham transform owns the same 16 x-positions x = j + k TPL at
// the output of an inverse transform as at the input of a forward one, so w, v_x, v_y never leave the SM: per row pair
// (y_A = 4a+p, y_B = y_A+2, packed as z = f(y_A) + i f(y_B)) the kernel reads three pruned intermediates and K and
// writes the two pruned intermediates  A~ = i k_x Gy~ + S'~  and  B~ = Gx~  (fft_passes.cuh, k_fwd_row_fused):
//   Gx = rhs1_x + lambda0 v_y w,  Gy = rhs1_y - lambda0 v_x w,  S' = -gamma_w K w,  rhs1 = -(beta |v|^2 + gamma_v K) v
// (PAPER.md:292-294, lines 1-3 of Algorithm 1 with lambda0 v.grad w = lambda0 div(v w)).
// HBM traffic per step for the row half: 3 x 0.5 U + 1 U (K) in, 2 x 0.5 U out = 3.5 U instead of 9.5 U for
// k_inv_row + k_fwd_row_fused.  Of the three packed fields one waits in shared memory (stash, [slot][thread], touched
// by its owner thread only), one in registers (H) and one is the live transform (V).
// For Nx = 1024, 2048, 4096 the transforms use the warp-local plan of fft_core.cuh (one CTA-wide exchange per transform);
// the thread then owns x = wl_j(j) + k TPL, K is read from its thread-order copy (perm_index_wl) and tabX is the
// warp-local twiddle table.
// Packing by rows (f(y_A) + i f(y_B)) makes i k_x commute with the packing, so A~ is formed BEFORE the unpack:
//   T(m) = i k_m Zgy(m) + Zs(m),  k_m the signed wavenumber of bin m  ->  2 unpacks for 3 transforms.
#pragma once
#include "fft_passes.cuh"

namespace ttsh {

template <typename T, int NX> struct RowStepCfg {
  using R = RowCfg<T, NX>;
  static constexpr bool WL = fft_wl_supported<NX>();                   // warp-local FFT plan (fft_core.cuh)
  static constexpr int TPL = R::TPL, L = R::L, THREADS = R::THREADS;
  static constexpr int LS = WL ? fft_wl_line_elems<T, NX>() + 4 : R::LS;
  static constexpr int ST = NX;                                        // stash elements per line
  static constexpr size_t SMEM = (size_t)L * (LS + ST) * sizeof(cplx<T>);
  static constexpr int MINB = 1;
  static constexpr bool FITS = SMEM <= 227 * 1024;
};

// inverse row transform of one packed row pair into registers: out[k] = f(y_A, x) + i f(y_B, x), x = j + k TPL.
// MODE = RM_ONE or RM_NIKX_MEANY (ttsh_common.cuh).  1/2 rule only: retained mx = 0..NX/4.
// With the warp-local plan the thread owns x = wl_j(j) + k TPL instead (tabX is then the warp-local table).
template <typename T, int NX, int MODE>
__device__ __forceinline__ void inv_row_regs(const cplx<T>* __restrict__ row, int j, cplx<T>* __restrict__ line,
                                             const cplx<T>* __restrict__ tabX, T scale, T dkx, T meany, cplx<T> (&out)[16]) {
  auto mult = [&](cplx<T> w, int mx) -> cplx<T> {
    if (MODE == RM_ONE) return w;
    const T kx = dkx * (T)mx;
    return mx == 0 ? mk<T>(meany, (T)0) : kx * mul_ni(w);        // RM_NIKX_MEANY
  };
  auto combine = [&](Pair<T> r, int mx, bool neg) -> cplx<T> {
    cplx<T> wa = mult(r.a, mx), wb = mult(r.b, mx);
    if (mx == 0) { wa.y = 0; wb.y = 0; }
    if (neg) { wa = conj(wa); wb = conj(wb); }
    return scale * mk<T>(wa.x - wb.y, wa.y + wb.x);
  };
  auto zero_pair = [&]() -> Pair<T> { Pair<T> r; r.a = mk<T>(0, 0); r.b = mk<T>(0, 0); return r; };
  auto issue = [&](int m, int k) -> Pair<T> {
    if (k <= 3 || (k == 4 && j == 0)) return ld_pair(row + 2 * m);
    if (k >= 12) return ld_pair(row + 2 * (NX - m));
    return zero_pair();
  };
  auto finish = [&](int m, int k, Pair<T> r) -> cplx<T> {
    if (k <= 3) return combine(r, m, false);
    if (k == 4) return j == 0 ? combine(r, m, false) : mk<T>(0, 0);
    if (k >= 12) return combine(r, NX - m, true);
    return mk<T>(0, 0);
  };
  auto store = [&](int, int k, cplx<T> z) { out[k] = z; };
  if constexpr (fft_wl_supported<NX>()) fft_line_wl<T, NX, +1, false>(j, j, line, tabX, make_loader<2>(issue, finish), store);
  else fft_line<T, NX, +1, false>(j, line, tabX, make_loader<2>(issue, finish), store);
}

// forward transform of the 16 values a thread owns (slot k <-> x = jw + k TPL; jw = wl_j(j) for the warp-local plan, else j)
template <typename T, int NX, bool SYNC_LAST, class Load, class Store>
__device__ __forceinline__ void fwd_row_regs(int jw, int j, cplx<T>* __restrict__ line, const cplx<T>* __restrict__ tabX, Load load,
                                             Store store) {
  if constexpr (fft_wl_supported<NX>()) fft_line_wl<T, NX, -1, SYNC_LAST>(jw, j, line, tabX, load, store);
  else fft_line<T, NX, -1, SYNC_LAST>(j, line, tabX, load, store);
}
template <typename T, int NX> __device__ __forceinline__ int row_step_pad(int i) {
  if constexpr (fft_wl_supported<NX>()) return fft_wl_pad<T, NX>(i);
  else return fft_pad<NX>(i);
}

template <typename T, int NX>
__global__ void __launch_bounds__(RowStepCfg<T, NX>::THREADS, RowStepCfg<T, NX>::MINB)
k_row_step(const __grid_constant__ Geom g, const __grid_constant__ Model m, const cplx<T>* __restrict__ inW,
           const cplx<T>* __restrict__ inVx, const cplx<T>* __restrict__ inPsi, const T* __restrict__ K,
           cplx<T>* __restrict__ outA, cplx<T>* __restrict__ outB, const cplx<T>* __restrict__ tabX,
           const double* __restrict__ v0, int nblk) {
  using C = RowStepCfg<T, NX>;
  constexpr int TPL = C::TPL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int c = threadIdx.x / TPL, j = threadIdx.x % TPL;
  const int jw = C::WL ? (j >> 4) + (NX / 256) * (j & 15) : j;       // the x-class this thread owns: x = jw + k TPL
  cplx<T>* line = sm + c * C::LS;
  cplx<T>* stash = sm + C::L * C::LS + c * C::ST + j;      // slot k of this thread at stash[k TPL]
  const int Wx = g.Wx;
  const T scale_i = (T)g.inv_sqrt_nx, scale_f = (T)g.inv_sqrt_nx;
  const T dkx = (T)g.dkx;
  const T meany = (T)(v0[1] * g.inv_sqrt_ny);
  const T beta = (T)m.beta, gv = (T)m.gamma_v, lam = (T)m.lambda0;
  const T ngw = -(T)m.gamma_w * scale_f;
  const size_t in_stride = (size_t)g.Wxp * 2;               // elements per row pair of an inverse intermediate

#pragma unroll 1
  for (int blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
    const int rp = blk * C::L + c;
    const int a = rp >> 1, p = rp & 1;
    const size_t offA = (size_t)(4 * a + p) * NX, offB = offA + 2 * (size_t)NX;
    if (j == 0) {   // L2 prefetch of what this line reads in the CTA's next iteration
      const int nb = blk + gridDim.x;
      if (nb < nblk) {
        const int nrp = nb * C::L + c;
        const unsigned bytes = (unsigned)(in_stride * sizeof(cplx<T>));
        prefetch_l2_bulk(inW + (size_t)nrp * in_stride, bytes);
        prefetch_l2_bulk(inVx + (size_t)nrp * in_stride, bytes);
        prefetch_l2_bulk(inPsi + (size_t)nrp * in_stride, bytes);
        const size_t nA = (size_t)(4 * (nrp >> 1) + (nrp & 1)) * NX;
        prefetch_l2_bulk(K + nA, (unsigned)(NX * sizeof(T)));
        prefetch_l2_bulk(K + nA + 2 * (size_t)NX, (unsigned)(NX * sizeof(T)));
      }
    }
    cplx<T> H[16], V[16];
    // ---- a2 / a6: w, v_x, v_y of the two rows (x = j + k TPL) ----
    inv_row_regs<T, NX, RM_ONE>(inW + (size_t)rp * in_stride, j, line, tabX, scale_i, dkx, meany, V);
#pragma unroll
    for (int k = 0; k < 16; ++k) stash[k * TPL] = V[k];                     // w
    inv_row_regs<T, NX, RM_ONE>(inVx + (size_t)rp * in_stride, j, line, tabX, scale_i, dkx, meany, H);          // v_x
    inv_row_regs<T, NX, RM_NIKX_MEANY>(inPsi + (size_t)rp * in_stride, j, line, tabX, scale_i, dkx, meany, V);  // v_y
    // ---- a3: lines 1-2 of Algorithm 1, pointwise;  V <- Gx,  H <- Gy,  stash <- S'  (all scaled for the forward pass) ----
    {
      Quad<T> ka[4], kb[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const size_t e = ((size_t)q * TPL + j) * 4;
        ka[q] = ld_quad(K + offA + e);
        kb[q] = ld_quad(K + offB + e);
      }
#pragma unroll
      for (int k = 0; k < 16; ++k) {
        const cplx<T> w = stash[k * TPL];
        const T KA = ka[k >> 2].v[k & 3], KB = kb[k >> 2].v[k & 3];
        const T vxA = H[k].x, vxB = H[k].y, vyA = V[k].x, vyB = V[k].y;
        const T ccA = scale_f * (-beta * (vxA * vxA + vyA * vyA) - gv * KA);
        const T ccB = scale_f * (-beta * (vxB * vxB + vyB * vyB) - gv * KB);
        const T lwA = scale_f * lam * w.x, lwB = scale_f * lam * w.y;
        V[k] = mk<T>(ccA * vxA + lwA * vyA, ccB * vxB + lwB * vyB);          // Gx
        H[k] = mk<T>(ccA * vyA - lwA * vxA, ccB * vyB - lwB * vxB);          // Gy
        stash[k * TPL] = mk<T>(ngw * (KA * w.x), ngw * (KB * w.y));          // S'
      }
    }
    // ---- a4, transform 1: Gx -> B~ ----
    auto keep = [&](int k) -> bool { return k <= 3 || k >= 12 || (k == 4 && j == 0); };
    auto ident = [&](int, int, cplx<T> r) -> cplx<T> { return r; };
    {
      auto store = [&](int mm, int k, cplx<T> z) { if (keep(k)) line[row_step_pad<T, NX>(mm)] = z; };
      fwd_row_regs<T, NX, true>(jw, j, line, tabX, make_loader<1>([&](int, int k) -> cplx<T> { return V[k]; }, ident), store);
      __syncthreads();
      for (int mx = j; mx < Wx; mx += TPL) {
        const cplx<T> zp = line[row_step_pad<T, NX>(mx)];
        const cplx<T> zm = conj(line[row_step_pad<T, NX>((NX - mx) & (NX - 1))]);
        st_pair(outB + inter_pair_index(g, a, p, mx), (T)0.5 * (zp + zm), (T)0.5 * mul_ni(zp - zm));
      }
    }
    // ---- transform 2: Gy -> H <- i k_m Zgy(m) (retained bins only) ----
    cplx<T> zg0 = mk<T>(0, 0);
    {
      auto store = [&](int mm, int k, cplx<T> z) {
        if (k == 0) zg0 = z;                                       // thread j = 0: Zgy(0) = Gy~(0, y_A) + i Gy~(0, y_B)
        if (k <= 4) H[k] = (dkx * (T)mm) * mul_i(z);
        else if (k >= 12) H[k] = (dkx * (T)(mm - NX)) * mul_i(z);
      };
      fwd_row_regs<T, NX, false>(jw, j, line, tabX, make_loader<1>([&](int, int k) -> cplx<T> { return H[k]; }, ident), store);
    }
    // ---- transform 3: S' -> A~ = unpack(i k_m Zgy + Zs) ----
    {
      auto store = [&](int mm, int k, cplx<T> z) { if (keep(k)) line[row_step_pad<T, NX>(mm)] = z + H[k]; };
      fwd_row_regs<T, NX, true>(jw, j, line, tabX, make_loader<1>([&](int, int k) -> cplx<T> { return stash[k * TPL]; }, ident), store);
      __syncthreads();
      for (int mx = j; mx < Wx; mx += TPL) {
        const cplx<T> zp = line[row_step_pad<T, NX>(mx)];
        const cplx<T> zm = conj(line[row_step_pad<T, NX>((NX - mx) & (NX - 1))]);
        cplx<T> sa = (T)0.5 * (zp + zm), sb = (T)0.5 * mul_ni(zp - zm);
        if (mx == 0) {                // real numbers S'~(0,y) and Gy~(0,y) travel together (k_fwd_row_fused)
          sa = mk<T>(sa.x, zg0.x);
          sb = mk<T>(sb.x, zg0.y);
        }
        st_pair(outA + inter_pair_index(g, a, p, mx), sa, sb);
      }
    }
  }
}

}  // namespace ttsh
