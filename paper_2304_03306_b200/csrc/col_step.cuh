// col_step.cuh — the whole COLUMN half of the time loop in one kernel, for grids whose step is bound by its four kernel boundaries
// rather than by work (Ny <= 1024):
//
//   forward column pass of A~, B~ (a4)  ->  lines 3-13 of Algorithm 1 (a5)  ->  inverse column pass of w^, psi^, i k_y psi^ of the
//   NEXT step (a2 / a6).
//
// All three stages are local to a tile of CW adjacent x-wavenumbers: the forward pass produces every y-wavenumber of its columns,
// the spectral update is pointwise (the Hermitian pair (0, my), (0, -my) lies in one column; the mean flow belongs to tile 0, the only
// tile that uses it), and the inverse pass reads exactly those columns again.  So a CTA takes one tile through all three with the
// spectra in shared memory, and an Euler step is TWO launches, k_row_step and this one, instead of four.  Six groups of threads run
// the transforms of a stage side by side — forward: (A, B) x (even, odd rows), inverse: (w, psi, i k_y psi) x (even, odd rows) — so
// the dependency chain is two half-length transforms and the pointwise update.
//
// Every number is computed by the expressions of k_fwd_col, k_spectral_p2 and k_inv_col on the same operands (the odd-row part is
// added to the even-row part in shared memory where k_fwd_col uses red.global.add: one addend per entry either way).  The results
// agree with the four-launch step to ROUND-OFF, not bit for bit: inlined into one kernel, the compiler contracts a few
// multiply-adds of the odd-row twiddle and of the spectral update differently (test_fused_column_kernel_against_the_four_launch_step
// bounds the difference by 1e-13 in fp64, 2e-5 in fp32; ttsh.h says the same).  An ensemble picks this kernel or the four launches
// by count x tiles against the SM count (ttsh_ensemble_create), so its round-off depends on count and on the device.  1/2 rule only.
#pragma once
#include "fft_passes.cuh"
#include "spectral_point.cuh"

namespace ttsh {

template <typename T, int NY> struct ColStepCfg {
  using C = ColCfg<T, NY>;
  static constexpr int NG = 6, GT = C::THREADS, THREADS = NG * GT;
  static constexpr int HY = NY / 2 + 1;                                     // retained rows under the 1/2 rule
  static constexpr size_t TILE = ((size_t)HY * C::L * sizeof(cplx<T>) + 127) / 128 * 128;
  static constexpr size_t OFF_TILES = ((size_t)NG * C::SMEM + 127) / 128 * 128;
  static constexpr size_t SMEM = OFF_TILES + 2 * TILE;
  static constexpr bool OK = NY >= 128 && NY <= 1024 && THREADS <= 1024 && SMEM <= 227 * 1024;   // 64^2: 15.9 us fused, 15.0 us in four launches
};

template <class P> __device__ __forceinline__ P* col_step_off(P* p, size_t bytes) {
  return reinterpret_cast<P*>(reinterpret_cast<char*>(const_cast<typename std::remove_const<P>::type*>(p)) + bytes);
}

// srcA / srcB: forward intermediates of A~, B~ (written by the row kernel); w, psi: the state; dstW / dstPsi / dstVx: inverse
// intermediates of w, psi and v_x = i k_y psi^ (+ mean flow) for the next row kernel.  grid = (NT tiles, members): member b of an
// ensemble (ttsh_ensemble_step) uses every pointer + b * mstride bytes; the twiddle tables are member 0's.
template <typename T, int NY>
__global__ void __launch_bounds__(ColStepCfg<T, NY>::THREADS, 1)
k_col_step(const __grid_constant__ Geom g, const __grid_constant__ Model m, const cplx<T>* __restrict__ srcA,
           const cplx<T>* __restrict__ srcB, cplx<T>* w, cplx<T>* psi, double* v0, cplx<T>* __restrict__ dstW,
           cplx<T>* __restrict__ dstPsi, cplx<T>* __restrict__ dstVx, const cplx<T>* __restrict__ tabY,
           const cplx<T>* __restrict__ tabS, size_t mstride) {
  using C = ColCfg<T, NY>;
  using S = ColStepCfg<T, NY>;
  constexpr int NH = C::NH, L = C::L, TPL = C::TPL, GT = S::GT;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  cplx<T>* tileA = reinterpret_cast<cplx<T>*>(smem_raw + S::OFF_TILES);            // A^, then w^(t + dt):  (q, c) at q L + c
  cplx<T>* tileB = reinterpret_cast<cplx<T>*>(smem_raw + S::OFF_TILES + S::TILE);  // B^, then psi^(t + dt)
  const size_t moff = (size_t)blockIdx.y * mstride;            // ensemble member (bytes); 0 outside ensembles
  srcA = col_step_off(srcA, moff); srcB = col_step_off(srcB, moff); w = col_step_off(w, moff); psi = col_step_off(psi, moff);
  v0 = col_step_off(v0, moff); dstW = col_step_off(dstW, moff); dstPsi = col_step_off(dstPsi, moff); dstVx = col_step_off(dstVx, moff);
  const int grp = (int)threadIdx.x / GT, tid = (int)threadIdx.x % GT;
  int j, c;
  col_thread_map<C::LSHIFT>(tid, j, c);
  const int t = blockIdx.x;
  const int mx = t * L + c;
  const bool valid = mx < g.Wx;
  const int Hy = g.Hy;                                                           // = S::HY (host-checked)
  const T scale = (T)g.inv_sqrt_ny;
  cplx<T>* line = sm + (grp * L + c) * C::LS;
  const cplx<T> wj = ldg_c(tabS + j);                                             // W_Ny^j
  const int p = grp & 1, fld = grp >> 1;
  constexpr size_t KS = (size_t)TPL * L;                                          // elements per slot in a tile
  pdl_wait();
  pdl_trigger();

  // ---- a4: forward column pass (k_fwd_col, 1/2-rule branch): groups 0..3 = (A, B) x (even rows, odd rows); groups 4, 5 idle ----
  {
    const bool work = fld < 2;
    const cplx<T>* in = (fld == 0 ? srcA : srcB) + (size_t)t * 2 * NH * L + tid + (size_t)p * NH * L;
    cplx<T>* tl = (fld == 0 ? tileA : tileB) + c;
    cplx<T>* dpos = tl + (size_t)j * L;
    cplx<T>* dneg = tl + (size_t)(Hy - NH + j) * L;
    cplx<T> odd[16];
    auto load = make_loader(
        [&](int, int k) -> cplx<T> { return (work && valid) ? in[(size_t)k * (L * TPL)] : mk<T>(0, 0); },
        [&](int, int, cplx<T> raw) -> cplx<T> { return scale * raw; });
    auto store = [&](int, int k, cplx<T> val) {
      if (p == 0) {
        if (!(work && valid)) return;
        if (k < 8 || (k == 8 && j == 0)) dpos[k * KS] = val;
        if (k >= 8) dneg[k * KS] = val;
      } else {
        odd[k] = mul_w32_rt<-1>(val * wj, k);                                     // W_Ny^{mp} O[mp]
      }
    };
    fft_line<T, NH, -1, false>(j, line, tabY, load, store);
    __syncthreads();
    if (p == 1 && work && valid) {
#pragma unroll
      for (int k = 0; k < 16; ++k) {
        const cplx<T> tw = odd[k];
        if (k < 8 || (k == 8 && j == 0)) dpos[k * KS] = dpos[k * KS] + tw;
        if (k >= 8) dneg[k * KS] = dneg[k * KS] + mk<T>(-tw.x, -tw.y);
      }
    }
    __syncthreads();
  }
  // ---- a5: lines 3-13 on the tile (k_spectral_p2); the new w^, psi^ go to the state AND stay in the tiles ----
  {
    const size_t base = (size_t)t * Hy * L;
    const cplx<T>* Av = tileA - base;             // A[idx] of the tile-major spectrum for the idx of this tile
    const cplx<T>* Bv = tileB - base;
    for (int e = threadIdx.x; e < Hy * L; e += S::THREADS) {
      spectral_p2_point<T>(g, m, base + e, Av, Bv, w, psi, v0, [&](size_t i, cplx<T> wn, cplx<T> pn) {
        tileA[i - base] = wn;
        tileB[i - base] = pn;
      });
    }
    __syncthreads();
  }
  // ---- a2 / a6 of the next step: inverse column pass (k_inv_col, 1/2-rule branch): (w^, psi^, i k_y psi^) x (even, odd rows) ----
  {
    const int mode = fld == 2 ? SM_IKY_MEANX : SM_ONE;
    const cplx<T>* src = (fld == 0 ? tileA : tileB) + c;
    cplx<T>* dsel = fld == 0 ? dstW : (fld == 1 ? dstPsi : dstVx);
    cplx<T>* out = dsel + ((size_t)(j & ~1) * g.Wxp + mx) * 2 + (j & 1) + (size_t)p * g.Wxp * 2;
    const size_t slot_stride = (size_t)TPL * g.Wxp * 2;
    auto store = [&](int, int k, cplx<T> val) { out[(size_t)k * slot_stride] = val; };
    auto twist = [&](int k, cplx<T> a) -> cplx<T> {
      if (p) a = mul_w32_rt<+1>(mul_conj(a, wj), k);
      return scale * a;
    };
    auto issue = [&](int mp, int k) -> cplx<T> {
      const int q = k < 8 ? mp : Hy + mp - NH;
      return valid ? src[(size_t)q * L] : mk<T>(0, 0);
    };
    auto finish = [&](int mp, int k, cplx<T> raw) -> cplx<T> {
      if (!valid) return mk<T>(0, 0);
      cplx<T> v = apply_spec_mode<T>(mode, raw, mx, k < 8 ? mp : mp - NH, g, v0);
      if (k >= 8 && p) v = mk<T>(-v.x, -v.y);
      if (k == 8 && j == 0) v = v + apply_spec_mode<T>(mode, src[(size_t)mp * L], mx, mp, g, v0);
      return twist(k, v);
    };
    fft_line<T, NH, +1, false>(j, line, tabY, make_loader(issue, finish), store);
  }
}

}  // namespace ttsh
