// fft_rows_real.cuh — row passes for rows too long to pack in pairs: ONE real row per complex transform of HALF the length.
//
// The row passes of fft_passes.cuh pack two real rows into one complex FFT of length Nx; at Nx = 16384 (the grid of Fig. 6(f),
// PAPER.md:282) that line is 256 KB in fp64 and does not fit in shared memory.  Here a real row x[0..N) is the complex sequence
// z[n'] = x[2n'] + i x[2n'+1] of length N2 = N/2 (128 KB in fp64 at N = 16384), transformed by the same Stockham line transform
// (fft_core.cuh), with the textbook split / merge step of a real FFT around it (PAPER.md:319 defines the unitary DFT):
//
//   forward (R2C):  Z = FFT_N2(z);   E[m] = (Z[m] + conj Z[N2-m]) / 2,   O[m] = -i (Z[m] - conj Z[N2-m]) / 2,
//                   X[m] = E[m] + W_N^m O[m],          m = 0 .. Wx-1  (only the retained band is written)
//   inverse (C2R):  Z[m] = (X[m] + conj X[N2-m]) + i conj(W_N^m) (X[m] - conj X[N2-m]),   m = 0 .. N2-1,
//                   z = iFFT_N2(Z),   x[2n'] = Re z[n'],  x[2n'+1] = Im z[n']        (X[m] = 0 outside the retained band)
//
// W_N^m with m = j + k N/32 factors as W_N^j W_32^k (the trick of the column passes): one table load per thread (tabR[j] = W_N^j,
// j < N/32) and compile-time constants.  One CTA per ROW, N/32 threads; the two rows of an (A, B) pair of the intermediate
// layouts (ttsh_common.cuh) are handled by two CTAs that read / write the two 16-byte (fp64) halves of each pair.  Real rows are
// in NATURAL order on both sides (a thread's two samples x[2n'], x[2n'+1] are adjacent, consecutive threads are consecutive):
// the permuted internal layout of the pair kernels is not used on these grids (RM_PERM is ignored).
#pragma once
#include "fft_passes.cuh"

namespace ttsh {

template <typename T, int NX> struct RealRowCfg {
  static constexpr int N2 = NX / 2;
  static constexpr int TPL = fft_tpl<N2>();                 // NX / 32 threads per row
  static constexpr int LS = fft_line_elems<N2>() + 4;
  static constexpr size_t SMEM = (size_t)LS * sizeof(cplx<T>);
};

// row y of the pair layouts: y = 4a + p (A) or 4a + p + 2 (B)
__device__ __forceinline__ void real_row_locate(int y, int& a, int& p, int& isB) { a = y >> 2; p = y & 1; isB = (y >> 1) & 1; }

// ---------------------------------------------------------------------------------------
// inverse row pass (C2R).  grid = (Ny rows, fields, members)
// ---------------------------------------------------------------------------------------
template <typename T, int NX>
__global__ void __launch_bounds__(RealRowCfg<T, NX>::TPL)
k_inv_row_real(const __grid_constant__ Geom g, const __grid_constant__ Batch batch, const cplx<T>* __restrict__ tabX,
               const cplx<T>* __restrict__ tabR, const double* __restrict__ v0_, size_t mstride) {
  using C = RealRowCfg<T, NX>;
  constexpr int N2 = C::N2, TPL = C::TPL;
  pdl_wait();
  pdl_trigger();     // as in k_inv_row / k_fwd_row (compiled out unless TTSH_PDL_TRIGGER = 1, ttsh_common.cuh)
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* line = reinterpret_cast<cplx<T>*>(smem_raw);
  const int j = threadIdx.x;
  int a, p, isB;
  real_row_locate(blockIdx.x, a, p, isB);
  const size_t moff = (size_t)blockIdx.z * mstride;
  FieldOp op = batch.f[blockIdx.y];
  op.src = static_cast<const char*>(op.src) + moff;
  op.dst = static_cast<char*>(op.dst) + moff;
  const double* __restrict__ v0 = reinterpret_cast<const double*>(reinterpret_cast<const char*>(v0_) + moff);
  const int Wx = g.Wx;
  // element of column mx of this row: (rp Wxp + mx) 2 + isB
  const cplx<T>* __restrict__ row = static_cast<const cplx<T>*>(op.src) + (size_t)(2 * a + p) * g.Wxp * 2 + isB;
  T* __restrict__ dst = static_cast<T*>(op.dst) + (size_t)blockIdx.x * NX;
  const int mode = op.mode & RM_MODE_MASK;
  const T scale = (T)g.inv_sqrt_nx;
  const T dkx = (T)g.dkx;
  const T meany = (mode == RM_NIKX_MEANY) ? (T)(v0[1] * g.inv_sqrt_ny) : (T)0;
  const cplx<T> wj = ldg_c(tabR + j);            // W_N^j

  // X'[mx] = multiplier(mx) X[mx]; Re[] of the oracle's complex iDFT drops the anti-Hermitian part at mx = 0
  auto xval = [&](cplx<T> w, int mx) -> cplx<T> {
    if (mode == RM_IKX) w = (dkx * (T)mx) * mul_i(w);
    else if (mode == RM_NIKX_MEANY) w = mx == 0 ? mk<T>(meany, (T)0) : (dkx * (T)mx) * mul_ni(w);
    if (mx == 0) w.y = 0;
    return w;
  };
  struct Raw { cplx<T> p, q; };
  auto issue = [&](int m, int) -> Raw {
    Raw r;
    r.p = m < Wx ? ldg_c(row + 2 * (size_t)m) : mk<T>(0, 0);
    r.q = (m > 0 && N2 - m < Wx) ? ldg_c(row + 2 * (size_t)(N2 - m)) : mk<T>(0, 0);
    return r;
  };
  auto finish = [&](int m, int k, Raw r) -> cplx<T> {
    const cplx<T> xp = m < Wx ? xval(r.p, m) : mk<T>(0, 0);
    const cplx<T> xq = (m > 0 && N2 - m < Wx) ? conj(xval(r.q, N2 - m)) : mk<T>(0, 0);
    const cplx<T> s = xp + xq, d = xp - xq;
    const cplx<T> t = mul_w32_rt<+1>(mul_conj(d, wj), k);        // conj(W_N^m) d,  m = j + k N/32
    return scale * (s + mul_i(t));
  };
  auto store = [&](int o, int, cplx<T> z) { *reinterpret_cast<cplx<T>*>(dst + 2 * (size_t)o) = z; };   // x[2o], x[2o+1]
  fft_line<T, N2, +1, false>(j, line, tabX, make_loader<2>(issue, finish), store);
}

// ---------------------------------------------------------------------------------------
// forward row pass (R2C).  grid = (Ny rows, fields, members)
// ---------------------------------------------------------------------------------------
template <typename T, int NX>
__global__ void __launch_bounds__(RealRowCfg<T, NX>::TPL)
k_fwd_row_real(const __grid_constant__ Geom g, const __grid_constant__ Batch batch, const cplx<T>* __restrict__ tabX,
               const cplx<T>* __restrict__ tabR, size_t mstride) {
  using C = RealRowCfg<T, NX>;
  constexpr int N2 = C::N2, TPL = C::TPL;
  pdl_wait();
  pdl_trigger();     // as in k_inv_row / k_fwd_row (compiled out unless TTSH_PDL_TRIGGER = 1, ttsh_common.cuh)
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* line = reinterpret_cast<cplx<T>*>(smem_raw);
  const int j = threadIdx.x;
  int a, p, isB;
  real_row_locate(blockIdx.x, a, p, isB);
  const size_t moff = (size_t)blockIdx.z * mstride;
  FieldOp op = batch.f[blockIdx.y];
  op.src = static_cast<const char*>(op.src) + moff;
  op.dst = static_cast<char*>(op.dst) + moff;
  const int Wx = g.Wx;
  const T* __restrict__ src = static_cast<const T*>(op.src) + (size_t)blockIdx.x * NX;
  cplx<T>* __restrict__ dst = static_cast<cplx<T>*>(op.dst) + isB;
  const T scale = (T)g.inv_sqrt_nx;
  const cplx<T> wj = ldg_c(tabR + j);            // W_N^j

  auto load = make_loader<1>([&](int n, int) -> cplx<T> { return ldg_c(reinterpret_cast<const cplx<T>*>(src + 2 * (size_t)n)); },
                             [&](int, int, cplx<T> raw) -> cplx<T> { return scale * raw; });
  auto store = [&](int m, int, cplx<T> z) { line[fft_pad<N2>(m)] = z; };
  fft_line<T, N2, -1, true>(j, line, tabX, load, store);
  __syncthreads();
  // X[mx] = E + W_N^mx O,  mx = j + i N/32 (i is uniform over the CTA: the constant W_32^i is selected without divergence)
  for (int i = 0, mx = j; mx < Wx; ++i, mx += TPL) {
    const cplx<T> zp = line[fft_pad<N2>(mx)];
    const cplx<T> zm = conj(line[fft_pad<N2>((N2 - mx) & (N2 - 1))]);
    const cplx<T> e = (T)0.5 * (zp + zm), o = (T)0.5 * mul_ni(zp - zm);
    dst[inter_pair_index(g, a, p, mx)] = e + mul_w32_rt<-1>(o * wj, i);
  }
}

}  // namespace ttsh
