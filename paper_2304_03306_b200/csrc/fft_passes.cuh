// fft_passes.cuh — the four passes of the pruned 2-D R2C / C2R transforms (PAPER.md:319 defines the DFT).
//
//   inverse:  pruned spectrum [Hy][Wxp] --inv_col--> intermediate [Ny][Wxp] --inv_row--> real [Ny][Nx]
//   forward:  real [Ny][Nx] --fwd_row--> intermediate [Ny][Wxp] --fwd_col--> pruned spectrum [Hy][Wxp]
//
// Row passes pack two real rows (y, y+1) of one field into one complex length-Nx FFT
// (z = row_y + i row_{y+1}); all global accesses are unit-stride in x.
// Column passes never hold a full column: because at most Ny/2+1 of the Ny y-wavenumbers are retained,
// the length-Ny transform is split by the parity p of y into two length-Ny/2 transforms
//   inverse:  f[2y'+p] = Ny^-1/2 sum_{m'} (X[m'] + (-1)^p X[m'+Ny/2]) W_Ny^{-p m'} W_{Ny/2}^{-m' y'}
//   forward:  X[m]     = Ny^-1/2 (E[m mod Ny/2] + W_Ny^m O[m mod Ny/2]),  E/O = FFT_{Ny/2} of the even/odd rows
// so a CTA needs only L * Ny/2 complex values of shared memory for L adjacent columns (L * 16 B or L * 8 B
// contiguous per row in HBM).  Multipliers (i k_y, 1/k^2, i k_x, the low-pass of Algorithm 2, the mean flow)
// are applied while loading, so the derivative fields never exist in spectral form in HBM.
#pragma once
#include "fft_core.cuh"
#ifndef TTSH_PF_DIST
#define TTSH_PF_DIST 296
#endif
#ifndef TTSH_ROW_MINB
#define TTSH_ROW_MINB 2
#endif
#ifndef TTSH_COL_ELEMS
#define TTSH_COL_ELEMS 4096
#endif

namespace ttsh {

// ---------------------------------------------------------------------------------------
// launch geometry
// ---------------------------------------------------------------------------------------
template <typename T, int NX> struct RowCfg {
  static constexpr int TPL = fft_tpl<NX>();
  static constexpr int L = (TPL >= 256) ? 1 : (TPL >= 128 ? 2 : 4);          // row pairs per CTA
  static constexpr int THREADS = L * TPL;
  static constexpr int LS = fft_line_elems<NX>() + 4;                          // line stride (elements)
  static constexpr size_t SMEM = (size_t)L * LS * sizeof(cplx<T>);
  static constexpr int MINB = THREADS <= 256 ? TTSH_ROW_MINB : 1;              // caps registers per thread
};
template <typename T, int NY> struct ColCfg {
  static constexpr int NH = NY / 2;
  static constexpr int TPL = fft_tpl<NH>();
  static constexpr int LMAX = sizeof(T) == 8 ? 8 : 8;
  static constexpr int LBUDGET = (int)(TTSH_COL_ELEMS * 16 / sizeof(cplx<T>)) / NH;     // keep L*NH*sizeof <= 64 KiB
  static constexpr int L = LBUDGET < 1 ? 1 : (LBUDGET > LMAX ? LMAX : LBUDGET); // adjacent columns per CTA
  static constexpr int THREADS = L * TPL;
  static constexpr int LS = fft_line_elems<NH>() + (sizeof(T) == 8 ? 8 / (L > 8 ? 8 : L) : 16 / (L > 16 ? 16 : L));
  static constexpr size_t SMEM = (size_t)L * LS * sizeof(cplx<T>);
  static constexpr int MINB = THREADS <= 256 ? 2 : 1;
};

// spectral multiplier of the inverse column pass (SpecMode), computed from integer wavenumber indices
template <typename T>
__device__ __forceinline__ cplx<T> apply_spec_mode(int mode, cplx<T> w, int mx, int my, const Geom& g, const double* v0) {
  if (mode == SM_ONE) return w;
  const T kx = (T)(g.dkx * mx), ky = (T)(g.dky * my);
  if (mode == SM_IKY) return ky * mul_i(w);
  if (mode == SM_LOWPASS4) return is_cut(mx, my, g.Nx, g.Ny, 1, 4) ? mk<T>(0, 0) : w;
  const bool zero = (mx == 0 && my == 0);
  const T ik2 = zero ? (T)0 : (T)1 / (kx * kx + ky * ky);
  if (mode == SM_PSI) return ik2 * w;
  /* SM_IKY_PSI_MEANX */
  if (zero) return mk<T>((T)v0[0], (T)0);
  return (ky * ik2) * mul_i(w);
}

// ---------------------------------------------------------------------------------------
// inverse column pass
// ---------------------------------------------------------------------------------------
template <typename T, int NY>
__global__ void __launch_bounds__(ColCfg<T, NY>::THREADS, ColCfg<T, NY>::MINB)
k_inv_col(const __grid_constant__ Geom g, const __grid_constant__ Batch batch, const cplx<T>* __restrict__ tabY,
          const cplx<T>* __restrict__ tabS, const double* __restrict__ v0) {
  using C = ColCfg<T, NY>;
  constexpr int NH = C::NH, L = C::L;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int c = threadIdx.x % L, j = threadIdx.x / L;
  const int mx = blockIdx.x * L + c;
  const bool valid = mx < g.Wx;
  const FieldOp op = batch.f[blockIdx.y];
  const cplx<T>* __restrict__ src = static_cast<const cplx<T>*>(op.src);
  cplx<T>* __restrict__ dst = static_cast<cplx<T>*>(op.dst);
  const int mode = op.mode;
  const T scale = (T)g.inv_sqrt_ny;
  const int My = g.My, Hy = g.Hy, Wxp = g.Wxp;
  cplx<T>* line = sm + c * C::LS;

#pragma unroll 1
  for (int p = 0; p < 2; ++p) {
    // a_p[mp] = (X[mp] + (-1)^p X[mp+NH]) W_Ny^{-p mp}; X[mp] is retained iff mp <= My, X[mp+NH] (my = mp-NH) iff
    // NH-mp <= My.  With the 1/2 rule both hold only at mp = NH/2, so one load per point is issued up front and the
    // rare second term is fetched in finish().
    auto issue = [&](int mp) -> cplx<T> {
      const bool use1 = mp <= My, use2 = NH - mp <= My;
      const int q = use1 ? mp : Hy + mp - NH;
      return (valid && (use1 || use2)) ? ld_l2_256(src + (size_t)q * Wxp + mx) : mk<T>(0, 0);
    };
    auto finish = [&](int mp, cplx<T> raw) -> cplx<T> {
      const bool use1 = mp <= My, use2 = NH - mp <= My;
      if (!valid || !(use1 || use2)) return mk<T>(0, 0);
      cplx<T> a = apply_spec_mode<T>(mode, raw, mx, use1 ? mp : mp - NH, g, v0);
      if (!use1 && p) a = mk<T>(-a.x, -a.y);
      if (use1 && use2) {
        const cplx<T> b = apply_spec_mode<T>(mode, src[(size_t)(Hy + mp - NH) * Wxp + mx], mx, mp - NH, g, v0);
        a = p ? a - b : a + b;
      }
      if (p) a = mul_conj(a, ldg_c(tabS + mp));   // * W_Ny^{-mp}  (inverse sign)
      return scale * a;
    };
    auto load = make_loader(issue, finish);
    auto store = [&](int yp, cplx<T> val) {
      if (valid) dst[(size_t)(2 * yp + p) * Wxp + mx] = val;
    };
    fft_line<T, NH, +1, false>(j, line, tabY, load, store);
  }
}

// ---------------------------------------------------------------------------------------
// forward column pass
// ---------------------------------------------------------------------------------------
template <typename T, int NY>
__global__ void __launch_bounds__(ColCfg<T, NY>::THREADS, ColCfg<T, NY>::MINB)
k_fwd_col(const __grid_constant__ Geom g, const __grid_constant__ Batch batch, const cplx<T>* __restrict__ tabY,
          const cplx<T>* __restrict__ tabS) {
  using C = ColCfg<T, NY>;
  constexpr int NH = C::NH, L = C::L;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int c = threadIdx.x % L, j = threadIdx.x / L;
  const int mx = blockIdx.x * L + c;
  const bool valid = mx < g.Wx;
  const FieldOp op = batch.f[blockIdx.y];
  const cplx<T>* __restrict__ src = static_cast<const cplx<T>*>(op.src);
  cplx<T>* dst = static_cast<cplx<T>*>(op.dst);
  const T scale = (T)g.inv_sqrt_ny;
  const int My = g.My, Hy = g.Hy, Wxp = g.Wxp;
  cplx<T>* line = sm + c * C::LS;

#pragma unroll 1
  for (int p = 0; p < 2; ++p) {
    auto load = make_loader(
        [&](int yp) -> cplx<T> { return valid ? ld_l2_256(src + (size_t)(2 * yp + p) * Wxp + mx) : mk<T>(0, 0); },
        [&](int, cplx<T> raw) -> cplx<T> { return scale * raw; });
    auto store = [&](int mp, cplx<T> val) {
      if (!valid) return;
      if (p == 0) {
        if (mp <= My) dst[(size_t)mp * Wxp + mx] = val;
        if (NH - mp <= My) dst[(size_t)(Hy + mp - NH) * Wxp + mx] = val;
      } else {
        const cplx<T> t = val * ldg_c(tabS + mp);                 // W_Ny^{mp} O[mp];  W_Ny^{mp+NH} = -W_Ny^{mp}
        // fire-and-forget reductions instead of read-modify-write: no L2 round trip on the critical path
        if (mp <= My) red_add(dst + (size_t)mp * Wxp + mx, t);
        if (NH - mp <= My) red_add(dst + (size_t)(Hy + mp - NH) * Wxp + mx, mk<T>(-t.x, -t.y));
      }
    };
    fft_line<T, NH, -1, false>(j, line, tabY, load, store);
  }
}

// ---------------------------------------------------------------------------------------
// inverse row pass (C2R, two rows per complex transform)
// ---------------------------------------------------------------------------------------
template <typename T, int NX>
__global__ void __launch_bounds__(RowCfg<T, NX>::THREADS, RowCfg<T, NX>::MINB)
k_inv_row(const __grid_constant__ Geom g, const __grid_constant__ Batch batch, const cplx<T>* __restrict__ tabX, const double* __restrict__ v0) {
  using C = RowCfg<T, NX>;
  constexpr int TPL = C::TPL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int c = threadIdx.x / TPL, j = threadIdx.x % TPL;
  const int rp = blockIdx.x * C::L + c;             // row pair; Ny/2 is a multiple of L
  const FieldOp op = batch.f[blockIdx.y];
  const int Wx = g.Wx, Wxp = g.Wxp;
  const cplx<T>* __restrict__ srcA = static_cast<const cplx<T>*>(op.src) + (size_t)(2 * rp) * Wxp;
  const cplx<T>* __restrict__ srcB = srcA + Wxp;
  T* __restrict__ dstA = static_cast<T*>(op.dst) + (size_t)(2 * rp) * NX;
  T* __restrict__ dstB = dstA + NX;
  const int mode = op.mode;
  const T scale = (T)g.inv_sqrt_nx;
  const T dkx = (T)g.dkx;
  const T meany = (mode == RM_NIKX_MEANY) ? (T)(v0[1] * g.inv_sqrt_ny) : (T)0;
  if (threadIdx.x == 0) {
    int nb = blockIdx.x + TTSH_PF_DIST, ny = blockIdx.y;
    if (nb >= (int)gridDim.x) { nb -= gridDim.x; ny += 1; }
    if (ny < (int)gridDim.y && nb < (int)gridDim.x)
      prefetch_l2_bulk(static_cast<const cplx<T>*>(batch.f[ny].src) + (size_t)(2 * nb * C::L) * Wxp,
                       2 * C::L * Wxp * sizeof(cplx<T>));
  }

  auto mult = [&](cplx<T> a, int mx) -> cplx<T> {
    if (mode == RM_ONE) return a;
    const T kx = dkx * (T)mx;
    if (mode == RM_IKX) return kx * mul_i(a);
    return mx == 0 ? mk<T>(meany, (T)0) : kx * mul_ni(a);        // RM_NIKX_MEANY
  };
  struct RawAB { cplx<T> a, b; };
  auto issue = [&](int m) -> RawAB {
    const int mx = m > NX / 2 ? NX - m : m;
    RawAB r;
    r.a = mk<T>(0, 0); r.b = mk<T>(0, 0);
    if (mx < Wx) { r.a = srcA[mx]; r.b = srcB[mx]; }
    return r;
  };
  auto finish = [&](int m, RawAB r) -> cplx<T> {
    // Z(m) = A(m) + i B(m) with A, B the Hermitian x-spectra of the two real rows
    const bool neg = m > NX / 2;
    const int mx = neg ? NX - m : m;
    if (mx >= Wx) return mk<T>(0, 0);
    cplx<T> a = mult(r.a, mx), b = mult(r.b, mx);
    if (mx == 0) { a.y = 0; b.y = 0; }             // Re[] of the oracle's complex iDFT: drop the anti-Hermitian part
    if (neg) { a = conj(a); b = conj(b); }
    return scale * mk<T>(a.x - b.y, a.y + b.x);
  };
  auto load = make_loader(issue, finish);
  auto store = [&](int x, cplx<T> z) {
    dstA[x] = z.x;
    dstB[x] = z.y;
  };
  fft_line<T, NX, +1, false>(j, sm + c * C::LS, tabX, load, store);
}

// ---------------------------------------------------------------------------------------
// forward row pass (R2C, two rows per complex transform)
// ---------------------------------------------------------------------------------------
template <typename T, int NX>
__global__ void __launch_bounds__(RowCfg<T, NX>::THREADS, RowCfg<T, NX>::MINB)
k_fwd_row(const __grid_constant__ Geom g, const __grid_constant__ Batch batch, const cplx<T>* __restrict__ tabX) {
  using C = RowCfg<T, NX>;
  constexpr int TPL = C::TPL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int c = threadIdx.x / TPL, j = threadIdx.x % TPL;
  const int rp = blockIdx.x * C::L + c;
  const FieldOp op = batch.f[blockIdx.y];
  const int Wx = g.Wx, Wxp = g.Wxp;
  const T* __restrict__ srcA = static_cast<const T*>(op.src) + (size_t)(2 * rp) * NX;
  const T* __restrict__ srcB = srcA + NX;
  cplx<T>* __restrict__ dstA = static_cast<cplx<T>*>(op.dst) + (size_t)(2 * rp) * Wxp;
  cplx<T>* __restrict__ dstB = dstA + Wxp;
  const T scale = (T)g.inv_sqrt_nx;
  cplx<T>* line = sm + c * C::LS;
  if (threadIdx.x == 0) {   // L2 prefetch for the CTA that runs ~one wave later (C::L row pairs = 2 L contiguous rows)
    int nb = blockIdx.x + TTSH_PF_DIST, ny = blockIdx.y;
    if (nb >= (int)gridDim.x) { nb -= gridDim.x; ny += 1; }
    if (ny < (int)gridDim.y && nb < (int)gridDim.x)
      prefetch_l2_bulk(static_cast<const T*>(batch.f[ny].src) + (size_t)(2 * nb * C::L) * NX, 2 * C::L * NX * sizeof(T));
  }

  auto load = make_loader([&](int x) -> cplx<T> { return mk<T>(srcA[x], srcB[x]); },
                          [&](int, cplx<T> raw) -> cplx<T> { return scale * raw; });
  auto store = [&](int m, cplx<T> z) { line[fft_pad<NX>(m)] = z; };
  fft_line<T, NX, -1, true>(j, line, tabX, load, store);
  __syncthreads();
  // unpack: A(m) = (Z(m) + conj Z(-m))/2,  B(m) = -i (Z(m) - conj Z(-m))/2,  m = 0..Wx-1
  for (int mx = j; mx < Wx; mx += TPL) {
    const cplx<T> zp = line[fft_pad<NX>(mx)];
    const cplx<T> zm = conj(line[fft_pad<NX>((NX - mx) & (NX - 1))]);
    dstA[mx] = (T)0.5 * (zp + zm);
    dstB[mx] = (T)0.5 * mul_ni(zp - zm);
  }
}

}  // namespace ttsh
