// fft_passes.cuh — the four passes of the pruned 2-D R2C / C2R transforms (PAPER.md:319 defines the DFT).
//
//   inverse:  pruned spectrum --k_inv_col--> intermediate --k_inv_row--> real [Ny][Nx]
//   forward:  real [Ny][Nx] --k_fwd_row--> intermediate --k_fwd_col--> pruned spectrum
//   (tile-major layouts of the two complex arrays: ttsh_common.cuh)
//
// Row passes pack two real rows of one field (same parity: y = 4a+p and 4a+p+2) into one complex length-Nx FFT
// (z = row_A + i row_B); the real side is unit-stride, the intermediate side moves (A, B) pairs with one
// 32-byte (fp64, LDG.256/STG.256) or 16-byte (fp32) access per thread, 2 CW elements contiguous per tile.
// Column passes never hold a full column: because at most Ny/2+1 of the Ny y-wavenumbers are retained,
// the length-Ny transform is split by the parity p of y into two length-Ny/2 transforms
//   inverse:  f[2y'+p] = Ny^-1/2 sum_{m'} (X[m'] + (-1)^p X[m'+Ny/2]) W_Ny^{-p m'} W_{Ny/2}^{-m' y'}
//   forward:  X[m]     = Ny^-1/2 (E[m mod Ny/2] + W_Ny^m O[m mod Ny/2]),  E/O = FFT_{Ny/2} of the even/odd rows
// so a CTA needs CW * Ny/2 complex values of shared memory for its CW adjacent columns, and — the arrays being
// tile-major — every global access of a column CTA is `base + threadIdx.x + r * blockDim.x`: fully coalesced.
// Multipliers (i k_y, 1/k^2, i k_x, the low-pass of Algorithm 2, the mean flow) are applied while loading, so the
// derivative fields never exist in spectral form in HBM.
#pragma once
#include "fft_core.cuh"
#ifndef TTSH_PF_DIST
#define TTSH_PF_DIST 296
#endif
#ifndef TTSH_PF_DIST_FUSED
#define TTSH_PF_DIST_FUSED 64
#endif
#ifndef TTSH_PF_DIST_COL
#define TTSH_PF_DIST_COL 148
#endif
#ifndef TTSH_ROW_MINB
#define TTSH_ROW_MINB 2
#endif
#ifndef TTSH_COL_BYTES
#define TTSH_COL_BYTES 65536
#endif

namespace ttsh {

// ---------------------------------------------------------------------------------------
// launch geometry
// ---------------------------------------------------------------------------------------
template <typename T, int NX> struct RowCfg {
  static constexpr int TPL = fft_tpl<NX>();
  static constexpr int L = (TPL >= 256) ? 1 : (TPL >= 64 ? 2 : 4);           // row pairs per CTA
  static constexpr int THREADS = L * TPL;
  static constexpr int LS = fft_line_elems<NX>() + 4;                          // line stride (elements)
  static constexpr size_t SMEM = (size_t)L * LS * sizeof(cplx<T>);
  static constexpr int MINB = THREADS <= 256 ? TTSH_ROW_MINB : 1;              // caps registers per thread
};
// columns per CTA of the column pass = tile width CW of the two complex arrays: CW * Ny/2 complex values near 64 KiB
// of shared memory (fp64 4096: 2 columns, fp32 4096: 4), at least 2 and at most 8 columns (1 at Ny = 16384)
__host__ __device__ constexpr int col_tile_width(int Ny, int elem_bytes) {
  if (Ny >= 16384) return 1;      // 8192-point half-length transforms: one column per CTA (128 KB in fp64)
  int cw = (TTSH_COL_BYTES / elem_bytes) / (Ny / 2);
#ifndef TTSH_COL_CAP_SMALL
#define TTSH_COL_CAP_SMALL 4
#endif
  // small grids: more, smaller CTAs (the GPU has 148 SMs to fill, and the fused column kernel of col_step.cuh runs ONE CTA per tile
  // with six transform groups): two columns at Ny = 1024, one below (measured with k_col_step, fp64 step: 1024^2 32.4 us with
  // two columns, 37.1 with one; 512^2 18.7 with one, 24.3 with four; 256^2 16.4 / 18.8; 128^2 15.2 / 16.8)
  if (Ny >= 128 && Ny <= 512) return 1;
  const int cap = Ny >= 2048 ? 8 : (Ny == 1024 ? 2 : TTSH_COL_CAP_SMALL);      // Ny = 64 (four launches per step): four columns
  // Ny = 8192 in fp64: one 4096-point column (64 KB) per 256-thread CTA, two CTAs per SM, instead of two columns in one 512-thread CTA
  // per SM (8192^2: k_inv_col 437 -> 349 us, k_fwd_col 289 -> 237 us; k_row_step_real writes whole 32-byte pairs and pays 34 us)
  if (cw < 2) return Ny >= 8192 ? 1 : 2;
  return cw > cap ? cap : cw;
}
template <typename T, int NY> struct ColCfg {
  static constexpr int NH = NY / 2;
  static constexpr int TPL = fft_tpl<NH>();
  static constexpr int L = col_tile_width(NY, (int)sizeof(cplx<T>));
  static constexpr int LSHIFT = L == 1 ? 0 : (L == 2 ? 1 : (L == 4 ? 2 : 3));
  static constexpr int THREADS = L * TPL;
  // line stride: a 128-byte wavefront holds W = 128 / sizeof(cplx<T>) elements and is filled by W threads = W/L consecutive
  // butterflies x L lines (col_thread_map), so the lines must start W/L elements apart modulo W to land in distinct banks
  static constexpr int LS = fft_line_elems<NH>() + (128 / (int)sizeof(cplx<T>)) / L;
  static constexpr size_t SMEM = (size_t)L * LS * sizeof(cplx<T>);
  static constexpr int MINB = (THREADS <= 256 || sizeof(T) == 4) ? 2 : 1;    // fp32: 512 threads x 64 registers
  // small Ny: a transform has few threads (Ny = 64: 8), so a CTA of the kernels' G > 1 variant runs G independent work items
  // (tile x field x member) side by side, each with its own line buffers (ensembles; a single small system keeps G = 1:
  // more, smaller CTAs spread over more SMs)
  static constexpr int GMAX = THREADS >= 128 ? 1 : 128 / THREADS;   // used when the launch has enough items to fill the GPU anyway
};

// 2-element (A, B) pair access of the row passes
template <typename T> struct Pair { cplx<T> a, b; };
__device__ __forceinline__ Pair<double> ld_pair(const cplx<double>* p) {
  Pair<double> r;
  asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.a.x), "=d"(r.a.y), "=d"(r.b.x), "=d"(r.b.y) : "l"(p));
  return r;
}
__device__ __forceinline__ Pair<float> ld_pair(const cplx<float>* p) {
  Pair<float> r;
  asm volatile("ld.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.a.x), "=f"(r.a.y), "=f"(r.b.x), "=f"(r.b.y) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_pair(cplx<double>* p, cplx<double> a, cplx<double> b) {
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(a.x), "d"(a.y), "d"(b.x), "d"(b.y));
}
__device__ __forceinline__ void st_pair(cplx<float>* p, cplx<float> a, cplx<float> b) {
  asm volatile("st.global.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
}

// one complex value (one row's half of a pair)
__device__ __forceinline__ cplx<double> ld_c(const cplx<double>* p) {
  cplx<double> r;
  asm volatile("ld.global.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
  return r;
}
__device__ __forceinline__ cplx<float> ld_c(const cplx<float>* p) {
  cplx<float> r;
  asm volatile("ld.global.v2.f32 {%0, %1}, [%2];" : "=f"(r.x), "=f"(r.y) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_c(cplx<double>* p, cplx<double> a) {
  asm volatile("st.global.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(a.x), "d"(a.y));
}
__device__ __forceinline__ void st_c(cplx<float>* p, cplx<float> a) {
  asm volatile("st.global.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a.x), "f"(a.y));
}

// 4 consecutive scalars of a (permuted) real row: one 32-byte (fp64) / 16-byte (fp32) access
template <typename T> struct Quad { T v[4]; };
__device__ __forceinline__ Quad<double> ld_quad(const double* p) {
  Quad<double> r;
  asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.v[0]), "=d"(r.v[1]), "=d"(r.v[2]), "=d"(r.v[3]) : "l"(p));
  return r;
}
__device__ __forceinline__ Quad<float> ld_quad(const float* p) {
  Quad<float> r;
  asm volatile("ld.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_quad(double* p, double a, double b, double c, double d) {
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d));
}
__device__ __forceinline__ void st_quad(float* p, float a, float b, float c, float d) {
  asm volatile("st.global.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d));
}

// spectral multiplier of the inverse column pass (SpecMode).  mode is uniform per CTA.  No division: psi^ = w^/k^2 is kept
// as a second spectrum by the spectral kernel (line 13 of Algorithm 1 is evaluated once per mode there).
template <typename T>
__device__ __forceinline__ cplx<T> apply_spec_mode(int mode, cplx<T> w, int mx, int my, const Geom& g, const double* v0) {
  if (mode == SM_ONE) return w;
  if (mode == SM_LOWPASS4) return is_cut(g, mx, my, 1, 4) ? mk<T>(0, 0) : w;
  const T ky = (T)g.dky * (T)my;
  if (mode == SM_IKY_MEANX && mx == 0 && my == 0) return mk<T>((T)v0[0], (T)0);
  return ky * mul_i(w);
}

// thread -> (FFT index j, column c) of a column CTA: threadIdx.x enumerates the intermediate block [Ny/4][CW][2] in
// memory order, e = (a CW + c) 2 + b, j = 2a + b, so that element y' = j + r TPL of column c is at e + r blockDim.x.
template <int LSHIFT> __device__ __forceinline__ void col_thread_map(int e, int& j, int& c) {
  c = (e >> 1) & ((1 << LSHIFT) - 1);
  j = ((e >> (1 + LSHIFT)) << 1) | (e & 1);
}

// ---------------------------------------------------------------------------------------
// inverse column pass.  grid = (2 parities, NT tiles, fields): one half-length transform per CTA (both read the same
// 64 KB spectrum tile - adjacent in launch order, so the second read hits L2; splitting them doubles the number of CTAs
// and halves the tail of the last wave)
// ---------------------------------------------------------------------------------------
template <typename T, int NY, int G>
__global__ void __launch_bounds__(G * ColCfg<T, NY>::THREADS, ColCfg<T, NY>::MINB)
k_inv_col(const __grid_constant__ Geom g, const __grid_constant__ Batch batch, const cplx<T>* __restrict__ tabY,
          const cplx<T>* __restrict__ tabS, const double* __restrict__ v0_, int nf, int nmembers, size_t mstride) {
  using C = ColCfg<T, NY>;
  constexpr int NH = C::NH, L = C::L, TPL = C::TPL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  // grid = (2 parities, ceil(items / G)); item = tile + NT * (field + nf * member), G items per CTA
  const int sub = G == 1 ? 0 : (int)threadIdx.x / C::THREADS, tid = G == 1 ? (int)threadIdx.x : (int)threadIdx.x % C::THREADS;
  int j, c;
  col_thread_map<C::LSHIFT>(tid, j, c);
  const int nitems = g.NT * nf * nmembers;
  int item = blockIdx.y * G + sub;
  const bool live = G == 1 || item < nitems;   // an idle group of the last CTA still takes part in the barriers
  if (!live) item = nitems - 1;
  const int t = item % g.NT, zf = item / g.NT;
  const int mx = t * L + c;
  const bool valid = live && mx < g.Wx;
  const int member = zf / nf;                      // member 0 only outside ensembles
  const size_t moff = (size_t)member * mstride;    // bytes
  FieldOp op = batch.f[zf - member * nf];
  op.src = static_cast<const char*>(op.src) + moff;
  op.dst = static_cast<char*>(op.dst) + moff;
  const double* __restrict__ v0 = reinterpret_cast<const double*>(reinterpret_cast<const char*>(v0_) + moff);
  const int My = g.My, Hy = g.Hy;
  const cplx<T>* __restrict__ src = static_cast<const cplx<T>*>(op.src) + (size_t)t * Hy * L + c;   // (q, c) at q L
  // inverse intermediate is pair-row-major: row y = 2y'+p of column mx at ((2 (y'>>1) + p) Wxp + mx) 2 + (y'&1);
  // y' = j + k TPL keeps the parity of j, so slot k adds k TPL Wxp 2 elements
  cplx<T>* __restrict__ dst = static_cast<cplx<T>*>(op.dst) + ((size_t)(j & ~1) * g.Wxp + mx) * 2 + (j & 1);
  const size_t slot_stride = (size_t)TPL * g.Wxp * 2;
  const int mode = op.mode;
  const T scale = (T)g.inv_sqrt_ny;
  cplx<T>* line = sm + (sub * L + c) * C::LS;

  const bool half_rule = (2 * My == NH);     // the paper's 1/2 rule: |my| <= Ny/4 (uniform branch)
  const cplx<T> wj = ldg_c(tabS + j);         // W_Ny^j
  // L2 prefetch of the spectrum tile the CTAs about one wave later read (bulk prefetch: 16-byte granules, so not for the
  // one-column fp32 tiles of Ny = 16384, whose rows are 8 bytes)
  if ((L * sizeof(cplx<T>)) % 16 == 0 && G == 1 && threadIdx.x == 0 && blockIdx.x == 0) {
    const int ni = item + TTSH_PF_DIST_COL;
    if (ni < nitems) {
      const int nt = ni % g.NT, nz = ni / g.NT;
      prefetch_l2_bulk(reinterpret_cast<const cplx<T>*>(static_cast<const char*>(batch.f[nz % nf].src) + (size_t)(nz / nf) * mstride) +
                           (size_t)nt * Hy * L, (unsigned)(Hy * L * sizeof(cplx<T>)));
    }
  }

  pdl_wait();        // everything above touches only tables and addresses; the spectra below are the predecessor's output
  pdl_trigger();
  {
    const int p = blockIdx.x;
    // a_p[mp] = (X[mp] + (-1)^p X[mp+NH]) W_Ny^{-p mp}; X[mp] is retained iff mp <= My, X[mp+NH] (my = mp-NH) iff
    // NH-mp <= My.
    // tail columns of the last tile are written too (zeros inside the row pitch), the row pass never reads them
    cplx<T>* out = dst + (size_t)p * g.Wxp * 2;
    auto store = [&](int, int k, cplx<T> val) { if (live) out[(size_t)k * slot_stride] = val; };
    // * W_Ny^{-mp} (inverse sign) for the odd rows; mp = j + k TPL, so W_Ny^{mp} = W_Ny^j W_32^k: one table load per thread
    auto twist = [&](int k, cplx<T> a) -> cplx<T> {
      if (p) a = mul_w32_rt<+1>(mul_conj(a, wj), k);
      return scale * a;
    };
    if (half_rule) {
      // My = NH/2 = 8 TPL: slot k < 8 holds X[mp] only, k > 8 holds X[mp+NH] only, k = 8 holds X[mp+NH] plus, for the
      // single point mp = NH/2 (j = 0), X[NH/2]: the selection is a compile-time function of the slot.
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
    } else {
      // general dealias fraction: one load per point up front, the (possibly common) second term in finish()
      auto issue = [&](int mp, int) -> cplx<T> {
        const bool use1 = mp <= My, use2 = NH - mp <= My;
        const int q = use1 ? mp : Hy + mp - NH;
        return (valid && (use1 || use2)) ? src[(size_t)q * L] : mk<T>(0, 0);
      };
      auto finish = [&](int mp, int k, cplx<T> raw) -> cplx<T> {
        const bool use1 = mp <= My, use2 = NH - mp <= My;
        if (!valid || !(use1 || use2)) return mk<T>(0, 0);
        cplx<T> v = apply_spec_mode<T>(mode, raw, mx, use1 ? mp : mp - NH, g, v0);
        if (!use1 && p) v = mk<T>(-v.x, -v.y);
        if (use1 && use2) {
          const cplx<T> b = apply_spec_mode<T>(mode, src[(size_t)(Hy + mp - NH) * L], mx, mp - NH, g, v0);
          v = p ? v - b : v + b;
        }
        return twist(k, v);
      };
      fft_line<T, NH, +1, false>(j, line, tabY, make_loader(issue, finish), store);
    }
  }
}

// ---------------------------------------------------------------------------------------
// forward column pass.  grid = (NT tiles, fields)
// ---------------------------------------------------------------------------------------
template <typename T, int NY, int G>
__global__ void __launch_bounds__(G * ColCfg<T, NY>::THREADS, ColCfg<T, NY>::MINB)
k_fwd_col(const __grid_constant__ Geom g, const __grid_constant__ Batch batch, const cplx<T>* __restrict__ tabY,
          const cplx<T>* __restrict__ tabS, int nf, int nmembers, size_t mstride) {
  using C = ColCfg<T, NY>;
  constexpr int NH = C::NH, L = C::L, TPL = C::TPL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  // grid = ceil(items / G); item = tile + NT * (field + nf * member), G items per CTA
  const int sub = G == 1 ? 0 : (int)threadIdx.x / C::THREADS, tid = G == 1 ? (int)threadIdx.x : (int)threadIdx.x % C::THREADS;
  int j, c;
  col_thread_map<C::LSHIFT>(tid, j, c);
  const int nitems = g.NT * nf * nmembers;
  int item = blockIdx.x * G + sub;
  const bool live = G == 1 || item < nitems;
  if (!live) item = nitems - 1;
  const int t = item % g.NT, zf = item / g.NT;
  const bool valid = live && t * L + c < g.Wx;
  const int member = zf / nf;
  const size_t moff = (size_t)member * mstride;
  FieldOp op = batch.f[zf - member * nf];
  op.src = static_cast<const char*>(op.src) + moff;
  op.dst = static_cast<char*>(op.dst) + moff;
  const int My = g.My, Hy = g.Hy;
  const cplx<T>* __restrict__ src = static_cast<const cplx<T>*>(op.src) + (size_t)t * 2 * NH * L + tid;
  cplx<T>* dst = static_cast<cplx<T>*>(op.dst) + (size_t)t * Hy * L + c;
  const T scale = (T)g.inv_sqrt_ny;
  cplx<T>* line = sm + (sub * L + c) * C::LS;
  const cplx<T> wj = ldg_c(tabS + j);         // W_Ny^j

  const bool half_rule = (2 * My == NH);
  // output rows: X[mp] (my = mp >= 0) at row mp, X[mp+NH] (my = mp-NH < 0) at row Hy+mp-NH; mp = j + k TPL
  cplx<T>* dpos = dst + (size_t)j * L;
  cplx<T>* dneg = dst + (size_t)(Hy - NH + j) * L;
  constexpr size_t KS = (size_t)TPL * L;     // elements per slot

  pdl_wait();
  pdl_trigger();
#pragma unroll 1
  for (int p = 0; p < 2; ++p) {
    const cplx<T>* in = src + (size_t)p * NH * L;
    auto load = make_loader(
        [&](int, int k) -> cplx<T> { return valid ? in[(size_t)k * (L * TPL)] : mk<T>(0, 0); },
        [&](int, int, cplx<T> raw) -> cplx<T> { return scale * raw; });
    // pass 0 stores E; pass 1 accumulates W_Ny^{mp} O[mp] = W_Ny^j W_32^k O (one table load per thread; W_Ny^{mp+NH} =
    // -W_Ny^{mp}) with fire-and-forget reductions instead of a read-modify-write.
    if (half_rule) {
      // My = NH/2 = 8 TPL: slot k < 8 -> row mp only, k > 8 -> row Hy+mp-NH only, k = 8 -> the latter plus, for j = 0, row NH/2
      if (p == 0) {
        auto store = [&](int, int k, cplx<T> val) {
          if (!valid) return;
          if (k < 8 || (k == 8 && j == 0)) dpos[k * KS] = val;
          if (k >= 8) dneg[k * KS] = val;
        };
        fft_line<T, NH, -1, false>(j, line, tabY, load, store);
      } else {
        auto store = [&](int, int k, cplx<T> val) {
          if (!valid) return;
          const cplx<T> tw = mul_w32_rt<-1>(val * wj, k);
          if (k < 8 || (k == 8 && j == 0)) red_add(dpos + k * KS, tw);
          if (k >= 8) red_add(dneg + k * KS, mk<T>(-tw.x, -tw.y));
        };
        fft_line<T, NH, -1, false>(j, line, tabY, load, store);
      }
    } else {
      auto store = [&](int mp, int k, cplx<T> val) {
        if (!valid) return;
        if (p == 0) {
          if (mp <= My) dpos[k * KS] = val;
          if (NH - mp <= My) dneg[k * KS] = val;
        } else {
          const cplx<T> tw = mul_w32_rt<-1>(val * wj, k);
          if (mp <= My) red_add(dpos + k * KS, tw);
          if (NH - mp <= My) red_add(dneg + k * KS, mk<T>(-tw.x, -tw.y));
        }
      };
      fft_line<T, NH, -1, false>(j, line, tabY, load, store);
    }
  }
}

// ---------------------------------------------------------------------------------------
// inverse row pass (C2R, two rows per complex transform).  grid = (Ny/2 / L row pairs, fields)
// ---------------------------------------------------------------------------------------
template <typename T, int NX>
__global__ void __launch_bounds__(RowCfg<T, NX>::THREADS, RowCfg<T, NX>::MINB)
k_inv_row(const __grid_constant__ Geom g, const __grid_constant__ Batch batch, const cplx<T>* __restrict__ tabX,
          const double* __restrict__ v0_, size_t mstride) {
  using C = RowCfg<T, NX>;
  pdl_wait();      // launched with programmatic dependent launch: inputs and v0 come from the preceding kernels
  constexpr int TPL = C::TPL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int c = threadIdx.x / TPL, j = threadIdx.x % TPL;
  const int rp = blockIdx.x * C::L + c;             // row pair: rows yA = 4a+p, yB = yA+2; Ny/2 is a multiple of L
  const int a = rp >> 1, p = rp & 1;
  const size_t moff = (size_t)blockIdx.z * mstride;     // grid.z = member (tangent vectors at a uniform stride); 0 otherwise
  FieldOp op = batch.f[blockIdx.y];
  op.src = static_cast<const char*>(op.src) + moff;
  op.dst = static_cast<char*>(op.dst) + moff;
  const double* __restrict__ v0 = reinterpret_cast<const double*>(reinterpret_cast<const char*>(v0_) + moff);
  const int Wx = g.Wx;
  const cplx<T>* __restrict__ src = static_cast<const cplx<T>*>(op.src);
  T* __restrict__ dstA = static_cast<T*>(op.dst) + (size_t)(4 * a + p) * NX;
  T* __restrict__ dstB = dstA + 2 * NX;
  const int mode = op.mode & RM_MODE_MASK;
  const T scale = (T)g.inv_sqrt_nx;
  const T dkx = (T)g.dkx;
  const T meany = (mode == RM_NIKX_MEANY) ? (T)(v0[1] * g.inv_sqrt_ny) : (T)0;

  auto mult = [&](cplx<T> w, int mx) -> cplx<T> {
    if (mode == RM_ONE) return w;
    const T kx = dkx * (T)mx;
    if (mode == RM_IKX) return kx * mul_i(w);
    return mx == 0 ? mk<T>(meany, (T)0) : kx * mul_ni(w);        // RM_NIKX_MEANY
  };
  const cplx<T>* __restrict__ row = src + (size_t)rp * g.Wxp * 2;        // (A, B) pair of column mx at row + 2 mx
  if (threadIdx.x == 0) {   // L2 prefetch of the contiguous input of the CTA that runs about one wave later
    int nb = blockIdx.x + TTSH_PF_DIST, ny = blockIdx.y;
    if (nb >= (int)gridDim.x) { nb -= gridDim.x; ny += 1; }
    if (ny < (int)gridDim.y)
      prefetch_l2_bulk(reinterpret_cast<const cplx<T>*>(static_cast<const char*>(batch.f[ny].src) + moff) + (size_t)nb * C::L * g.Wxp * 2,
                       (unsigned)(C::L * g.Wxp * 2 * sizeof(cplx<T>)));
  }
  auto zero_pair = [&]() -> Pair<T> { Pair<T> r; r.a = mk<T>(0, 0); r.b = mk<T>(0, 0); return r; };
  // Z(m) = A(m) + i B(m) with A, B the Hermitian x-spectra of the two real rows; neg: m stands for -mx
  auto combine = [&](Pair<T> r, int mx, bool neg) -> cplx<T> {
    cplx<T> wa = mult(r.a, mx), wb = mult(r.b, mx);
    if (mx == 0) { wa.y = 0; wb.y = 0; }           // Re[] of the oracle's complex iDFT: drop the anti-Hermitian part
    if (neg) { wa = conj(wa); wb = conj(wb); }
    return scale * mk<T>(wa.x - wb.y, wa.y + wb.x);
  };
  // output rows: natural order (caller-owned buffers) or the permuted internal layout (perm_index, fft_core.cuh): the
  // 4 slots k0..k0+3 of this thread are then 4 consecutive scalars -> one wide store per row
  const bool perm = (op.mode & RM_PERM) != 0;
  auto store = make_vec_store([&](int k0, const cplx<T>* z) {
    if (perm) {
      const size_t e = ((size_t)(k0 >> 2) * TPL + j) * 4;
      st_quad(dstA + e, z[0].x, z[1].x, z[2].x, z[3].x);
      st_quad(dstB + e, z[0].y, z[1].y, z[2].y, z[3].y);
    } else {
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        dstA[j + (k0 + i) * TPL] = z[i].x;
        dstB[j + (k0 + i) * TPL] = z[i].y;
      }
    }
  });
  if (4 * (Wx - 1) == NX) {
    // the paper's 1/2 rule: retained mx = 0..NX/4 = 4 TPL.  Input slot k (m = j + k TPL): k <= 3 holds +mx = m, k = 4 only
    // the single point m = NX/4 (j = 0), k = 5..11 nothing, k = 12..15 holds -mx with mx = NX - m: compile-time pruning.
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
    fft_line<T, NX, +1, false>(j, sm + c * C::LS, tabX, make_loader<2>(issue, finish), store);
  } else {
    auto issue = [&](int m, int) -> Pair<T> {
      const int mx = m > NX / 2 ? NX - m : m;
      return mx < Wx ? ld_pair(row + 2 * mx) : zero_pair();
    };
    auto finish = [&](int m, int, Pair<T> r) -> cplx<T> {
      const bool neg = m > NX / 2;
      const int mx = neg ? NX - m : m;
      return mx < Wx ? combine(r, mx, neg) : mk<T>(0, 0);
    };
    fft_line<T, NX, +1, false>(j, sm + c * C::LS, tabX, make_loader<2>(issue, finish), store);
  }
}

// ---------------------------------------------------------------------------------------
// forward row pass (R2C, two rows per complex transform).  grid = (Ny/2 / L row pairs, fields)
// ---------------------------------------------------------------------------------------
template <typename T, int NX>
__global__ void __launch_bounds__(RowCfg<T, NX>::THREADS, RowCfg<T, NX>::MINB)
k_fwd_row(const __grid_constant__ Geom g, const __grid_constant__ Batch batch, const cplx<T>* __restrict__ tabX, size_t mstride) {
  using C = RowCfg<T, NX>;
  pdl_wait();
  constexpr int TPL = C::TPL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int c = threadIdx.x / TPL, j = threadIdx.x % TPL;
  const int rp = blockIdx.x * C::L + c;
  const int a = rp >> 1, p = rp & 1;
  const size_t moff = (size_t)blockIdx.z * mstride;     // grid.z = member
  FieldOp op = batch.f[blockIdx.y];
  op.src = static_cast<const char*>(op.src) + moff;
  op.dst = static_cast<char*>(op.dst) + moff;
  const int Wx = g.Wx;
  const T* __restrict__ srcA = static_cast<const T*>(op.src) + (size_t)(4 * a + p) * NX;
  const T* __restrict__ srcB = srcA + 2 * NX;
  cplx<T>* __restrict__ dst = static_cast<cplx<T>*>(op.dst);
  const T scale = (T)g.inv_sqrt_nx;
  cplx<T>* line = sm + c * C::LS;
  if (threadIdx.x == 0) {   // L2 prefetch of the rows of the CTA pair that runs about one wave later (4 consecutive rows)
    int nb = blockIdx.x + TTSH_PF_DIST, ny = blockIdx.y;
    if (nb >= (int)gridDim.x) { nb -= gridDim.x; ny += 1; }
    if (ny < (int)gridDim.y && ((nb * C::L) & 1) == 0)
      prefetch_l2_bulk(reinterpret_cast<const T*>(static_cast<const char*>(batch.f[ny].src) + moff) + (size_t)(2 * nb * C::L) * NX,
                       (C::L >= 2 ? 2 * C::L : 4) * NX * sizeof(T));
  }

  const bool perm = (op.mode & RM_PERM) != 0;     // input rows in the permuted internal layout (else natural order)
  auto load = make_vec_loader<1, cplx<T>>(
      [&](int k0, cplx<T>* out) {
        if (perm) {
          const size_t e = ((size_t)(k0 >> 2) * TPL + j) * 4;
          const Quad<T> qa = ld_quad(srcA + e), qb = ld_quad(srcB + e);
#pragma unroll
          for (int i = 0; i < 4; ++i) out[i] = mk<T>(qa.v[i], qb.v[i]);
        } else {
#pragma unroll
          for (int i = 0; i < 4; ++i) out[i] = mk<T>(srcA[j + (k0 + i) * TPL], srcB[j + (k0 + i) * TPL]);
        }
      },
      [&](int, int, cplx<T> raw) -> cplx<T> { return scale * raw; });
  auto store = [&](int m, int, cplx<T> z) { line[fft_pad<NX>(m)] = z; };
  fft_line<T, NX, -1, true>(j, line, tabX, load, store);
  __syncthreads();
  // unpack: A(m) = (Z(m) + conj Z(-m))/2,  B(m) = -i (Z(m) - conj Z(-m))/2,  m = 0..Wx-1
  for (int mx = j; mx < Wx; mx += TPL) {
    const cplx<T> zp = line[fft_pad<NX>(mx)];
    const cplx<T> zm = conj(line[fft_pad<NX>((NX - mx) & (NX - 1))]);
    st_pair(dst + inter_pair_index(g, a, p, mx), (T)0.5 * (zp + zm), (T)0.5 * mul_ni(zp - zm));
  }
}

// ---------------------------------------------------------------------------------------
// fused real-space + forward row pass (conservative advection form; a3 + the row half of a4 in one kernel).
// One CTA line handles one row pair (yA = 4a+p, yB = yA+2) and runs three packed complex FFTs whose inputs are
// evaluated on the fly from v_x, v_y, w, K — the right-hand sides never exist in HBM:
//   FFT 1: Gx(yA) + i Gy(yA),  FFT 2: Gx(yB) + i Gy(yB),  FFT 3: S'(yA) + i S'(yB)
//   Gx = rhs1_x + lambda0 v_y w,  Gy = rhs1_y - lambda0 v_x w,  S' = -gamma_w K w   (pointwise.cuh, k_realspace_cons)
// Line 3 of Algorithm 1 is rhs^ = i kx Gy^ - i ky Gx^ + S'^, and i kx is still diagonal after the row pass, so only TWO
// intermediates leave the kernel:   A~ = i kx Gy~ + S'~   and   B~ = Gx~    (then rhs^ = A^ - i ky B^ in k_spectral_p2).
// At mx = 0, where i kx Gy~ vanishes but the mean-flow update (line 8) needs Gy^(0,0), the real numbers S'~(0,y) and
// Gy~(0,y) travel together as A~(0,y) = S'~ + i Gy~; the spectral kernel separates them by Hermitian symmetry.
// Spectra of the first two FFTs wait in a shared-memory stash until their partners arrive.
// Reads 4 real fields (+ K, w a second time from L2), writes 2 pruned intermediates.  grid = (Ny/2 / L)
// ---------------------------------------------------------------------------------------
template <typename T> struct Raw4 { T a, b, c, d; };

template <typename T, int NX>
__global__ void __launch_bounds__(RowCfg<T, NX>::THREADS, RowCfg<T, NX>::MINB)
k_fwd_row_fused(const __grid_constant__ Geom g, const __grid_constant__ Model m, const T* __restrict__ vx,
                const T* __restrict__ vy, const T* __restrict__ w, const T* __restrict__ K, cplx<T>* __restrict__ outA,
                cplx<T>* __restrict__ outB, const cplx<T>* __restrict__ tabX) {
  using C = RowCfg<T, NX>;
  pdl_wait();
  constexpr int TPL = C::TPL;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int c = threadIdx.x / TPL, j = threadIdx.x % TPL;
  const int rp = blockIdx.x * C::L + c;
  const int a = rp >> 1, p = rp & 1;
  const int Wx = g.Wx;
  const int stash_elems = 2 * ((Wx + 3) & ~3);
  cplx<T>* line = sm + c * C::LS;
  cplx<T>* stash = sm + C::L * C::LS + c * stash_elems;      // 2 complex per mx, owned by the thread of that mx
  const size_t offA = (size_t)(4 * a + p) * NX, offB = offA + 2 * (size_t)NX;
  const T scale = (T)g.inv_sqrt_nx;
  const T dkx = (T)g.dkx;
  const T beta = (T)m.beta, gv = (T)m.gamma_v, gw = (T)m.gamma_w, lam = (T)m.lambda0;
  if (threadIdx.x == 0) {   // L2 prefetch of the 4 consecutive rows (x 4 fields) a CTA pair about one wave later reads
    const int nb = blockIdx.x + TTSH_PF_DIST_FUSED;   // 12 row loads per CTA: a shorter distance keeps the rows in L2
    if (nb < (int)gridDim.x && ((nb * C::L) & 1) == 0) {
      const size_t off = (size_t)(2 * nb * C::L) * NX;
      const unsigned bytes = (C::L >= 2 ? 2 * C::L : 4) * NX * sizeof(T);
      prefetch_l2_bulk(vx + off, bytes); prefetch_l2_bulk(vy + off, bytes);
      prefetch_l2_bulk(w + off, bytes);  prefetch_l2_bulk(K + off, bytes);
    }
  }
  auto store = [&](int mm, int, cplx<T> z) { line[fft_pad<NX>(mm)] = z; };

#pragma unroll 1
  for (int f = 0; f < 2; ++f) {       // FFT 1 (row yA) and FFT 2 (row yB): Gx + i Gy
    const size_t off = f ? offB : offA;
    // inputs are in the permuted internal layout: slots k0..k0+3 of this thread are 4 consecutive scalars per field
    auto issue = [&](int k0, Raw4<T>* out) {
      const size_t e = off + ((size_t)(k0 >> 2) * TPL + j) * 4;
      const Quad<T> q0 = ld_quad(vx + e), q1 = ld_quad(vy + e), q2 = ld_quad(K + e), q3 = ld_quad(w + e);
#pragma unroll
      for (int i = 0; i < 4; ++i) { out[i].a = q0.v[i]; out[i].b = q1.v[i]; out[i].c = q2.v[i]; out[i].d = q3.v[i]; }
    };
    auto finish = [&](int, int, Raw4<T> r) -> cplx<T> {
      const T cc = -beta * (r.a * r.a + r.b * r.b) - gv * r.c;            // rhs1 = cc * v   (Alg. 1 line 1)
      return mk<T>(scale * (cc * r.a + lam * (r.b * r.d)), scale * (cc * r.b - lam * (r.a * r.d)));
    };
    fft_line<T, NX, -1, true>(j, line, tabX, make_vec_loader<2, Raw4<T>>(issue, finish), store);
    __syncthreads();
    // unpack: Gx~(m) = (Z(m) + conj Z(-m))/2,  Gy~(m) = -i (Z(m) - conj Z(-m))/2
    for (int mx = j; mx < Wx; mx += TPL) {
      const cplx<T> zp = line[fft_pad<NX>(mx)];
      const cplx<T> zm = conj(line[fft_pad<NX>((NX - mx) & (NX - 1))]);
      const cplx<T> gx = (T)0.5 * (zp + zm), gy = (T)0.5 * mul_ni(zp - zm);
      if (f == 0) {
        stash[2 * mx] = gx;
        stash[2 * mx + 1] = gy;
      } else {   // the same thread wrote stash[2 mx ..] in the first pass
        st_pair(outB + inter_pair_index(g, a, p, mx), stash[2 * mx], gx);     // B~ = Gx~ of rows (yA, yB)
        stash[2 * mx] = gy;                                                   // stash now holds Gy~ of (yB, yA)
      }
    }
  }
  {                                    // FFT 3: S'(yA) + i S'(yB), then A~ = i kx Gy~ + S'~
    auto issue = [&](int k0, Raw4<T>* out) {
      const size_t e = ((size_t)(k0 >> 2) * TPL + j) * 4;
      const Quad<T> q0 = ld_quad(K + offA + e), q1 = ld_quad(w + offA + e), q2 = ld_quad(K + offB + e), q3 = ld_quad(w + offB + e);
#pragma unroll
      for (int i = 0; i < 4; ++i) { out[i].a = q0.v[i]; out[i].b = q1.v[i]; out[i].c = q2.v[i]; out[i].d = q3.v[i]; }
    };
    auto finish = [&](int, int, Raw4<T> r) -> cplx<T> {
      const T s = -gw * scale;
      return mk<T>(s * (r.a * r.b), s * (r.c * r.d));                      // damping part of rhs2   (line 2)
    };
    fft_line<T, NX, -1, true>(j, line, tabX, make_vec_loader<2, Raw4<T>>(issue, finish), store);
    __syncthreads();
    for (int mx = j; mx < Wx; mx += TPL) {
      const cplx<T> zp = line[fft_pad<NX>(mx)];
      const cplx<T> zm = conj(line[fft_pad<NX>((NX - mx) & (NX - 1))]);
      cplx<T> sa = (T)0.5 * (zp + zm), sb = (T)0.5 * mul_ni(zp - zm);       // S'~ of rows yA, yB
      const cplx<T> gyA = stash[2 * mx + 1], gyB = stash[2 * mx];
      if (mx == 0) {                   // all four numbers are real here: pack Gy~(0,y) into the imaginary part
        sa = mk<T>(sa.x, gyA.x);
        sb = mk<T>(sb.x, gyB.x);
      } else {
        const T kx = dkx * (T)mx;
        sa = sa + kx * mul_i(gyA);
        sb = sb + kx * mul_i(gyB);
      }
      st_pair(outA + inter_pair_index(g, a, p, mx), sa, sb);
    }
  }
}

}  // namespace ttsh
