// row_step_real.cuh — the row half of one Euler step in ONE kernel (row_step.cuh) on ONE REAL ROW per transform:
//   Nx = 8192, the paper's production width.  In fp64 a packed row PAIR (128 KB per field) no longer fits in shared
//              memory; in fp32 it does, but the four-stage plan of an 8192-point transform is slower than what follows (8192^2 fp32:
//              749 -> 589 us for the row kernel).  256 threads, warp-local plan at M = Nx/2 = 4096.
//   Nx = 16384 in fp32 (the grid of Fig. 6(f); in fp64 a line of M = 8192 complex doubles does not leave room for the
//              staging slots): 512 threads x 128 registers, plain four-stage plan, BOTH waiting fields in tensor memory.
//              16384 x 4096 fp32: 1.76 ms per step with the 6-launch sequence of fft_rows_real.cuh, 1.17 ms with this kernel.
//
// One REAL row is transformed as a half-length complex sequence z[n] = f(2n) + i f(2n+1), n < M = Nx/2 (the textbook
// real-data FFT), so that the machinery of row_step.cuh applies unchanged at N = M: the transform plans of fft_core.cuh, one
// field live in registers (V), one waiting in registers (H), one parked by its owner thread (there: a shared-memory stash; here:
// tensor memory).  The pointwise stage
// (lines 1-2 of Algorithm 1) does not care that a complex slot now holds two neighbouring points of one row
// instead of one point of two rows.  What changes is the step between the half spectrum F (what the column passes read and
// write) and the transform Z of the packed sequence:
//
//   inverse:  Z2(m) = (F(m) + conj F(M-m)) + i W^{-m} (F(m) - conj F(M-m)),  W = exp(-2 pi i / Nx);  z = iDFT_M(Z2) / sqrt(Nx).
//             Under the 1/2 rule F(m) = 0 for m > M/2, so a slot needs ONE bin:
//               m < M/2:  Z2(m) = F(m) + i conj(W^m) F(m)          m = 0:  F(0) (1 + i)  (F(0) real)
//               m > M/2:  Z2(m) = c - i conj(W^m) c,  c = conj F(M-m)          m = M/2:  2 conj F(M/2)
//   forward:  F(k) = E(k) + W^k O(k),  E = (Z(k) + conj Z(M-k)) / 2,  O = -i (Z(k) - conj Z(M-k)) / 2,  k = 0..M/2 (retained).
//             i k_x does not commute with this step, so the three forward transforms are merged separately and
//             A~ = i k_x Gy~ + S'~ is formed on the merged bins (a thread merges the same bins k = j + TPL i of every transform, TPL = M/16).
//   W^m for m = j + TPL k is W^j W_32^k: one table entry per thread (tabR, W^j for j < TPL) and compile-time constants.
//
// A CTA takes a row pair (rows 4a+p and 4a+p+2 share the (A, B) pairs of the intermediates, ttsh_common.cuh) and runs its two
// rows one after the other.  Everything a row reads arrives by cp.async.bulk + mbarrier in two staging slots, each copy issued
// right after the barrier that ends the previous use of its slot, i.e. more than one transform ahead of its consumer:
//   slot 0:  w~ pairs -> psi~ pairs -> w~ of the next row          slot 1:  v_x~ pairs -> K row -> v_x~ of the next row
// (the same pairs again for the second row of the pair).  The waiting field (w, then S') is parked in TENSOR MEMORY (tmem.cuh) by its
// owner thread: that frees the 64 KB of shared memory the second slot needs and takes the stash traffic off the shared-memory pipe.
// The merged bins of the pair's FIRST row wait there too, so that the second row writes whole 32-byte (A, B) pairs of the forward
// intermediates (one full sector per bin) instead of 16-byte halves.
// K comes in the thread order of the plan: (K(y, 2n), K(y, 2n+1)) for n = own(t) + TPL k at (k TPL + t) 2 (k_reperm_real), own(t) =
// wl_j(t) for the warp-local plan, t for the plain one.
#pragma once
#include "row_step.cuh"
#include "tmem.cuh"

namespace ttsh {

template <typename T, int NX> struct RowStepRealCfg {
  static constexpr int M = NX / 2;                                  // complex length
  static constexpr bool WL = fft_wl_supported<M>();                 // warp-local plan (M = 4096), else the plain Stockham plan (M = 8192)
  static constexpr int TPL = M / 16, THREADS = TPL;
  static constexpr int LS = (WL ? fft_wl_line_elems<T, M>() : fft_line_elems<M>()) + 4;
  // tensor memory (tmem.cuh), per thread: the waiting field (16 complex values) and the merged bins of the pair's first row (B~ and
  // A~, 9 complex values each), in pieces of 16 columns = 4 complex doubles / 8 complex floats; THREADS / 128 warps per lane quarter
  static constexpr int CH = 16 / (2 * (int)sizeof(T) / 4);
  // the 512-thread variant (M = 8192) has 128 registers per thread: its second waiting field (v_x, then Gy) is parked as well
  static constexpr bool HTM = THREADS > 256;
  static constexpr int TMEM_NEED = (HTM ? 2 : 1) * 16 * (16 / CH) + 2 * 16 * ((9 + CH - 1) / CH);
  // allocate no more than the kernel uses (the next power of two >= columns per warp x warps per lane quarter, >= 32): a CTA
  // holds its columns for the whole persistent loop, and a second CTA on the same SM (another handle on another stream; fp32 at
  // NX = 8192 leaves room for two) would otherwise block in tcgen05.alloc until the first one ends.  fp64: 2 x 160 -> 512;
  // fp32 at NX = 8192: 2 x 96 -> 256; fp32 at NX = 16384: 4 x 128 = 512
  static constexpr unsigned tmem_cols_for(unsigned need) { unsigned c = 32; while (c < need) c *= 2; return c; }
  static constexpr unsigned TMEM_COLS = tmem_cols_for((unsigned)(THREADS >= 128 ? THREADS / 128 : 1) * TMEM_NEED);
  static constexpr int TMEM_PER_WARP = (int)TMEM_COLS / (THREADS >= 128 ? THREADS / 128 : 1);
  static constexpr size_t OFF_TAB = (size_t)LS * sizeof(cplx<T>);
  // a copy of the warp-local table in shared memory in fp64 (row_step.cuh, SMEM_TAB, says why); fp32 and the plain plan read it through L1
  static constexpr bool SMEM_TAB = WL && sizeof(T) == 8;
  static constexpr size_t TAB_BYTES = SMEM_TAB ? (size_t)fft_wl_tw_elems_rt(M) * sizeof(cplx<T>) : 0;
  // two staging slots, used in turn by the (A, B) pairs of w~, v_x~, psi~ (2 Wxp <= 2 (NX/4 + 8) complex values) and by the row of K
  static constexpr size_t SLOT = ((size_t)(NX / 4 + 8) * 2 * sizeof(cplx<T>) + 127) / 128 * 128;
  static constexpr size_t OFF_SLOTS = (OFF_TAB + TAB_BYTES + 127) / 128 * 128;
  static constexpr size_t OFF_BAR = OFF_SLOTS + 2 * SLOT;
  static constexpr size_t SMEM = OFF_BAR + 32;
  static constexpr bool FITS = THREADS % 128 == 0 && THREADS <= 1024 && TMEM_COLS <= 512 && TMEM_NEED <= TMEM_PER_WARP && SMEM <= 227 * 1024;
};

// W^m = wj W_32^k for m = j + TPL k (forward sign), k a compile-time constant after unrolling
template <typename T> __device__ __forceinline__ cplx<T> real_row_tw(cplx<T> wj, int k) { return mul_w32_rt<-1>(wj, k); }

// inverse transform of one real row into registers: out[k] = f(2n) + i f(2n+1), n = wl_j(j) + k TPL.
// row: bin m of this row at row[2 m] (its half of the staged (A, B) pairs of the inverse intermediate, shared memory).
// MODE = RM_ONE or RM_NIKX_MEANY (ttsh_common.cuh).  1/2 rule only: retained m = 0..M/2.
template <typename T, int M, bool WL, int MODE, class Hook>
__device__ __forceinline__ void inv_real_row_regs(const cplx<T>* __restrict__ row, int j, cplx<T> wj, cplx<T>* __restrict__ line,
                                                  const cplx<T>* __restrict__ tab, T scale, T dkx, T meany, cplx<T> (&out)[16], Hook hook) {
  constexpr int TPL = M / 16;
  auto mult = [&](cplx<T> w, int mx) -> cplx<T> {
    if (MODE == RM_ONE) return mx == 0 ? mk<T>(w.x, (T)0) : w;
    const T kx = dkx * (T)mx;
    return mx == 0 ? mk<T>(meany, (T)0) : kx * mul_ni(w);        // RM_NIKX_MEANY
  };
  auto issue = [&](int mm, int k) -> cplx<T> {
    if (k < 8 || (k == 8 && j == 0)) return row[2 * mm];
    return row[2 * (M - mm)];
  };
  auto finish = [&](int mm, int k, cplx<T> raw) -> cplx<T> {
    const cplx<T> wm = real_row_tw(wj, k);                        // W^mm
    if (k < 8) {
      const cplx<T> F = mult(raw, mm);
      const cplx<T> z = F + mul_i(mul_conj(F, wm));
      return scale * ((k == 0 && j == 0) ? mk<T>(F.x, F.x) : z);
    }
    const bool mid = (k == 8 && j == 0);
    const cplx<T> c = conj(mult(raw, mid ? M / 2 : M - mm));
    const cplx<T> z = c - mul_i(mul_conj(c, wm));
    return scale * (mid ? mk<T>(c.x + c.x, c.y + c.y) : z);
  };
  auto store = [&](int, int k, cplx<T> z) { out[k] = z; };
  if constexpr (WL) fft_line_wl<T, M, +1, false>(j, j, line, tab, make_loader<1>(issue, finish), store, hook);
  else fft_line<T, M, +1, false>(j, line, tab, make_loader<1>(issue, finish), store, hook);
}

// ENS: the persistent grid runs over the row pairs of `members` systems whose workspaces lie mstride bytes apart; rpm = Ny/2.
// K2: K in thread order (k_reperm_real); tabW: the warp-local table of length M (fill_stage_tables_wl); tabR: W_NX^j, j < M/16.
template <typename T, int NX, bool ENS>
__global__ void __launch_bounds__(RowStepRealCfg<T, NX>::THREADS, 1)
k_row_step_real(const __grid_constant__ Geom g, const __grid_constant__ Model m, const cplx<T>* __restrict__ inW,
                const cplx<T>* __restrict__ inVx, const cplx<T>* __restrict__ inPsi, const T* __restrict__ K2,
                cplx<T>* __restrict__ outA, cplx<T>* __restrict__ outB, const cplx<T>* __restrict__ tabW,
                const cplx<T>* __restrict__ tabR, const double* __restrict__ v0, int nblk, int rpm, size_t mstride) {
  using C = RowStepRealCfg<T, NX>;
  constexpr int M = C::M, TPL = C::TPL;
  constexpr bool WL = C::WL;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx<T>* line = reinterpret_cast<cplx<T>*>(smem_raw);
  const int j = threadIdx.x;
  const int jw = WL ? (j >> 4) + (M / 256) * (j & 15) : j;         // the thread owns slots n = jw + k TPL
  cplx<T>* stab = reinterpret_cast<cplx<T>*>(smem_raw + C::OFF_TAB);
  unsigned char* slot0 = smem_raw + C::OFF_SLOTS;
  unsigned char* slot1 = slot0 + C::SLOT;
  unsigned long long* bar0 = reinterpret_cast<unsigned long long*>(smem_raw + C::OFF_BAR);
  unsigned long long* bar1 = bar0 + 1;
  unsigned* tmem_holder = reinterpret_cast<unsigned*>(bar0 + 2);
  const T scale_i = (T)g.inv_sqrt_nx, scale_f = (T)g.inv_sqrt_nx;
  const T dkx = (T)g.dkx;
  const T beta = (T)m.beta, gv = (T)m.gamma_v, lam = (T)m.lambda0;
  const T ngw = -(T)m.gamma_w * scale_f;
  const size_t in_stride = (size_t)g.Wxp * 2;               // elements per row pair of an inverse intermediate
  const unsigned in_bytes = (unsigned)(in_stride * sizeof(cplx<T>)), k_bytes = (unsigned)(NX * sizeof(T));
  const bool leader = (j == 0);
  unsigned ph0 = 0, ph1 = 0;
  constexpr int CH = TmemPack<T>::CH, NCH = 16 / CH;          // complex values per 16 columns of tensor memory; pieces per field
  constexpr int NBP = (9 + CH - 1) / CH, NB = NBP * CH;        // the 9 merged bins of a thread in NBP pieces
  auto locate = [&](int rpg, int& rp_, size_t& mo_) {
    if constexpr (ENS) { const int mb = rpg / rpm; rp_ = rpg - mb * rpm; mo_ = (size_t)mb * mstride; }
    else { rp_ = rpg; mo_ = 0; }
  };
  if (leader) { mbar_init(bar0, 1); mbar_init(bar1, 1); }
  mbar_fence_init();
  if (j < 32) tmem_alloc(tmem_holder, C::TMEM_COLS);
  tmem_fence_before_sync();
  // the table of the warp-local plan: a copy in shared memory in fp64, through L1 in fp32 (row_step.cuh, SMEM_TAB, says why)
  if constexpr (C::SMEM_TAB) {
    for (int i = j; i < fft_wl_tw_elems_rt(M); i += C::THREADS) stab[i] = ldg_c(tabW + i);     // host-written at ttsh_create
  } else stab = const_cast<cplx<T>*>(tabW);
  const cplx<T> wj = ldg_c(tabR + j);                              // W_NX^j
  __syncthreads();
  tmem_fence_after_sync();
  const unsigned tmem_base = *tmem_holder;
  const unsigned tstash = tmem_warp_addr(tmem_base, j >> 5, C::TMEM_PER_WARP * (j >> 7));   // this thread's columns: slot k of the waiting field at column 4 k
  constexpr bool HTM = C::HTM;
  const unsigned tH = tstash + 16 * NCH;                                         // v_x, then Gy (HTM only)
  const unsigned tparkB = tH + (HTM ? 16 * NCH : 0), tparkA = tparkB + 16 * NBP; // merged B~ / A~ bins of the pair's first row
  pdl_wait();          // inputs, K and v0 below are written by the preceding launches
  pdl_trigger();
  T meany = (T)0;
  if constexpr (!ENS) meany = (T)(v0[1] * g.inv_sqrt_ny);
  if (leader && (int)blockIdx.x < nblk) {
    int rp0; size_t mo0;
    locate(blockIdx.x, rp0, mo0);
    bulk_load(slot0, byte_off(inW, mo0) + (size_t)rp0 * in_stride, in_bytes, bar0);
    bulk_load(slot1, byte_off(inVx, mo0) + (size_t)rp0 * in_stride, in_bytes, bar1);
  }

#pragma unroll 1
  for (int blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
    int rp; size_t mo;
    locate(blk, rp, mo);
    if constexpr (ENS) meany = (T)(byte_off(v0, mo)[1] * g.inv_sqrt_ny);
    const int a = rp >> 1, p = rp & 1;
    const int nb = blk + gridDim.x;
    if (leader && nb < nblk) {   // L2 prefetch of what the CTA reads in its next iteration
      int nrp; size_t nmo;
      locate(nb, nrp, nmo);
      prefetch_l2_bulk(byte_off(inW, nmo) + (size_t)nrp * in_stride, in_bytes);
      prefetch_l2_bulk(byte_off(inVx, nmo) + (size_t)nrp * in_stride, in_bytes);
      prefetch_l2_bulk(byte_off(inPsi, nmo) + (size_t)nrp * in_stride, in_bytes);
      const size_t ny = (size_t)(4 * (nrp >> 1) + (nrp & 1)) * NX;
      prefetch_l2_bulk(byte_off(K2, nmo) + ny, k_bytes);
      prefetch_l2_bulk(byte_off(K2, nmo) + ny + 2 * (size_t)NX, k_bytes);
    }
#pragma unroll 1
    for (int r = 0; r < 2; ++r) {
      const size_t y = (size_t)(4 * a + p + 2 * r);
      const cplx<T>* row0 = reinterpret_cast<const cplx<T>*>(slot0) + r;      // this row's half of the staged pairs
      const cplx<T>* row1 = reinterpret_cast<const cplx<T>*>(slot1) + r;
      const cplx<T>* kslot = reinterpret_cast<const cplx<T>*>(slot1);
      // (row pair, member offset) of the row after this one
      int xrp = rp; size_t xmo = mo; bool xok = true;
      if (r == 1) { xok = nb < nblk; if (xok) locate(nb, xrp, xmo); }
      cplx<T> H[HTM ? 1 : 16], V[16];
      // ---- a2 / a6: w, v_x, v_y of the row ----
      mbar_wait(bar0, ph0); ph0 ^= 1;
      inv_real_row_regs<T, M, WL, RM_ONE>(row0, j, wj, line, stab, scale_i, dkx, meany, V,
                                      [&]() { if (leader) bulk_load(slot0, byte_off(inPsi, mo) + (size_t)rp * in_stride, in_bytes, bar0); });
#pragma unroll
      for (int q = 0; q < NCH; ++q) tmem_stc(tstash + 16 * q, V + CH * q);   // w waits in tensor memory
      mbar_wait(bar1, ph1); ph1 ^= 1;
      if constexpr (HTM) {
        inv_real_row_regs<T, M, WL, RM_ONE>(row1, j, wj, line, stab, scale_i, dkx, meany, V,
                                        [&]() { if (leader) bulk_load(slot1, byte_off(K2, mo) + y * NX, k_bytes, bar1); });                  // v_x
#pragma unroll
        for (int q = 0; q < NCH; ++q) tmem_stc(tH + 16 * q, V + CH * q);
      } else {
        inv_real_row_regs<T, M, WL, RM_ONE>(row1, j, wj, line, stab, scale_i, dkx, meany, H,
                                        [&]() { if (leader) bulk_load(slot1, byte_off(K2, mo) + y * NX, k_bytes, bar1); });                  // v_x
      }
      mbar_wait(bar0, ph0); ph0 ^= 1;
      inv_real_row_regs<T, M, WL, RM_NIKX_MEANY>(row0, j, wj, line, stab, scale_i, dkx, meany, V, [&]() {                                        // v_y
        if (leader && xok) bulk_load(slot0, byte_off(inW, xmo) + (size_t)xrp * in_stride, in_bytes, bar0);
      });
      // ---- a3: lines 1-2 of Algorithm 1 on the two points of every slot;  V <- Gx,  H <- Gy,  tensor memory <- S' ----
      mbar_wait(bar1, ph1); ph1 ^= 1;
      tmem_wait_st();
      {
        TmemQuad wq[2], uq;
        tmem_ldc_issue(tstash, wq[0]);
#pragma unroll
        for (int q = 0; q < NCH; ++q) {
          if constexpr (HTM) tmem_ldc_issue(tH + 16 * q, uq);
          tmem_wait_ld(wq[q & 1]);
          if constexpr (HTM) tmem_wait_ld(uq);
          if (q < NCH - 1) tmem_ldc_issue(tstash + 16 * (q + 1), wq[(q + 1) & 1]);
          cplx<T> s4[CH], g4[CH];
#pragma unroll
          for (int i = 0; i < CH; ++i) {
            const int k = CH * q + i;
            const cplx<T> kk = kslot[k * TPL + j];
            const cplx<T> w = tmem_getc(wq[q & 1], i, T());
            const T kA = kk.x, kB = kk.y;
            cplx<T> vx;
            if constexpr (HTM) vx = tmem_getc(uq, i, T()); else vx = H[k];
            const T vxA = vx.x, vxB = vx.y, vyA = V[k].x, vyB = V[k].y;
            const T ccA = scale_f * (-beta * (vxA * vxA + vyA * vyA) - gv * kA);
            const T ccB = scale_f * (-beta * (vxB * vxB + vyB * vyB) - gv * kB);
            const T lwA = scale_f * lam * w.x, lwB = scale_f * lam * w.y;
            V[k] = mk<T>(ccA * vxA + lwA * vyA, ccB * vxB + lwB * vyB);          // Gx
            g4[i] = mk<T>(ccA * vyA - lwA * vxA, ccB * vyB - lwB * vxB);         // Gy
            if constexpr (!HTM) H[k] = g4[i];
            s4[i] = mk<T>(ngw * (kA * w.x), ngw * (kB * w.y));                   // S'
          }
          tmem_stc(tstash + 16 * q, s4);
          if constexpr (HTM) tmem_stc(tH + 16 * q, g4);
        }
      }
      // ---- a4: three forward transforms, each merged into the half spectrum of the row on the bins k = j + TPL i ----
      auto ident = [&](int, int, cplx<T> z) -> cplx<T> { return z; };
      auto to_line = [&](int mm, int, cplx<T> z) { line[row_step_pad<T, M, WL>(mm)] = z; };
      auto merged = [&](int i) -> cplx<T> {                          // F(k), k = j + TPL i
        const int k = j + TPL * i;
        const cplx<T> zp = line[row_step_pad<T, M, WL>(k)];
        const cplx<T> zm = conj(line[row_step_pad<T, M, WL>((M - k) & (M - 1))]);
        const cplx<T> e = (T)0.5 * (zp + zm), o = (T)0.5 * mul_ni(zp - zm);
        return e + real_row_tw(wj, i) * o;
      };
      fwd_row_regs<T, M, true, WL>(jw, j, line, stab, make_loader<1>([&](int, int k) -> cplx<T> { return V[k]; }, ident), to_line, [&]() {
        if (!leader || !xok) return;                           // K has been consumed: stage v_x~ of the next row
        bulk_load(slot1, byte_off(inVx, xmo) + (size_t)xrp * in_stride, in_bytes, bar1);
      });
      __syncthreads();
      // The merged bins of the pair's first row wait in tensor memory; the second row then writes whole (A, B) pairs (32 bytes: one
      // full sector per bin instead of two half-written ones, and half as many store instructions).
      auto emit = [&](cplx<T>* out, unsigned tpark, const cplx<T> (&mb)[NB]) {
        if (r == 0) {
#pragma unroll
          for (int q = 0; q < NBP; ++q) tmem_stc(tpark + 16 * q, mb + CH * q);
        } else {
          TmemQuad pq[NBP];
#pragma unroll
          for (int q = 0; q < NBP; ++q) tmem_ldc_issue(tpark + 16 * q, pq[q]);
#pragma unroll
          for (int q = 0; q < NBP; ++q) tmem_wait_ld(pq[q]);
#pragma unroll
          for (int i = 0; i < 9; ++i)
            if (i < 8 || leader) st_pair(out + inter_pair_index(g, a, p, j + TPL * i), tmem_getc(pq[i / CH], i % CH, T()), mb[i]);
        }
      };
      {
        cplx<T> mb[NB];
#pragma unroll
        for (int i = 0; i < NB; ++i) mb[i] = (i < 8 || (i == 8 && leader)) ? merged(i < 9 ? i : 8) : mk<T>(0, 0);
        tmem_wait_st();
        emit(byte_off(outB, mo), tparkB, mb);                                          // B~ = Gx~
      }
      cplx<T> ikg[9];
      T gy0 = (T)0;
      auto unpark = [&](unsigned tp) {                               // V <- the field parked at tp
        tmem_wait_st();
        TmemQuad sq[NCH];
#pragma unroll
        for (int q = 0; q < NCH; ++q) tmem_ldc_issue(tp + 16 * q, sq[q]);
#pragma unroll
        for (int q = 0; q < NCH; ++q) tmem_wait_ld(sq[q]);
#pragma unroll
        for (int k = 0; k < 16; ++k) V[k] = tmem_getc(sq[k / CH], k % CH, T());
      };
      if constexpr (HTM) {
        unpark(tH);                                                  // Gy
        fwd_row_regs<T, M, true, WL>(jw, j, line, stab, make_loader<1>([&](int, int k) -> cplx<T> { return V[k]; }, ident), to_line);
      } else {
        fwd_row_regs<T, M, true, WL>(jw, j, line, stab, make_loader<1>([&](int, int k) -> cplx<T> { return H[k]; }, ident), to_line);
      }
      __syncthreads();
#pragma unroll
      for (int i = 0; i < 9; ++i) {
        ikg[i] = mk<T>(0, 0);
        if (i < 8 || leader) {
          const cplx<T> gy = merged(i);
          if (i == 0) gy0 = gy.x;
          ikg[i] = (dkx * (T)(j + TPL * i)) * mul_i(gy);
        }
      }
      unpark(tstash);                                                // S'
      fwd_row_regs<T, M, true, WL>(jw, j, line, stab, make_loader<1>([&](int, int k) -> cplx<T> { return V[k]; }, ident), to_line);
      __syncthreads();
      {
        cplx<T> mb[NB];
#pragma unroll
        for (int i = 0; i < NB; ++i) {
          mb[i] = mk<T>(0, 0);
          if (i < 8 || (i == 8 && leader)) {
            mb[i] = merged(i < 9 ? i : 8) + ikg[i < 9 ? i : 8];
            if (i == 0 && leader) mb[i] = mk<T>(mb[i].x, gy0);   // real numbers S'~(0, y) and Gy~(0, y) travel together (k_fwd_row_fused)
          }
        }
        tmem_wait_st();
        emit(byte_off(outA, mo), tparkA, mb);                                          // A~ = i k_x Gy~ + S'~
      }
    }
  }
  tmem_fence_before_sync();
  __syncthreads();
  if (j < 32) tmem_dealloc(tmem_base, C::TMEM_COLS);
}

}  // namespace ttsh
