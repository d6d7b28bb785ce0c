// row_step_t3.cuh — the row half of one Euler step (row_step.cuh: a2/a6 row pass -> lines 1-2 of Algorithm 1 -> a4 row pass,
// PAPER.md:292-294) for Nx = 4096 in fp64, laid out for TWELVE warps per SM instead of eight.
//
// Why another layout: k_row_step keeps two of the three packed fields of a row pair in registers / a private stash, which takes
// all 64 K registers for 8 warps, and 8 warps run the fp64 pipe and the shared-memory data pipe one after the other (DESIGN.md §6:
// 126 us of arithmetic + 125 us of exchanges = 258 us).  The stage micro-benchmark there says 12 warps in independent teams overlap
// the two pipes.  Here a row pair (y_A = 4a+p, y_B = y_A+2) lives in THREE shared-memory lines (3 x 68 KB), one team of 4 warps each,
// every transform runs IN PLACE, and a thread holds one radix-16 butterfly (16 values) at a time:
//
//   line 0 (team 0):  w(y_A) + i w(y_B)            -> S'(y_A) + i S'(y_B)
//   line 1 (team 1):  v_x(y_A) + i v_y(y_A) = u_A  -> Gx(y_A) + i Gy(y_A) = (cc_A - i lw_A) u_A
//   line 2 (team 2):  v_x(y_B) + i v_y(y_B) = u_B  -> Gx(y_B) + i Gy(y_B)
//
// (cc = -beta |v|^2 - gamma_v K, lw = lambda0 w: lines 1-2 of Algorithm 1 in the conservative form, row_step.cuh.)  Packing the two
// velocity components of ONE row makes the pointwise stage local to the thread that finishes the inverse transform of u: it needs
// only the real number w(y, x) from line 0 and K(y, x), so u never makes the round trip through shared memory between the inverse
// and the forward transform, and there is no separate pointwise phase.
//
//   inverse (decimation in frequency), N = 16 x 16 x 16, input bin m = j + 256 r, output x = s + 16 s' + 256 s'' at position
//   256 s + 16 s' + s'' (digit-reversed; the pointwise stage does not care and K comes in that order, k_reperm_t3):
//     A  butterfly j in [0,256):  v[r] = Z[j + 256 r]  ->  DFT16  ->  x W_N^{j s}     -> position j + 256 s        (team barrier)
//     B  block s, c in [0,16):    v[r'] = [256 s + c + 16 r'] -> DFT16 -> x W_256^{c s'} -> position 256 s + c + 16 s'   (__syncwarp)
//     C  block s, s' in [0,16):   v[c] = [256 s + 16 s' + c]  -> DFT16                -> position 256 s + 16 s' + s''
//   forward (decimation in time) = the same three stages backwards (C', B' with the twiddles on the inputs, A'), output bin
//   256 k0 + 16 k1 + k2 at that position: natural order, so the unpack reads bins m and N - m directly.
//   A warp owns four 256-point blocks through B, C, C', B': only A and A' are team-wide.
//
// Stage A reads its inputs (the pruned inverse intermediates, retained bins |m| <= N/4 only) straight from global memory into
// registers, one row pair AHEAD (issued before the unpack of the previous row pair); butterflies j and 256 - j need the same eight
// bins (one as Z(m), the other as Z(N - m)), so a thread runs that pair and every bin is loaded once.
// Stage A' runs the same butterfly pairs, so a thread ends up with Z(m) and Z(N - m) of its eight bins in registers and unpacks
// them there; a team writes its own row's half of the output pairs
//   B~ = (Gx~(y_A), Gx~(y_B)),   A~ = i k_x Gy~ + S'~   (fft_passes.cuh, k_fwd_row_fused),
// S'~ coming from line 0.  Stage A of the next row pair writes exactly the columns the thread read in A', so no barrier separates
// the two.  Synchronisation per row pair: team barriers after A and before A', and four handshakes with team 0 (bar.arrive /
// bar.sync): "w is in line 0", "S' is in line 0", "S'~ is in line 0", "line 0 is free".  No CTA-wide barrier in the loop.
#pragma once
#include "fft_passes.cuh"

namespace ttsh {

template <typename T, int NX> struct RowStep3Cfg {
  static constexpr int TEAM = 128, THREADS = 3 * TEAM;
  static constexpr int LS = NX + NX / 16;                         // padded line: i + (i >> 4)
  static constexpr int NA = 5;                                    // stage A / A' base powers 1, 2, 3, 4, 8 of W_N^j (12 = 8 + 4 derived)
  static constexpr int NBP = 6;                                   // stage B / B' base powers 1, 2, 3, 4, 8, 12 of W_256^c
  static constexpr int TW_ELEMS = NA * 256 + NBP * 16;
  static constexpr size_t OFF_TW = (size_t)3 * LS * sizeof(cplx<T>);
  static constexpr size_t SMEM = OFF_TW + (size_t)TW_ELEMS * sizeof(cplx<T>);
  static constexpr bool FITS = NX == 4096 && SMEM <= 227 * 1024;
};
__host__ __device__ constexpr int row_step3_tw_elems() { return 5 * 256 + 6 * 16; }
__host__ __device__ constexpr int row_step3_powA(int b) { return b < 4 ? b + 1 : 8; }

__device__ __forceinline__ int t3_pad(int i) { return i + (i >> 4); }
// real-space x of line position p (and back: the map is an involution on 3 hex digits)
__host__ __device__ __forceinline__ int t3_digit_reverse(int p) { return (p >> 8) + 16 * ((p >> 4) & 15) + 256 * (p & 15); }
__device__ __forceinline__ void named_bar(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }
__device__ __forceinline__ void named_bar_arrive(int id, int nthreads) {
  __threadfence_block();                         // the arriving thread's shared-memory writes are visible to the waiting threads
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ Quad<double> ldg_quad(const double* p) {
  Quad<double> r;
  asm volatile("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.v[0]), "=d"(r.v[1]), "=d"(r.v[2]), "=d"(r.v[3]) : "l"(p));
  return r;
}
__device__ __forceinline__ Quad<float> ldg_quad(const float* p) {
  Quad<float> r;
  asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]) : "l"(p));
  return r;
}
template <int DIR, typename T> __device__ __forceinline__ TwBase<16, T> t3_twA(const cplx<T>* __restrict__ tw, int j) {
  TwBase<16, T> b;
#pragma unroll
  for (int i = 0; i < 5; ++i) { const cplx<T> w = tw[i * 256 + j]; b.w[i] = DIR < 0 ? w : conj(w); }
  b.w[5] = b.w[4] * b.w[3];
  return b;
}
template <int DIR, typename T> __device__ __forceinline__ TwBase<16, T> t3_twB(const cplx<T>* __restrict__ tw, int c) {
  TwBase<16, T> b;
#pragma unroll
  for (int i = 0; i < 6; ++i) { const cplx<T> w = tw[5 * 256 + i * 16 + c]; b.w[i] = DIR < 0 ? w : conj(w); }
  return b;
}

// stages B, C (inverse) or C', B' (forward) of the four blocks a warp owns; wq = warp of the team, l = lane
template <int DIR, typename T>
__device__ __forceinline__ void t3_warp_stages(cplx<T>* __restrict__ line, const cplx<T>* __restrict__ tw, int wq, int l) {
  const int c = l & 15;
  const int s0 = 4 * wq + (l >> 4);
  if constexpr (DIR > 0) {
    {
      const TwBase<16, T> tb = t3_twB<DIR>(tw, c);
#pragma unroll
      for (int pi = 0; pi < 2; ++pi) {
        cplx<T>* blk = line + 272 * (s0 + 2 * pi) + c;
        cplx<T> v[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = blk[17 * r];
        dft16<DIR>(v);
        apply_stage_twiddles<16>(v, tb);
#pragma unroll
        for (int r = 0; r < 16; ++r) blk[17 * r] = v[r];
      }
    }
    __syncwarp();
#pragma unroll
    for (int pi = 0; pi < 2; ++pi) {
      cplx<T>* blk = line + 272 * (s0 + 2 * pi) + 17 * c;
      cplx<T> v[16];
#pragma unroll
      for (int r = 0; r < 16; ++r) v[r] = blk[r];
      dft16<DIR>(v);
#pragma unroll
      for (int r = 0; r < 16; ++r) blk[r] = v[r];
    }
  } else {
#pragma unroll
    for (int pi = 0; pi < 2; ++pi) {
      cplx<T>* blk = line + 272 * (s0 + 2 * pi) + 17 * c;
      cplx<T> v[16];
#pragma unroll
      for (int r = 0; r < 16; ++r) v[r] = blk[r];
      dft16<DIR>(v);
#pragma unroll
      for (int r = 0; r < 16; ++r) blk[r] = v[r];
    }
    __syncwarp();
    const TwBase<16, T> tb = t3_twB<DIR>(tw, c);
#pragma unroll
    for (int pi = 0; pi < 2; ++pi) {
      cplx<T>* blk = line + 272 * (s0 + 2 * pi) + c;
      cplx<T> v[16];
#pragma unroll
      for (int r = 0; r < 16; ++r) v[r] = blk[17 * r];
      apply_stage_twiddles<16>(v, tb);
      dft16<DIR>(v);
#pragma unroll
      for (int r = 0; r < 16; ++r) blk[17 * r] = v[r];
    }
  }
}


// one radix-16 butterfly of stage A (inverse): v = the 16 bins j + 256 r (zeros outside the retained band already in place)
template <typename T>
__device__ __forceinline__ void t3_inverse_A_butterfly(cplx<T> (&v)[16], int j, cplx<T>* __restrict__ line, const cplx<T>* __restrict__ tw) {
  const TwBase<16, T> tb = t3_twA<+1>(tw, j);
  dft16<+1>(v);
  apply_stage_twiddles<16>(v, tb);
  cplx<T>* col = line + j + (j >> 4);
#pragma unroll
  for (int s = 0; s < 16; ++s) col[272 * s] = v[s];
}

// one radix-16 butterfly of stage A' (forward): bins 256 k0 + i, k0 = 0..15, left in registers
template <typename T>
__device__ __forceinline__ void t3_forward_A_butterfly(cplx<T> (&v)[16], int i, const cplx<T>* __restrict__ line, const cplx<T>* __restrict__ tw) {
  const cplx<T>* col = line + i + (i >> 4);
  const TwBase<16, T> tb = t3_twA<-1>(tw, i);
#pragma unroll
  for (int n0 = 0; n0 < 16; ++n0) v[n0] = col[272 * n0];
  apply_stage_twiddles<16>(v, tb);
  dft16<-1>(v);
}
// ENS: the persistent grid runs over the row pairs of `members` systems whose workspaces lie mstride bytes apart
// (ttsh_ensemble_step); rpm = Ny/2 row pairs per member.  K3: one plane of NX values per row, (rp 2 + r) NX + e, in the order the
// pointwise stage reads it: line position p = 256 s + 16 c + 4 q + i (x = digit-reversed p) at e = ((4 s + q) 16 + c) 4 + i, so that
// the 16 threads c of a block read 512 contiguous bytes per access (k_reperm_t3); tab3: [5][256] W_N^{j b}, b = 1, 2, 3, 4, 8, then [6][16] W_256^{c b}, b = 1, 2, 3, 4, 8, 12.
template <typename T, int NX, bool ENS>
__global__ void __launch_bounds__(RowStep3Cfg<T, NX>::THREADS, 1)
k_row_step_t3(const __grid_constant__ Geom g, const __grid_constant__ Model m, const cplx<T>* __restrict__ inW,
              const cplx<T>* __restrict__ inVx, const cplx<T>* __restrict__ inPsi, const T* __restrict__ K3,
              cplx<T>* __restrict__ outA, cplx<T>* __restrict__ outB, const cplx<T>* __restrict__ tab3,
              const double* __restrict__ v0, int nblk, int rpm, size_t mstride) {
  using C = RowStep3Cfg<T, NX>;
  constexpr int BAR_W = 5, BAR_S = 6;             // "w is in line 0" (team 0 -> teams 1, 2), "S' is in line 0" (teams 1, 2 -> team 0)
  constexpr int BAR_Z = 7, BAR_F = 8;             // "S'~ is in line 0" (team 0 -> teams 1, 2), "line 0 is free" (teams 1, 2 -> team 0)
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx<T>* lines = reinterpret_cast<cplx<T>*>(smem_raw);
  cplx<T>* tw = reinterpret_cast<cplx<T>*>(smem_raw + C::OFF_TW);
  const int tid = threadIdx.x;
  const int f = tid >> 7, t = tid & 127, wq = t >> 5, l = t & 31;
  cplx<T>* line = lines + f * C::LS;
  const int Wx = g.Wx;
  const T scale_i = (T)g.inv_sqrt_nx, scale_f = (T)g.inv_sqrt_nx;
  const T dkx = (T)g.dkx;
  const T beta = (T)m.beta, gv = (T)m.gamma_v, lam = (T)m.lambda0;
  const T ngw = -(T)m.gamma_w * scale_f;
  const size_t in_stride = (size_t)g.Wxp * 2;               // elements per row pair of an inverse intermediate
  const unsigned in_bytes = (unsigned)(in_stride * sizeof(cplx<T>)), k_bytes = (unsigned)(2 * NX * sizeof(T));
  auto locate = [&](int rpg, int& rp_, size_t& mo_) {
    if constexpr (ENS) { const int mb = rpg / rpm; rp_ = rpg - mb * rpm; mo_ = (size_t)mb * mstride; }
    else { rp_ = rpg; mo_ = 0; }
  };
  // the eight bins of this thread's butterfly pair (j, 256 - j): lo[k] = t + 256 k, hi[k] = 256 - t + 256 k.  Thread 0 runs j = 0
  // (bins 0, 256, 512, 768, 1024) and j = 128 (bins 128, 384, 640, 896): lo[k] = 256 k, hi = 128, 384, 640, 1024, and bin 896 in ex.
  const bool t0 = (t == 0);
  auto bin_lo = [&](int k) -> int { return t + 256 * k; };
  auto bin_hi = [&](int k) -> int { return t0 ? (k < 3 ? 128 + 256 * k : 1024) : 256 - t + 256 * k; };
  // raw record of one bin: team 0: (w~(m, y_A), w~(m, y_B)); team 1 / 2: (v_x~(m, y), psi~(m, y)) of the team's row
  auto fetch = [&](const cplx<T>* rowW, const cplx<T>* rowVx, const cplx<T>* rowPsi, int mx) -> Pair<T> {
    if (f == 0) return ld_pair(rowW + 2 * mx);
    Pair<T> r;
    r.a = ld_c(rowVx + 2 * mx + (f - 1));
    r.b = ld_c(rowPsi + 2 * mx + (f - 1));
    return r;
  };
  Pair<T> lo[4], hi[4], ex;
  ex.a = mk<T>(0, 0); ex.b = mk<T>(0, 0);
  auto prefetch = [&](int rpg) {
    int rp_; size_t mo_;
    locate(rpg, rp_, mo_);
    const cplx<T>* rowW = byte_off(inW, mo_) + (size_t)rp_ * in_stride;
    const cplx<T>* rowVx = byte_off(inVx, mo_) + (size_t)rp_ * in_stride;
    const cplx<T>* rowPsi = byte_off(inPsi, mo_) + (size_t)rp_ * in_stride;
#pragma unroll
    for (int k = 0; k < 4; ++k) lo[k] = fetch(rowW, rowVx, rowPsi, bin_lo(k));
#pragma unroll
    for (int k = 0; k < 4; ++k) hi[k] = fetch(rowW, rowVx, rowPsi, bin_hi(k));
    if (t0) ex = fetch(rowW, rowVx, rowPsi, 896);
  };

  for (int i = tid; i < C::TW_ELEMS; i += C::THREADS) tw[i] = ldg_c(tab3 + i);   // host-written at ttsh_create
  __syncthreads();
  pdl_wait();          // inputs, K and v0 below are written by the preceding launches
  pdl_trigger();
  T meany = (T)0;
  if constexpr (!ENS) meany = (T)(v0[1] * g.inv_sqrt_ny);
  if ((int)blockIdx.x < nblk) prefetch(blockIdx.x);

#pragma unroll 1
  for (int blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
    int rp; size_t mo;
    locate(blk, rp, mo);
    if constexpr (ENS) meany = (T)(byte_off(v0, mo)[1] * g.inv_sqrt_ny);
    const int a = rp >> 1, p = rp & 1;
    const int nb = blk + gridDim.x;
    if (t == 0 && nb < nblk) {   // L2 prefetch of what the CTA reads in its next iteration
      int nrp; size_t nmo;
      locate(nb, nrp, nmo);
      const cplx<T>* src = f == 0 ? inW : (f == 1 ? inVx : inPsi);
      prefetch_l2_bulk(byte_off(src, nmo) + (size_t)nrp * in_stride, in_bytes);
      if (f == 0) prefetch_l2_bulk(byte_off(K3, nmo) + (size_t)nrp * 2 * NX, k_bytes);
    }
    // ---- a2 / a6, stage A: Z(m) = scale (wa + i wb), Z(N - m) = scale (conj wa + i conj wb) with
    //      team 0: wa = w~(m, y_A), wb = w~(m, y_B);  team 1 / 2: wa = v_x~(m, y), wb = v_y~(m, y) = -i k_x psi~ (mean flow at m = 0)
    {
      auto prep = [&](Pair<T> r, int mx) -> Pair<T> {
        if (f != 0) r.b = mx == 0 ? mk<T>(meany, (T)0) : (dkx * (T)mx) * mul_ni(r.b);
        if (mx == 0) { r.a.y = 0; r.b.y = 0; }
        return r;
      };
      auto zpos = [&](Pair<T> r) -> cplx<T> { return scale_i * mk<T>(r.a.x - r.b.y, r.a.y + r.b.x); };
      auto zneg = [&](Pair<T> r) -> cplx<T> { return scale_i * mk<T>(r.a.x + r.b.y, r.b.x - r.a.y); };
      auto sel = [&](Pair<T> x, Pair<T> y) -> Pair<T> {          // t0 ? x : y
        Pair<T> r;
        r.a = mk<T>(t0 ? x.a.x : y.a.x, t0 ? x.a.y : y.a.y);
        r.b = mk<T>(t0 ? x.b.x : y.b.x, t0 ? x.b.y : y.b.y);
        return r;
      };
#pragma unroll
      for (int k = 0; k < 4; ++k) { lo[k] = prep(lo[k], bin_lo(k)); hi[k] = prep(hi[k], bin_hi(k)); }
      ex = prep(ex, 896);
      cplx<T> v[16];
      // butterfly j = t:  bins t + 256 k as Z(m), bins 1024 - t - 256 k as Z(N - m)
#pragma unroll
      for (int k = 0; k < 4; ++k) v[k] = zpos(lo[k]);
      v[4] = t0 ? zpos(hi[3]) : mk<T>(0, 0);
#pragma unroll
      for (int k = 5; k < 12; ++k) v[k] = mk<T>(0, 0);
      v[12] = zneg(hi[3]);
      v[13] = zneg(sel(lo[3], hi[2]));
      v[14] = zneg(sel(lo[2], hi[1]));
      v[15] = zneg(sel(lo[1], hi[0]));
      t3_inverse_A_butterfly<T>(v, t, line, tw);
      // butterfly j = 256 - t (thread 0: j = 128)
      v[0] = zpos(hi[0]); v[1] = zpos(hi[1]); v[2] = zpos(hi[2]); v[3] = zpos(sel(ex, hi[3]));
#pragma unroll
      for (int k = 4; k < 12; ++k) v[k] = mk<T>(0, 0);
      v[12] = zneg(sel(ex, lo[3]));
      v[13] = zneg(sel(hi[2], lo[2]));
      v[14] = zneg(sel(hi[1], lo[1]));
      v[15] = zneg(sel(hi[0], lo[0]));
      t3_inverse_A_butterfly<T>(v, t0 ? 128 : 256 - t, line, tw);
    }
    named_bar(1 + f, C::TEAM);
    if (f == 0) {
      t3_warp_stages<+1>(line, tw, wq, l);                  // w in place
      named_bar_arrive(BAR_W, C::THREADS);
      named_bar(BAR_S, C::THREADS);                         // S' of both rows is in line 0
      t3_warp_stages<-1>(line, tw, wq, l);
    } else {
      // stage B, then per 16-point block: stage C -> lines 1-2 of Algorithm 1 -> stage C' in registers, then stage B'
      const int c = l & 15;
      const int s0 = 4 * wq + (l >> 4);
      const T* kplane = byte_off(K3, mo) + ((size_t)rp * 2 + (f - 1)) * NX;
      {
        const TwBase<16, T> tb = t3_twB<+1>(tw, c);
#pragma unroll
        for (int pi = 0; pi < 2; ++pi) {
          cplx<T>* bl = line + 272 * (s0 + 2 * pi) + c;
          cplx<T> v[16];
#pragma unroll
          for (int r = 0; r < 16; ++r) v[r] = bl[17 * r];
          dft16<+1>(v);
          apply_stage_twiddles<16>(v, tb);
#pragma unroll
          for (int r = 0; r < 16; ++r) bl[17 * r] = v[r];
        }
      }
      __syncwarp();
#pragma unroll 1
      for (int pi = 0; pi < 2; ++pi) {
        const int s = s0 + 2 * pi;
        cplx<T>* bl = line + 272 * s + 17 * c;
        Quad<T> kq[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) kq[q] = ldg_quad(kplane + ((4 * s + q) * 16 + c) * 4);     // K at positions 256 s + 16 c + 4 q + (0..3)
        cplx<T> v[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) v[r] = bl[r];
        dft16<+1>(v);
        if (pi == 0) named_bar(BAR_W, C::THREADS);          // w of the whole row pair is in line 0
        T* wl = reinterpret_cast<T*>(lines + 272 * s + 17 * c) + (f - 1);      // Re (row y_A) or Im (row y_B) of line 0
#pragma unroll
        for (int r = 0; r < 16; ++r) {
          const T w = wl[2 * r], kk = kq[r >> 2].v[r & 3];
          const T vx = v[r].x, vy = v[r].y;
          const T cc = scale_f * (-beta * (vx * vx + vy * vy) - gv * kk);
          const T lw = scale_f * lam * w;
          v[r] = mk<T>(cc * vx + lw * vy, cc * vy - lw * vx);                  // Gx + i Gy
          wl[2 * r] = ngw * (kk * w);                                          // S'
        }
        dft16<-1>(v);
#pragma unroll
        for (int r = 0; r < 16; ++r) bl[r] = v[r];
      }
      named_bar_arrive(BAR_S, C::THREADS);
      __syncwarp();
      {
        const TwBase<16, T> tb = t3_twB<-1>(tw, c);
#pragma unroll
        for (int pi = 0; pi < 2; ++pi) {
          cplx<T>* bl = line + 272 * (s0 + 2 * pi) + c;
          cplx<T> v[16];
#pragma unroll
          for (int r = 0; r < 16; ++r) v[r] = bl[17 * r];
          apply_stage_twiddles<16>(v, tb);
          dft16<-1>(v);
#pragma unroll
          for (int r = 0; r < 16; ++r) bl[17 * r] = v[r];
        }
      }
    }
    named_bar(1 + f, C::TEAM);
    // ---- stage A' for the butterfly pair (i, 256 - i): the thread then holds Z(m) AND Z(N - m) of its eight bins m ----
    const int i2 = t0 ? 128 : 256 - t;
    if (f == 0) {
      // S'~: the retained bins go back to line 0 in place, where teams 1 and 2 pick them up
      cplx<T> v[16];
      t3_forward_A_butterfly<T>(v, t, line, tw);
      {
        cplx<T>* col = line + t + (t >> 4);
#pragma unroll
        for (int k0 = 0; k0 < 4; ++k0) col[272 * k0] = v[k0];
        if (t0) col[272 * 4] = v[4];
#pragma unroll
        for (int k0 = 12; k0 < 16; ++k0) col[272 * k0] = v[k0];
      }
      t3_forward_A_butterfly<T>(v, i2, line, tw);
      {
        cplx<T>* col = line + i2 + (i2 >> 4);
#pragma unroll
        for (int k0 = 0; k0 < 4; ++k0) col[272 * k0] = v[k0];
#pragma unroll
        for (int k0 = 12; k0 < 16; ++k0) col[272 * k0] = v[k0];
      }
      named_bar_arrive(BAR_Z, C::THREADS);
      prefetch(nb < nblk ? nb : blk);          // last iteration: a harmless re-read, so that the registers are dead through the loop body
      named_bar(BAR_F, C::THREADS);            // teams 1 and 2 have read S'~: line 0 is free for the next row pair
    } else {
      // Z1 = transform of Gx(y) + i Gy(y) of the team's row y:  Gx~(m) = (Z1(m) + conj Z1(N-m)) / 2,  Gy~(m) = -i (Z1(m) - conj Z1(N-m)) / 2;
      // S'~(m, y_A) / S'~(m, y_B) are the same two combinations of Z0 (line 0).  Outputs: this row's half of the pairs
      //   B~ = Gx~,   A~ = i k_x Gy~ + S'~   (column m = 0: the real numbers S'~(0, y) + i Gy~(0, y) travel together, k_fwd_row_fused)
      cplx<T> a1[5], b1[4], a2[4], b2[4];
      {
        cplx<T> v[16];
        t3_forward_A_butterfly<T>(v, t, line, tw);
#pragma unroll
        for (int k = 0; k < 5; ++k) a1[k] = v[k];
#pragma unroll
        for (int k = 0; k < 4; ++k) b1[k] = v[12 + k];
        t3_forward_A_butterfly<T>(v, i2, line, tw);
#pragma unroll
        for (int k = 0; k < 4; ++k) { a2[k] = v[k]; b2[k] = v[12 + k]; }
      }
      prefetch(nb < nblk ? nb : blk);
      named_bar(BAR_Z, C::THREADS);
      const cplx<T>* l0 = lines;
      cplx<T>* oB = byte_off(outB, mo) + (f - 1);
      cplx<T>* oA = byte_off(outA, mo) + (f - 1);
      auto emit = [&](int mx, cplx<T> zp, cplx<T> zmr) {
        const cplx<T> zm = conj(zmr);
        const T h = (T)0.5;
        const cplx<T> gx = h * (zp + zm), gy = h * mul_ni(zp - zm);
        const cplx<T> z0p = l0[t3_pad(mx)], z0m = conj(l0[t3_pad((NX - mx) & (NX - 1))]);
        const cplx<T> sA = h * (z0p + z0m), sB = h * mul_ni(z0p - z0m);
        const cplx<T> sv = f == 1 ? sA : sB;
        cplx<T> oa = sv + (dkx * (T)mx) * mul_i(gy);
        if (mx == 0) oa = mk<T>(sv.x, gy.x);
        const size_t o = inter_pair_index(g, a, p, mx);
        st_c(oB + o, gx);
        st_c(oA + o, oa);
      };
      auto selc = [&](cplx<T> x, cplx<T> y) -> cplx<T> { return mk<T>(t0 ? x.x : y.x, t0 ? x.y : y.y); };
      // bins t + 256 k: Z(m) from butterfly t; Z(N - m) from butterfly 256 - t (thread 0: from butterfly 0 itself, bin 0 is its own mirror)
      emit(t, a1[0], selc(a1[0], b2[3]));
      emit(t + 256, a1[1], selc(b1[3], b2[2]));
      emit(t + 512, a1[2], selc(b1[2], b2[1]));
      emit(t + 768, a1[3], selc(b1[1], b2[0]));
      // bins 256 - t + 256 k (thread 0: 128 + 256 k, both halves from butterfly 128)
#pragma unroll
      for (int k = 0; k < 4; ++k) emit(i2 + 256 * k, a2[k], selc(b2[3 - k], b1[3 - k]));
      if (t0) emit(NX / 4, a1[4], b1[0]);
      named_bar_arrive(BAR_F, C::THREADS);
    }
  }
}

}  // namespace ttsh
