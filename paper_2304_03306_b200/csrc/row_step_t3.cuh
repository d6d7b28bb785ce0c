// row_step_t3.cuh — the row half of one Euler step (row_step.cuh: a2/a6 row pass -> lines 1-2 of Algorithm 1 -> a4 row pass,
// PAPER.md:292-294) for Nx = 4096 in fp64, laid out for TWELVE warps per SM instead of eight.
//
// Why another layout: k_row_step keeps two of the three packed fields of a row pair in registers / a private stash, which takes
// all 64 K registers for 8 warps, and 8 warps run the fp64 pipe and the shared-memory data pipe one after the other (DESIGN.md §6:
// 126 us of arithmetic + 125 us of exchanges = 258 us).  The stage micro-benchmark there says 12 warps in independent teams overlap
// the two pipes.  Here the three fields of a row pair live in THREE shared-memory lines (3 x 68 KB), one team of 4 warps per field,
// and every transform runs IN PLACE, so a thread holds one radix-16 butterfly (16 values) at a time and does two per stage:
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
// Per row pair: 1 team barrier + CTA barrier | pointwise on all positions by all 384 threads | CTA barrier + 1 team barrier |
// unpack (team 1: B~ from Gx~;  teams 0 and 2 together: A~ = unpack(i k_m Zgy + Zs)).  Inputs are read straight from global memory
// (L2-prefetched one row pair ahead) by the first inverse stage, which is pruned to the retained bins like row_step.cuh.
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

// stage A of the inverse transform of one packed row pair: the staged pairs (A, B) of column mx at row[2 mx] (global memory, inverse
// intermediate layout), Z(m) = scale (wa + i wb), Z(N - m) = scale (conj wa + i conj wb); retained mx = 0..NX/4 only (1/2 rule).
template <typename T, int NX, int MODE>
__device__ __forceinline__ void t3_inverse_A(const cplx<T>* __restrict__ row, int t, cplx<T>* __restrict__ line, const cplx<T>* __restrict__ tw,
                                             T scale, T dkx, T meany) {
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
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {
    const int j = t + 128 * h;
    Pair<T> lo[4], hi[4], mid;
#pragma unroll
    for (int k = 0; k < 4; ++k) lo[k] = ld_pair(row + 2 * (j + 256 * k));
#pragma unroll
    for (int k = 0; k < 4; ++k) hi[k] = ld_pair(row + 2 * (NX - (j + 256 * (12 + k))));
    mid.a = mk<T>(0, 0); mid.b = mk<T>(0, 0);
    if (j == 0) mid = ld_pair(row + 2 * (NX / 4));
    const TwBase<16, T> tb = t3_twA<+1>(tw, j);
    cplx<T> v[16];
#pragma unroll
    for (int k = 0; k < 4; ++k) v[k] = combine(lo[k], j + 256 * k, false);
    v[4] = j == 0 ? combine(mid, NX / 4, false) : mk<T>(0, 0);
#pragma unroll
    for (int k = 5; k < 12; ++k) v[k] = mk<T>(0, 0);
#pragma unroll
    for (int k = 0; k < 4; ++k) v[12 + k] = combine(hi[k], NX - (j + 256 * (12 + k)), true);
    dft16<+1>(v);
    apply_stage_twiddles<16>(v, tb);
#pragma unroll
    for (int s = 0; s < 16; ++s) line[j + (j >> 4) + 272 * s] = v[s];
  }
}

// stage A' of the forward transform: bins 256 k0 + i in place; only the retained bins (|m| <= NX/4) are stored
template <typename T, int NX>
__device__ __forceinline__ void t3_forward_A(int t, cplx<T>* __restrict__ line, const cplx<T>* __restrict__ tw) {
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {
    const int i = t + 128 * h;
    cplx<T>* col = line + i + (i >> 4);
    const TwBase<16, T> tb = t3_twA<-1>(tw, i);
    cplx<T> v[16];
#pragma unroll
    for (int n0 = 0; n0 < 16; ++n0) v[n0] = col[272 * n0];
    apply_stage_twiddles<16>(v, tb);
    dft16<-1>(v);
#pragma unroll
    for (int k0 = 0; k0 < 4; ++k0) col[272 * k0] = v[k0];
    if (i == 0) col[272 * 4] = v[4];
#pragma unroll
    for (int k0 = 12; k0 < 16; ++k0) col[272 * k0] = v[k0];
  }
}

// ENS: the persistent grid runs over the row pairs of `members` systems whose workspaces lie mstride bytes apart
// (ttsh_ensemble_step); rpm = Ny/2 row pairs per member.  K3: K in line-position order, (K(y_A, x(p)), K(y_B, x(p))) at
// ((rp NX) + p) 2 (k_reperm_t3); tab3: [5][256] W_N^{j b}, b = 1, 2, 3, 4, 8, then [6][16] W_256^{c b}, b = 1, 2, 3, 4, 8, 12.
template <typename T, int NX, bool ENS>
__global__ void __launch_bounds__(RowStep3Cfg<T, NX>::THREADS, 1)
k_row_step_t3(const __grid_constant__ Geom g, const __grid_constant__ Model m, const cplx<T>* __restrict__ inW,
              const cplx<T>* __restrict__ inVx, const cplx<T>* __restrict__ inPsi, const T* __restrict__ K3,
              cplx<T>* __restrict__ outA, cplx<T>* __restrict__ outB, const cplx<T>* __restrict__ tab3,
              const double* __restrict__ v0, int nblk, int rpm, size_t mstride) {
  using C = RowStep3Cfg<T, NX>;
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
  const cplx<T>* in_f = f == 0 ? inW : (f == 1 ? inVx : inPsi);

  for (int i = tid; i < C::TW_ELEMS; i += C::THREADS) tw[i] = ldg_c(tab3 + i);   // host-written at ttsh_create
  __syncthreads();
  pdl_wait();          // inputs, K and v0 below are written by the preceding launches
  pdl_trigger();
  T meany = (T)0;
  if constexpr (!ENS) meany = (T)(v0[1] * g.inv_sqrt_ny);

#pragma unroll 1
  for (int blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
    int rp; size_t mo;
    locate(blk, rp, mo);
    if constexpr (ENS) meany = (T)(byte_off(v0, mo)[1] * g.inv_sqrt_ny);
    const int a = rp >> 1, p = rp & 1;
    const int nb = blk + gridDim.x;
    if (t == 0 && nb < nblk) {   // L2 prefetch of what this team reads in the CTA's next iteration
      int nrp; size_t nmo;
      locate(nb, nrp, nmo);
      prefetch_l2_bulk(byte_off(in_f, nmo) + (size_t)nrp * in_stride, in_bytes);
      if (f == 0) prefetch_l2_bulk(byte_off(K3, nmo) + (size_t)nrp * 2 * NX, k_bytes);
    }
    // ---- a2 / a6: w (team 0), v_x (team 1), v_y (team 2) of the two rows, in place in the team's line ----
    {
      const cplx<T>* row = byte_off(in_f, mo) + (size_t)rp * in_stride;
      if (f == 2) t3_inverse_A<T, NX, RM_NIKX_MEANY>(row, t, line, tw, scale_i, dkx, meany);
      else t3_inverse_A<T, NX, RM_ONE>(row, t, line, tw, scale_i, dkx, meany);
    }
    named_bar(1 + f, C::TEAM);
    t3_warp_stages<+1>(line, tw, wq, l);
    // ---- a3: lines 1-2 of Algorithm 1 on every position (x = digit-reversed p; K comes in the same order) ----
    constexpr int NP = (NX + C::THREADS - 1) / C::THREADS;
    cplx<T> kk[NP];
    {
      const T* krow = byte_off(K3, mo) + (size_t)rp * 2 * NX;
#pragma unroll
      for (int i = 0; i < NP; ++i) {
        const int pos = tid + i * C::THREADS;
        kk[i] = pos < NX ? ldg_c(reinterpret_cast<const cplx<T>*>(krow) + pos) : mk<T>(0, 0);
      }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < NP; ++i) {
      const int pos = tid + i * C::THREADS;
      if (pos < NX) {
        const int q = t3_pad(pos);
        const cplx<T> w = lines[q], vx = lines[C::LS + q], vy = lines[2 * C::LS + q];
        const T kA = kk[i].x, kB = kk[i].y;
        const T vxA = vx.x, vxB = vx.y, vyA = vy.x, vyB = vy.y;
        const T ccA = scale_f * (-beta * (vxA * vxA + vyA * vyA) - gv * kA);
        const T ccB = scale_f * (-beta * (vxB * vxB + vyB * vyB) - gv * kB);
        const T lwA = scale_f * lam * w.x, lwB = scale_f * lam * w.y;
        lines[q] = mk<T>(ngw * (kA * w.x), ngw * (kB * w.y));                                  // S'
        lines[C::LS + q] = mk<T>(ccA * vxA + lwA * vyA, ccB * vxB + lwB * vyB);                // Gx
        lines[2 * C::LS + q] = mk<T>(ccA * vyA - lwA * vxA, ccB * vyB - lwB * vxB);            // Gy
      }
    }
    __syncthreads();
    // ---- a4: forward transforms of S' (team 0), Gx (team 1), Gy (team 2) ----
    t3_warp_stages<-1>(line, tw, wq, l);
    named_bar(1 + f, C::TEAM);
    t3_forward_A<T, NX>(t, line, tw);
    if (f == 1) {
      // B~ = Gx~: unpack the packed transform of (Gx(y_A), Gx(y_B))
      named_bar(2, C::TEAM);
      for (int mx = t; mx < Wx; mx += C::TEAM) {
        const cplx<T> zp = line[t3_pad(mx)];
        const cplx<T> zm = conj(line[t3_pad((NX - mx) & (NX - 1))]);
        st_pair(byte_off(outB, mo) + inter_pair_index(g, a, p, mx), (T)0.5 * (zp + zm), (T)0.5 * mul_ni(zp - zm));
      }
      named_bar(2, C::TEAM);                       // line 1 is free for the next row pair
    } else {
      // A~ = unpack(i k_m Zgy(m) + Zs(m)), k_m the signed wavenumber of bin m: teams 0 and 2 together
      named_bar(4, 2 * C::TEAM);
      const cplx<T>* ls = lines;
      const cplx<T>* lg = lines + 2 * C::LS;
      const cplx<T> zg0 = lg[0];                   // Zgy(0) = Gy~(0, y_A) + i Gy~(0, y_B)
      for (int mx = (f >> 1) * C::TEAM + t; mx < Wx; mx += 2 * C::TEAM) {
        const int qp = t3_pad(mx), qm = t3_pad((NX - mx) & (NX - 1));
        const T kx = dkx * (T)mx;
        const cplx<T> zp = ls[qp] + kx * mul_i(lg[qp]);
        const cplx<T> zm = conj(ls[qm] + (-kx) * mul_i(lg[qm]));
        cplx<T> sa = (T)0.5 * (zp + zm), sb = (T)0.5 * mul_ni(zp - zm);
        if (mx == 0) {                // real numbers S'~(0,y) and Gy~(0,y) travel together (k_fwd_row_fused)
          sa = mk<T>(sa.x, zg0.x);
          sb = mk<T>(sb.x, zg0.y);
        }
        st_pair(byte_off(outA, mo) + inter_pair_index(g, a, p, mx), sa, sb);
      }
      named_bar(4, 2 * C::TEAM);                   // lines 0 and 2 are free for the next row pair
    }
  }
}

}  // namespace ttsh
