// row_step.cuh — the whole row half of one Euler step in ONE kernel (conservative advection form, 1/2 rule):
//
//   inverse row pass of w~, v_x~, psi~ (C2R, a2 + a6)  ->  rhs of Algorithm 1 lines 1-2 (a3)  ->  forward row pass (R2C, a4)
//
// All three operate on whole rows, and a thread of the Stockham transform owns the same 16 x-positions at the output of
// an inverse transform as at the input of a forward one, so w, v_x, v_y never leave the SM: per row pair
// (y_A = 4a+p, y_B = y_A+2, packed as z = f(y_A) + i f(y_B)) the kernel reads three pruned intermediates and K and
// writes the two pruned intermediates  A~ = i k_x Gy~ + S'~  and  B~ = Gx~  (fft_passes.cuh, k_fwd_row_fused):
//   Gx = rhs1_x + lambda0 v_y w,  Gy = rhs1_y - lambda0 v_x w,  S' = -gamma_w K w,  rhs1 = -(beta |v|^2 + gamma_v K) v
// (PAPER.md:292-294, lines 1-3 of Algorithm 1 with lambda0 v.grad w = lambda0 div(v w)).
// HBM traffic per step for the row half: 3 x 0.5 U + 1 U (K) in, 2 x 0.5 U out = 3.5 U instead of 9.5 U for
// k_inv_row + k_fwd_row_fused.  Of the three packed fields one waits in shared memory (stash, [slot][thread], touched
// by its owner thread only), one in registers (H) and one is the live transform (V).
//
// Inputs arrive by asynchronous bulk copies (cp.async.bulk + mbarrier, fft_core.cuh) into two staging slots per line, each
// issued one phase ahead by the line's first thread right after the barrier that ends the previous use of the slot:
//   slot 0:  w~  ->  psi~  ->  K(y_B)  ->  w~ of the next row pair        slot 1:  v_x~  ->  K(y_A)  ->  v_x~ of the next row pair
// so no thread ever waits on a global load; the first-stage loaders and the pointwise phase read shared memory.
//
// For Nx = 4096 (where fft_wl_supported) the transforms use the warp-local plan of fft_core.cuh (one CTA-wide exchange per transform);
// the thread then owns x = wl_j(j) + k TPL, K is read from its thread-order copy (perm_index_wl) and tabX is the
// warp-local twiddle table.
// Packing by rows (f(y_A) + i f(y_B)) makes i k_x commute with the packing, so A~ is formed BEFORE the unpack:
//   T(m) = i k_m Zgy(m) + Zs(m),  k_m the signed wavenumber of bin m  ->  2 unpacks for 3 transforms.
#pragma once
#include "fft_passes.cuh"

namespace ttsh {

// row pairs per CTA of the ensemble variant: lines of small grids have few threads (Nx = 64: 4), so a CTA takes several
// consecutive row pairs of one member (64 threads; shared memory per thread does not depend on Nx, about 4 such CTAs per SM)
template <int NX> __host__ __device__ constexpr int row_step_ens_lines() { return NX >= 1024 ? 1 : 1024 / NX; }

// TAN: the tangent-linear variant (ttsh_tangent_step): its pointwise stage reads the base fields w, v_x, v_y from the internal real
// fields (row layout perm_index: x = j + k TPL), so it always runs the plain Stockham plan, whose threads own exactly those points.
template <typename T, int NX, int LL = 1, bool TAN = false> struct RowStepCfg {
  using R = RowCfg<T, NX>;
  static constexpr bool WL = fft_wl_supported<NX>() && !TAN;           // warp-local FFT plan (fft_core.cuh)
  // one row pair per CTA: for Nx <= 2048 several small CTAs share an SM and drift apart (measured +2-10 % over two
  // row pairs per CTA, which pass every barrier together)
  static constexpr int TPL = R::TPL, L = LL, THREADS = LL * TPL;
  static constexpr int LS = WL ? fft_wl_line_elems<T, NX>() + 4 : R::LS;
  static constexpr int ST = NX;                                        // stash elements per line
  // staging slot (bytes): one row pair of an inverse intermediate, 2 Wxp <= 2 (NX/4 + 8) complex values, or one row of K
  static constexpr int SLOT = ((NX / 4 + 8) * 2 * (int)sizeof(cplx<T>) + 127) / 128 * 128;
  static constexpr size_t OFF_SLOTS = ((size_t)L * (LS + ST) * sizeof(cplx<T>) + 127) / 128 * 128;
  static constexpr size_t OFF_BARS = OFF_SLOTS + (size_t)L * 2 * SLOT;
  // warp-local plan: a copy of its twiddle table lives in shared memory (fft_core.cuh explains why)
  static constexpr size_t OFF_TAB = (OFF_BARS + (size_t)L * 2 * sizeof(unsigned long long) + 15) / 16 * 16;
  // fp64 only (C5: k_row_step 258.3 -> 253.5 us); in fp32 the L1 next to 101 KB of shared memory holds the 13 KB table and the
  // copy only adds shared-memory wavefronts (137.0 us from global memory, 145.6 us from the copy)
  static constexpr bool SMEM_TAB = WL && sizeof(T) == 8;
  static constexpr size_t SMEM = OFF_TAB + (SMEM_TAB ? (size_t)fft_wl_tw_elems_rt(NX) * sizeof(cplx<T>) : 0);
  static constexpr int MINB = 1;          // one CTA per SM also in fp32 at Nx = 4096 (two CTAs of 128 registers: 140 vs 136 us)
  static constexpr bool FITS = SMEM <= 227 * 1024;
};

// (A, B) pair / 4 consecutive scalars from a staging slot.  fp64: 32 bytes per lane as two LDS.128 whose order is swapped
// on lanes with bit 2 set, so that the 8 lanes of a wavefront cover all banks (lane stride 32 bytes would otherwise be a
// 2-way conflict).  fp32: one LDS.128.
__device__ __forceinline__ Pair<double> lds_pair(const cplx<double>* p, int sw) {
  const double2 u = *reinterpret_cast<const double2*>(p + sw), v = *reinterpret_cast<const double2*>(p + (sw ^ 1));
  Pair<double> r;
  r.a = sw ? mk<double>(v.x, v.y) : mk<double>(u.x, u.y);
  r.b = sw ? mk<double>(u.x, u.y) : mk<double>(v.x, v.y);
  return r;
}
__device__ __forceinline__ Pair<float> lds_pair(const cplx<float>* p, int) {
  const float4 u = *reinterpret_cast<const float4*>(p);
  Pair<float> r;
  r.a = mk<float>(u.x, u.y);
  r.b = mk<float>(u.z, u.w);
  return r;
}
__device__ __forceinline__ Quad<double> lds_quad(const double* p, int sw) {
  const double2 u = *reinterpret_cast<const double2*>(p + 2 * sw), v = *reinterpret_cast<const double2*>(p + 2 * (sw ^ 1));
  Quad<double> r;
  r.v[0] = sw ? v.x : u.x; r.v[1] = sw ? v.y : u.y; r.v[2] = sw ? u.x : v.x; r.v[3] = sw ? u.y : v.y;
  return r;
}
__device__ __forceinline__ Quad<float> lds_quad(const float* p, int) {
  const float4 u = *reinterpret_cast<const float4*>(p);
  Quad<float> r;
  r.v[0] = u.x; r.v[1] = u.y; r.v[2] = u.z; r.v[3] = u.w;
  return r;
}

// inverse row transform of one packed row pair into registers: out[k] = f(y_A, x) + i f(y_B, x), x = j + k TPL.
// row: the staged pairs of this row pair in shared memory ((A, B) of column mx at row + 2 mx).
// MODE = RM_ONE or RM_NIKX_MEANY (ttsh_common.cuh).  1/2 rule only: retained mx = 0..NX/4.
// With the warp-local plan the thread owns x = wl_j(j) + k TPL instead (tabX is then the warp-local table).
template <typename T, int NX, int MODE, bool WL, class Hook>
__device__ __forceinline__ void inv_row_regs(const cplx<T>* __restrict__ row, int j, cplx<T>* __restrict__ line,
                                             const cplx<T>* __restrict__ tabX, T scale, T dkx, T meany, cplx<T> (&out)[16],
                                             Hook hook) {
  const int sw = (j >> 2) & 1;
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
    if (k <= 3 || (k == 4 && j == 0)) return lds_pair(row + 2 * m, sw);
    if (k >= 12) return lds_pair(row + 2 * (NX - m), sw);
    return zero_pair();
  };
  auto finish = [&](int m, int k, Pair<T> r) -> cplx<T> {
    if (k <= 3) return combine(r, m, false);
    if (k == 4) return j == 0 ? combine(r, m, false) : mk<T>(0, 0);
    if (k >= 12) return combine(r, NX - m, true);
    return mk<T>(0, 0);
  };
  auto store = [&](int, int k, cplx<T> z) { out[k] = z; };
  if constexpr (WL) fft_line_wl<T, NX, +1, false>(j, j, line, tabX, make_loader<1>(issue, finish), store, hook);
  else fft_line<T, NX, +1, false>(j, line, tabX, make_loader<1>(issue, finish), store, hook);
}

// forward transform of the 16 values a thread owns (slot k <-> x = jw + k TPL; jw = wl_j(j) for the warp-local plan, else j)
template <typename T, int NX, bool SYNC_LAST, bool WL, class Load, class Store, class Hook = NoHook>
__device__ __forceinline__ void fwd_row_regs(int jw, int j, cplx<T>* __restrict__ line, const cplx<T>* __restrict__ tabX, Load load,
                                             Store store, Hook hook = Hook()) {
  if constexpr (WL) fft_line_wl<T, NX, -1, SYNC_LAST>(jw, j, line, tabX, load, store, hook);
  else fft_line<T, NX, -1, SYNC_LAST>(j, line, tabX, load, store, hook);
}
template <typename T, int NX, bool WL> __device__ __forceinline__ int row_step_pad(int i) {
  if constexpr (WL) return fft_wl_pad<T, NX>(i);
  else return fft_pad<NX>(i);
}

template <class P> __device__ __forceinline__ P* byte_off(P* p, size_t bytes) {
  return reinterpret_cast<P*>(reinterpret_cast<char*>(const_cast<typename std::remove_const<P>::type*>(p)) + bytes);
}

// LL row pairs per CTA.  ENS: the persistent grid runs over the row pairs of `members` systems whose workspaces lie mstride
// bytes apart (ttsh_ensemble_step); rpm = Ny/2 row pairs per member, a multiple of LL, so a CTA's lines share a member.
// TAN (with ENS: the members are the tangent vectors): inW / inVx / inPsi / outA / outB / v0 belong to the perturbation (dw~, dv_x~,
// dpsi~; per vector, mstride apart), K and the base fields bw, bvx, bvy (internal real fields of the handle) are shared, and the
// pointwise stage evaluates the derivative of lines 1-2 at the base state (pointwise.cuh, k_realspace_tangent).
template <typename T, int NX, int LL, bool ENS, bool TAN = false>
__global__ void __launch_bounds__(RowStepCfg<T, NX, LL, TAN>::THREADS, RowStepCfg<T, NX, LL, TAN>::MINB)
k_row_step(const __grid_constant__ Geom g, const __grid_constant__ Model m, const cplx<T>* __restrict__ inW,
           const cplx<T>* __restrict__ inVx, const cplx<T>* __restrict__ inPsi, const T* __restrict__ K,
           cplx<T>* __restrict__ outA, cplx<T>* __restrict__ outB, const cplx<T>* __restrict__ tabX,
           const double* __restrict__ v0, int nblk, int rpm, size_t mstride, const T* __restrict__ bw, const T* __restrict__ bvx,
           const T* __restrict__ bvy) {
  using C = RowStepCfg<T, NX, LL, TAN>;
  static_assert(!TAN || ENS, "the tangent variant runs over the vectors as members");
  constexpr int TPL = C::TPL;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int c = threadIdx.x / TPL, j = threadIdx.x % TPL;
  const int jw = C::WL ? (j >> 4) + (NX / 256) * (j & 15) : j;       // the x-class this thread owns: x = jw + k TPL
  cplx<T>* line = sm + c * C::LS;
  cplx<T>* stash = sm + C::L * C::LS + c * C::ST + j;      // slot k of this thread at stash[k TPL]
  unsigned char* slot0 = smem_raw + C::OFF_SLOTS + (size_t)(2 * c) * C::SLOT;
  unsigned char* slot1 = slot0 + C::SLOT;
  unsigned long long* bar0 = reinterpret_cast<unsigned long long*>(smem_raw + C::OFF_BARS) + 2 * c;
  unsigned long long* bar1 = bar0 + 1;
  const int Wx = g.Wx;
  const T scale_i = (T)g.inv_sqrt_nx, scale_f = (T)g.inv_sqrt_nx;
  const T dkx = (T)g.dkx;
  T meany = (T)0;                                            // v^_y(0) / sqrt(Ny): read after pdl_wait (the predecessor writes v0)
  // global row pair -> (row pair of its member, byte offset of the member's workspace)
  auto locate = [&](int rpg, int& rp_, size_t& mo_) {
    if constexpr (ENS) { const int mb = rpg / rpm; rp_ = rpg - mb * rpm; mo_ = (size_t)mb * mstride; }
    else { rp_ = rpg; mo_ = 0; }
  };
  const T beta = (T)m.beta, gv = (T)m.gamma_v, lam = (T)m.lambda0;
  const T ngw = -(T)m.gamma_w * scale_f;
  const size_t in_stride = (size_t)g.Wxp * 2;               // elements per row pair of an inverse intermediate
  const unsigned in_bytes = (unsigned)(in_stride * sizeof(cplx<T>)), k_bytes = (unsigned)(NX * sizeof(T));
  const bool leader = (j == 0);
  unsigned ph0 = 0, ph1 = 0;                                 // phase parity of the next completion of each slot's barrier

  if (leader) { mbar_init(bar0, 1); mbar_init(bar1, 1); }
  mbar_fence_init();
  if constexpr (C::SMEM_TAB) {      // twiddle table -> shared memory (host-written at ttsh_create: no dependence on the preceding launch)
    cplx<T>* stab = reinterpret_cast<cplx<T>*>(smem_raw + C::OFF_TAB);
    for (int i = threadIdx.x; i < fft_wl_tw_elems_rt(NX); i += C::THREADS) stab[i] = ldg_c(tabX + i);
    tabX = stab;
  }
  __syncthreads();
  pdl_wait();          // inputs, K and v0 below are written by the preceding launches
  pdl_trigger();
  if constexpr (!ENS) meany = (T)(v0[1] * g.inv_sqrt_ny);
  if (leader && (int)blockIdx.x < nblk) {
    int rp0; size_t mo0;
    locate(blockIdx.x * C::L + c, rp0, mo0);
    bulk_load(slot0, byte_off(inW, mo0) + (size_t)rp0 * in_stride, in_bytes, bar0);
    bulk_load(slot1, byte_off(inVx, mo0) + (size_t)rp0 * in_stride, in_bytes, bar1);
  }

#pragma unroll 1
  for (int blk = blockIdx.x; blk < nblk; blk += gridDim.x) {
    int rp; size_t mo;
    locate(blk * C::L + c, rp, mo);
    if constexpr (ENS) meany = (T)(byte_off(v0, mo)[1] * g.inv_sqrt_ny);
    const int a = rp >> 1, p = rp & 1;
    const size_t offA = (size_t)(4 * a + p) * NX, offB = offA + 2 * (size_t)NX;
    const size_t kmo = TAN ? 0 : mo;                    // K is shared by all tangent vectors
    const int nb = blk + gridDim.x;
    if (leader && nb < nblk) {   // L2 prefetch of what this line reads in the CTA's next iteration
      int nrp; size_t nmo;
      locate(nb * C::L + c, nrp, nmo);
      prefetch_l2_bulk(byte_off(inW, nmo) + (size_t)nrp * in_stride, in_bytes);
      prefetch_l2_bulk(byte_off(inVx, nmo) + (size_t)nrp * in_stride, in_bytes);
      prefetch_l2_bulk(byte_off(inPsi, nmo) + (size_t)nrp * in_stride, in_bytes);
      const size_t nA = (size_t)(4 * (nrp >> 1) + (nrp & 1)) * NX;
      const size_t nkmo = TAN ? 0 : nmo;
      prefetch_l2_bulk(byte_off(K, nkmo) + nA, k_bytes);
      prefetch_l2_bulk(byte_off(K, nkmo) + nA + 2 * (size_t)NX, k_bytes);
      if constexpr (TAN) {   // the six base rows of the next row pair
        prefetch_l2_bulk(bw + nA, k_bytes); prefetch_l2_bulk(bw + nA + 2 * (size_t)NX, k_bytes);
        prefetch_l2_bulk(bvx + nA, k_bytes); prefetch_l2_bulk(bvx + nA + 2 * (size_t)NX, k_bytes);
        prefetch_l2_bulk(bvy + nA, k_bytes); prefetch_l2_bulk(bvy + nA + 2 * (size_t)NX, k_bytes);
      }
    }
    cplx<T> H[16], V[16];
    // ---- a2 / a6: w, v_x, v_y of the two rows ----
    mbar_wait(bar0, ph0); ph0 ^= 1;
    inv_row_regs<T, NX, RM_ONE, C::WL>(reinterpret_cast<const cplx<T>*>(slot0), j, line, tabX, scale_i, dkx, meany, V,
                                [&]() { if (leader) bulk_load(slot0, byte_off(inPsi, mo) + (size_t)rp * in_stride, in_bytes, bar0); });
#pragma unroll
    for (int k = 0; k < 16; ++k) stash[k * TPL] = V[k];                     // w
    mbar_wait(bar1, ph1); ph1 ^= 1;
    inv_row_regs<T, NX, RM_ONE, C::WL>(reinterpret_cast<const cplx<T>*>(slot1), j, line, tabX, scale_i, dkx, meany, H,
                                [&]() { if (leader) bulk_load(slot1, byte_off(K, kmo) + offA, k_bytes, bar1); });             // v_x
    mbar_wait(bar0, ph0); ph0 ^= 1;
    inv_row_regs<T, NX, RM_NIKX_MEANY, C::WL>(reinterpret_cast<const cplx<T>*>(slot0), j, line, tabX, scale_i, dkx, meany, V,
                                       [&]() { if (leader) bulk_load(slot0, byte_off(K, kmo) + offB, k_bytes, bar0); });      // v_y
    // ---- a3: lines 1-2 of Algorithm 1, pointwise;  V <- Gx,  H <- Gy,  stash <- S'  (all scaled for the forward pass) ----
    mbar_wait(bar1, ph1); ph1 ^= 1;
    mbar_wait(bar0, ph0); ph0 ^= 1;
    {
      const int sw = (j >> 2) & 1;
      const T* KA = reinterpret_cast<const T*>(slot1);
      const T* KB = reinterpret_cast<const T*>(slot0);
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const Quad<T> ka = lds_quad(KA + (q * TPL + j) * 4, sw), kb = lds_quad(KB + (q * TPL + j) * 4, sw);
        if constexpr (TAN) {
          // derivative of lines 1-2 at the base state (u, v, om): with c = -beta (u^2 + v^2) - gamma_v K, dc = -2 beta (u du + v dv),
          //   dGx = dc u + c du + lambda0 (dv om + v dom),  dGy = dc v + c dv - lambda0 (du om + u dom),  dS' = -gamma_w K dom
          // one row at a time (three base quads in flight instead of six: the stage runs at the register limit)
          const size_t e = (size_t)(q * TPL + j) * 4;
#pragma unroll
          for (int r = 0; r < 2; ++r) {
            const size_t off = (r ? offB : offA) + e;
            const Quad<T> om = ld_quad(bw + off), u = ld_quad(bvx + off), v = ld_quad(bvy + off);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const int k = 4 * q + i;
              T* sp = reinterpret_cast<T*>(stash + k * TPL) + r;            // dw of row r, then dS' of row r
              const T kk = r ? kb.v[i] : ka.v[i], dom = *sp;
              const T du = r ? H[k].y : H[k].x, dv = r ? V[k].y : V[k].x;
              const T c = -beta * (u.v[i] * u.v[i] + v.v[i] * v.v[i]) - gv * kk;
              const T dc = (T)-2 * beta * (u.v[i] * du + v.v[i] * dv);
              const T gx = scale_f * (dc * u.v[i] + c * du + lam * (dv * om.v[i] + v.v[i] * dom));
              const T gy = scale_f * (dc * v.v[i] + c * dv - lam * (du * om.v[i] + u.v[i] * dom));
              if (r) { V[k].y = gx; H[k].y = gy; } else { V[k].x = gx; H[k].x = gy; }
              *sp = ngw * (kk * dom);
            }
          }
        } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int k = 4 * q + i;
          const cplx<T> w = stash[k * TPL];
          const T kA = ka.v[i], kB = kb.v[i];
          const T vxA = H[k].x, vxB = H[k].y, vyA = V[k].x, vyB = V[k].y;
          const T ccA = scale_f * (-beta * (vxA * vxA + vyA * vyA) - gv * kA);
          const T ccB = scale_f * (-beta * (vxB * vxB + vyB * vyB) - gv * kB);
          const T lwA = scale_f * lam * w.x, lwB = scale_f * lam * w.y;
          V[k] = mk<T>(ccA * vxA + lwA * vyA, ccB * vxB + lwB * vyB);          // Gx
          H[k] = mk<T>(ccA * vyA - lwA * vxA, ccB * vyB - lwB * vxB);          // Gy
          stash[k * TPL] = mk<T>(ngw * (kA * w.x), ngw * (kB * w.y));          // S'
        }
        }
      }
    }
    // ---- a4, transform 1: Gx -> B~ (its first barrier frees both slots: stage the next row pair) ----
    auto keep = [&](int k) -> bool { return k <= 3 || k >= 12 || (k == 4 && j == 0); };
    auto ident = [&](int, int, cplx<T> r) -> cplx<T> { return r; };
    {
      auto store = [&](int mm, int k, cplx<T> z) { if (keep(k)) line[row_step_pad<T, NX, C::WL>(mm)] = z; };
      fwd_row_regs<T, NX, true, C::WL>(jw, j, line, tabX, make_loader<1>([&](int, int k) -> cplx<T> { return V[k]; }, ident), store, [&]() {
        if (leader && nb < nblk) {
          int nrp; size_t nmo;
          locate(nb * C::L + c, nrp, nmo);
          bulk_load(slot0, byte_off(inW, nmo) + (size_t)nrp * in_stride, in_bytes, bar0);
          bulk_load(slot1, byte_off(inVx, nmo) + (size_t)nrp * in_stride, in_bytes, bar1);
        }
      });
      __syncthreads();
      for (int mx = j; mx < Wx; mx += TPL) {
        const cplx<T> zp = line[row_step_pad<T, NX, C::WL>(mx)];
        const cplx<T> zm = conj(line[row_step_pad<T, NX, C::WL>((NX - mx) & (NX - 1))]);
        st_pair(byte_off(outB, mo) + inter_pair_index(g, a, p, mx), (T)0.5 * (zp + zm), (T)0.5 * mul_ni(zp - zm));
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
      fwd_row_regs<T, NX, false, C::WL>(jw, j, line, tabX, make_loader<1>([&](int, int k) -> cplx<T> { return H[k]; }, ident), store);
    }
    // ---- transform 3: S' -> A~ = unpack(i k_m Zgy + Zs) ----
    {
      auto store = [&](int mm, int k, cplx<T> z) { if (keep(k)) line[row_step_pad<T, NX, C::WL>(mm)] = z + H[k]; };
      fwd_row_regs<T, NX, true, C::WL>(jw, j, line, tabX, make_loader<1>([&](int, int k) -> cplx<T> { return stash[k * TPL]; }, ident), store);
      __syncthreads();
      for (int mx = j; mx < Wx; mx += TPL) {
        const cplx<T> zp = line[row_step_pad<T, NX, C::WL>(mx)];
        const cplx<T> zm = conj(line[row_step_pad<T, NX, C::WL>((NX - mx) & (NX - 1))]);
        cplx<T> sa = (T)0.5 * (zp + zm), sb = (T)0.5 * mul_ni(zp - zm);
        if (mx == 0) {                // real numbers S'~(0,y) and Gy~(0,y) travel together (k_fwd_row_fused)
          sa = mk<T>(sa.x, zg0.x);
          sb = mk<T>(sb.x, zg0.y);
        }
        st_pair(byte_off(outA, mo) + inter_pair_index(g, a, p, mx), sa, sb);
      }
    }
  }
}

}  // namespace ttsh
