// fft_core.cuh — shared-memory Stockham autosort FFT of one line, radix-16/8/4 butterflies in registers.
//
// A line of length N is transformed cooperatively by TPL = N/16 threads; every thread owns 16 complex
// points per stage (one radix-16, two radix-8 or four radix-4 butterflies).  Stage s (radix R, Ns = product
// of the earlier radices) does, for butterfly j in [0, N/R):
//     k = j mod Ns;   v[r] = in[j + r N/R] * W_{Ns R}^{k r};   v = DFT_R(v);   out[(j-k) R + k + r Ns] = v[r]
// The first stage reads through a caller-supplied functor (global memory, with whatever multiplier or
// packing the pass needs) and the last stage writes through one, so a line makes one trip through
// shared memory per stage boundary only.  Shared-memory indices are padded (i + i >> log2(R0)) so that both
// the stride-R0 writes of the first stage and the unit-stride reads are bank-conflict free for 8- and 16-byte
// elements.  DIR = -1: forward (e^{-i...}), DIR = +1: inverse.  No normalisation here.
#pragma once
#include "ttsh_common.cuh"
#include <type_traits>

namespace ttsh {

// ---------------------------------------------------------------------------------------
// radix plans.  nstages / radix are constexpr so that they can be template arguments.
// ---------------------------------------------------------------------------------------
__host__ __device__ constexpr int fft_nstages_rt(int N) { return N <= 256 ? 2 : (N <= 4096 ? 3 : 4); }
__host__ __device__ constexpr int fft_radix_rt(int N, int s) {
  switch (N) {
    case 32:   return s == 0 ? 8 : 4;
    case 64:   return 8;
    case 128:  return s == 0 ? 16 : 8;
    case 256:  return 16;
    case 512:  return 8;
    case 1024: return s == 0 ? 16 : 8;
    case 2048: return s <= 1 ? 16 : 8;
    case 4096: return 16;
    case 8192: return s == 0 ? 16 : 8;
    default:   return 0;
  }
}
template <int N> __host__ __device__ constexpr int fft_nstages() { return fft_nstages_rt(N); }
template <int N> __host__ __device__ constexpr int fft_radix(int s) { return fft_radix_rt(N, s); }
// Per-stage twiddle tables.  Stage s >= 1 (radix R, Ns) needs w^r, r = 1..R-1, with w = W_{Ns R}^k, k = j mod Ns.  Only a
// base set is stored and loaded — R=16: w^1, w^2, w^3, w^4, w^8, w^12;  R=8: w^1..w^4;  R=4: w^1..w^3 — laid out
// [base][k] so that consecutive threads read consecutive entries (one coalesced request per base power); the other
// powers are one complex product each (w^{4a+b} = w^{4a} w^b), which keeps every twiddle within ~1.5 ulp and takes the
// twiddle traffic through L1 from 15 to 6 requests per radix-16 butterfly (L1 wavefronts were the top unit in ncu).
__host__ __device__ constexpr int fft_tw_nbase(int R) { return R == 16 ? 6 : (R == 8 ? 4 : R - 1); }
__host__ __device__ constexpr int fft_tw_base_power(int R, int b) { return (R == 16 && b >= 3) ? 4 * (b - 2) : b + 1; }
__host__ __device__ constexpr int fft_tw_offset_rt(int N, int s) {
  int off = 0, ns = fft_radix_rt(N, 0);
  for (int t = 1; t < s; ++t) { off += fft_tw_nbase(fft_radix_rt(N, t)) * ns; ns *= fft_radix_rt(N, t); }
  return off;
}
__host__ __device__ constexpr int fft_tw_elems_rt(int N) { return fft_tw_offset_rt(N, fft_nstages_rt(N)); }
template <int N> __host__ __device__ constexpr int fft_tpl() { return N / 16; }
template <int N> __host__ __device__ constexpr int fft_padshift() { return fft_radix<N>(0) == 16 ? 4 : 3; }
template <int N> __host__ __device__ constexpr int fft_line_elems() { return N + (N >> fft_padshift<N>()); }
template <int N> __device__ __forceinline__ int fft_pad(int i) { return i + (i >> fft_padshift<N>()); }

// ---------------------------------------------------------------------------------------
// small DFTs in registers.  Outputs in natural order.
// ---------------------------------------------------------------------------------------
template <int DIR, typename T> __device__ __forceinline__ cplx<T> mul_w4(cplx<T> a) {   // a * W_4^1
  return DIR < 0 ? mul_ni(a) : mul_i(a);
}

template <int DIR, typename T> __device__ __forceinline__ void dft2(cplx<T>& a, cplx<T>& b) {
  cplx<T> t = a - b; a = a + b; b = t;
}

template <int DIR, typename T>
__device__ __forceinline__ void dft4(cplx<T>& a0, cplx<T>& a1, cplx<T>& a2, cplx<T>& a3) {
  cplx<T> t0 = a0 + a2, t1 = a0 - a2, t2 = a1 + a3, t3 = mul_w4<DIR>(a1 - a3);
  a0 = t0 + t2; a1 = t1 + t3; a2 = t0 - t2; a3 = t1 - t3;
}

// a * W_8^n and a * W_16^n with compile-time n (DIR-aware); constants are exact to 0.5 ulp in double
template <int DIR, int n, typename T> __device__ __forceinline__ cplx<T> mul_w8(cplx<T> a) {
  constexpr T h = (T)0.70710678118654752440084436210485;
  if (n == 0) return a;
  if (n == 2) return mul_w4<DIR>(a);
  if (n == 1) return DIR < 0 ? mk<T>(h * (a.x + a.y), h * (a.y - a.x)) : mk<T>(h * (a.x - a.y), h * (a.y + a.x));
  /* n == 3 */ return DIR < 0 ? mk<T>(h * (a.y - a.x), -h * (a.x + a.y)) : mk<T>(-h * (a.x + a.y), h * (a.x - a.y));
}
template <int DIR, int n, typename T> __device__ __forceinline__ cplx<T> mul_w16(cplx<T> a) {
  // W_16^n = cos(n pi/8) + DIR * i sin(n pi/8), n = 0..9
  constexpr T c1 = (T)0.92387953251128675612818318939679, s1 = (T)0.38268343236508977172845998403040;
  if (n % 2 == 0) return mul_w8<DIR, n / 2>(a);
  T c = (n == 1) ? c1 : (n == 3) ? s1 : (n == 5) ? -s1 : (n == 7) ? -c1 : -c1;
  T s = (n == 1) ? s1 : (n == 3) ? c1 : (n == 5) ? c1 : (n == 7) ? s1 : -s1;   // n == 9: (-c1, -s1)
  s = DIR < 0 ? -s : s;
  return mk<T>(a.x * c - a.y * s, a.x * s + a.y * c);
}

// a * W_32^k, k = 0..15 (compile-time k): the split twiddles of the column passes factor as W_Ny^{j + k Ny/32} = W_Ny^j W_32^k
template <int DIR, int k, typename T> __device__ __forceinline__ cplx<T> mul_w32(cplx<T> a) {
  constexpr double C[16] = {1.0000000000000000000000000000000000, 0.9807852804032304491261822361342390, 0.9238795325112867561281831893967883, 0.8314696123025452370787883776179058, 0.7071067811865475244008443621048490, 0.5555702330196022247428308139485329, 0.3826834323650897717284599840303989, 0.1950903220161282678482848684770222, 0.0000000000000000000000000000000000, -0.1950903220161282678482848684770222, -0.3826834323650897717284599840303989, -0.5555702330196022247428308139485329, -0.7071067811865475244008443621048490, -0.8314696123025452370787883776179058, -0.9238795325112867561281831893967883, -0.9807852804032304491261822361342390};
  constexpr double S[16] = {0.0000000000000000000000000000000000, 0.1950903220161282678482848684770222, 0.3826834323650897717284599840303989, 0.5555702330196022247428308139485329, 0.7071067811865475244008443621048490, 0.8314696123025452370787883776179058, 0.9238795325112867561281831893967883, 0.9807852804032304491261822361342390, 1.0000000000000000000000000000000000, 0.9807852804032304491261822361342390, 0.9238795325112867561281831893967883, 0.8314696123025452370787883776179058, 0.7071067811865475244008443621048490, 0.5555702330196022247428308139485329, 0.3826834323650897717284599840303989, 0.1950903220161282678482848684770222};
  if constexpr (k == 0) return a;
  else if constexpr (k == 8) return mul_w4<DIR>(a);
  else {
    constexpr T c = (T)C[k], s = (T)(DIR < 0 ? -S[k] : S[k]);
    return mk<T>(a.x * c - a.y * s, a.x * s + a.y * c);
  }
}
template <int DIR, typename T> __device__ __forceinline__ cplx<T> mul_w32_rt(cplx<T> a, int k) {   // k constant after unrolling
  switch (k) {
#define TTSH_W32(K) case K: return mul_w32<DIR, K>(a);
    TTSH_W32(0) TTSH_W32(1) TTSH_W32(2) TTSH_W32(3) TTSH_W32(4) TTSH_W32(5) TTSH_W32(6) TTSH_W32(7)
    TTSH_W32(8) TTSH_W32(9) TTSH_W32(10) TTSH_W32(11) TTSH_W32(12) TTSH_W32(13) TTSH_W32(14) TTSH_W32(15)
#undef TTSH_W32
  }
  return a;
}

template <int DIR, typename T> __device__ __forceinline__ void dft8(cplx<T>* v) {
  // s = 2 s1 + s2, r = r1 + 4 r2:  W_8^{rs} = W_4^{r1 s1} W_8^{r1 s2} W_2^{r2 s2}
  dft4<DIR>(v[0], v[2], v[4], v[6]);
  dft4<DIR>(v[1], v[3], v[5], v[7]);
  v[3] = mul_w8<DIR, 1>(v[3]);
  v[5] = mul_w8<DIR, 2>(v[5]);
  v[7] = mul_w8<DIR, 3>(v[7]);
  // v[2 r1] = y[0][r1], v[2 r1 + 1] = y[1][r1]
  cplx<T> o[8];
#pragma unroll
  for (int r1 = 0; r1 < 4; ++r1) {
    o[r1] = v[2 * r1] + v[2 * r1 + 1];
    o[r1 + 4] = v[2 * r1] - v[2 * r1 + 1];
  }
#pragma unroll
  for (int r = 0; r < 8; ++r) v[r] = o[r];
}

template <int DIR, typename T> __device__ __forceinline__ void dft16(cplx<T>* v) {
  // s = 4 s1 + s2, r = r1 + 4 r2:  W_16^{rs} = W_4^{r1 s1} W_16^{r1 s2} W_4^{r2 s2}
#pragma unroll
  for (int s2 = 0; s2 < 4; ++s2) dft4<DIR>(v[s2], v[4 + s2], v[8 + s2], v[12 + s2]);   // v[4 r1 + s2] = y[s2][r1]
  v[5] = mul_w16<DIR, 1>(v[5]);   v[6] = mul_w16<DIR, 2>(v[6]);   v[7] = mul_w16<DIR, 3>(v[7]);
  v[9] = mul_w16<DIR, 2>(v[9]);   v[10] = mul_w16<DIR, 4>(v[10]); v[11] = mul_w16<DIR, 6>(v[11]);
  v[13] = mul_w16<DIR, 3>(v[13]); v[14] = mul_w16<DIR, 6>(v[14]); v[15] = mul_w16<DIR, 9>(v[15]);
#pragma unroll
  for (int r1 = 0; r1 < 4; ++r1) dft4<DIR>(v[4 * r1], v[4 * r1 + 1], v[4 * r1 + 2], v[4 * r1 + 3]);
  // now v[4 r1 + r2] = X[r1 + 4 r2]: transpose the 4x4 index
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = a + 1; b < 4; ++b) { cplx<T> t = v[4 * a + b]; v[4 * a + b] = v[4 * b + a]; v[4 * b + a] = t; }
}

template <int R, int DIR, typename T> __device__ __forceinline__ void dftR(cplx<T>* v) {
  if (R == 16) dft16<DIR>(v);
  else if (R == 8) dft8<DIR>(v);
  else if (R == 4) dft4<DIR>(v[0], v[1], v[2], v[3]);
  else dft2<DIR>(v[0], v[1]);
}

// 64/128-bit read-only loads of a complex value
__device__ __forceinline__ cplx<double> ldg_c(const cplx<double>* p) {
  double2 t = __ldg(reinterpret_cast<const double2*>(p)); return mk<double>(t.x, t.y);
}
__device__ __forceinline__ cplx<float> ldg_c(const cplx<float>* p) {
  float2 t = __ldg(reinterpret_cast<const float2*>(p)); return mk<float>(t.x, t.y);
}

// strided loads of the column passes: ask L2 to fetch the whole 256-byte block around the 16/32/64 bytes this CTA
// needs, so that DRAM sees 256-byte granules and the neighbouring CTAs (adjacent columns, running concurrently) hit L2
__device__ __forceinline__ cplx<double> ld_l2_256(const cplx<double>* p) {
  cplx<double> r;
  asm volatile("ld.global.L2::256B.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
  return r;
}
__device__ __forceinline__ cplx<float> ld_l2_256(const cplx<float>* p) {
  cplx<float> r;
  asm volatile("ld.global.L2::256B.v2.f32 {%0, %1}, [%2];" : "=f"(r.x), "=f"(r.y) : "l"(p));
  return r;
}

// asynchronous L2 prefetch of a contiguous span (bytes: multiple of 16, address 16-byte aligned); costs no registers
// and no shared memory.  Used to pull the rows of the CTA that will run about one wave later into L2, so that its
// load phase sees L2 latency instead of DRAM latency.
__device__ __forceinline__ void prefetch_l2_bulk(const void* p, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// mbarrier + 1-D bulk asynchronous copy global -> shared (TMA unit, SASS UBLKCP): the copy is issued by one thread and
// completes on the mbarrier with its byte count; consumers wait on the barrier's phase parity.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void bulk_load(void* dst_smem, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "MBAR_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra MBAR_DONE;\n"
      "bra MBAR_WAIT;\n"
      "MBAR_DONE:\n"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

// twiddle W_M^p from the forward-sign table (M = table length), conjugated for the inverse
template <int DIR, typename T> __device__ __forceinline__ cplx<T> twiddle(const cplx<T>* __restrict__ tab, int p) {
  cplx<T> w = ldg_c(tab + p);
  return DIR < 0 ? w : conj(w);
}

// loader = { issue(idx, k) -> Raw (global/shared loads only), finish(idx, k, Raw) -> cplx<T> } with idx = j + k TPL;
// the slot k = 0..15 is a compile-time constant after unrolling, so loaders can prune by k at compile time
template <int B, class I, class F> struct Loader {
  static constexpr int BATCHES = B;
  static constexpr int VEC = 1;
  I issue;
  F finish;
};
template <int B = 1, class I, class F> __device__ __forceinline__ Loader<B, I, F> make_loader(I i, F f) {
  return Loader<B, I, F>{i, f};
}
// vector loader: issue(k0, Raw* out) fills the 4 consecutive slots k0..k0+3 (k0 a multiple of 4) with wide loads
template <int B, class Raw, class I, class F> struct VecLoader {
  static constexpr int BATCHES = B;
  static constexpr int VEC = 4;
  using raw_t = Raw;
  I issue;
  F finish;
};
template <int B, class Raw, class I, class F> __device__ __forceinline__ VecLoader<B, Raw, I, F> make_vec_loader(I i, F f) {
  return VecLoader<B, Raw, I, F>{i, f};
}
// vector store of the last stage: f(k0, const cplx<T>* v4) receives the 4 consecutive slots k0..k0+3
template <class F> struct VecStore { F f; };
template <class F> __device__ __forceinline__ VecStore<F> make_vec_store(F f) { return VecStore<F>{f}; }
template <class S> struct is_vec_store : std::false_type {};
template <class F> struct is_vec_store<VecStore<F>> : std::true_type {};
// fire-and-forget accumulation  *p += v  (two scalar reductions; each address receives exactly one addend per pass,
// so the result does not depend on ordering).  No "memory" clobber on purpose: the asm is volatile (never dropped),
// the preceding plain store of the same thread to the same address is separated from it by a __syncthreads, and a
// clobber would stop ptxas from hoisting the twiddle loads of the neighbouring outputs above it.
__device__ __forceinline__ void red_add(cplx<double>* p, cplx<double> v) {
  asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&p->x), "d"(v.x));
  asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&p->y), "d"(v.y));
}
__device__ __forceinline__ void red_add(cplx<float>* p, cplx<float> v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(&p->x), "f"(v.x));
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(&p->y), "f"(v.y));
}

// stage twiddles: the base powers stored at tw[b * ns] are loaded first (TwBase), v[r] *= w^r, r = 1..R-1, is applied later, so
// that the table loads are in flight together with the shared-memory reads of the stage
template <int R, typename T> struct TwBase { cplx<T> w[fft_tw_nbase(R)]; };
template <int R, int DIR, typename T>
__device__ __forceinline__ TwBase<R, T> load_stage_twiddles(const cplx<T>* __restrict__ tw, int ns) {
  TwBase<R, T> b;
#pragma unroll
  for (int i = 0; i < fft_tw_nbase(R); ++i) b.w[i] = twiddle<DIR>(tw, i * ns);
  return b;
}
template <int R, typename T> __device__ __forceinline__ void apply_stage_twiddles(cplx<T>* v, const TwBase<R, T>& b) {
  if constexpr (R == 16) {
    const cplx<T> w1 = b.w[0], w2 = b.w[1], w3 = b.w[2], w4 = b.w[3], w8 = b.w[4], w12 = b.w[5];
    v[1] = v[1] * w1;   v[2] = v[2] * w2;   v[3] = v[3] * w3;   v[4] = v[4] * w4;   v[8] = v[8] * w8;   v[12] = v[12] * w12;
    v[5] = v[5] * (w4 * w1);   v[6] = v[6] * (w4 * w2);   v[7] = v[7] * (w4 * w3);
    v[9] = v[9] * (w8 * w1);   v[10] = v[10] * (w8 * w2); v[11] = v[11] * (w8 * w3);
    v[13] = v[13] * (w12 * w1); v[14] = v[14] * (w12 * w2); v[15] = v[15] * (w12 * w3);
  } else if constexpr (R == 8) {
    const cplx<T> w1 = b.w[0], w2 = b.w[1], w3 = b.w[2], w4 = b.w[3];
    v[1] = v[1] * w1; v[2] = v[2] * w2; v[3] = v[3] * w3; v[4] = v[4] * w4;
    v[5] = v[5] * (w4 * w1); v[6] = v[6] * (w4 * w2); v[7] = v[7] * (w4 * w3);
  } else {
#pragma unroll
    for (int r = 1; r < R; ++r) v[r] = v[r] * b.w[r - 1];
  }
}
template <int R, int DIR, typename T>
__device__ __forceinline__ void apply_stage_twiddles(cplx<T>* v, const cplx<T>* __restrict__ tw, int ns) {
  apply_stage_twiddles<R>(v, load_stage_twiddles<R, DIR>(tw, ns));
}

// ---------------------------------------------------------------------------------------
// one line.  j = thread index within the line's TPL threads; sm = this line's padded buffer.
// tab = the per-stage twiddle tables of length N (fft_tw_offset_rt).
// SYNC_LAST: the last-stage store goes to shared memory, so it needs the read/write barrier too.
// EVERY thread of the CTA must call this (it contains __syncthreads()).
// ---------------------------------------------------------------------------------------
// Hook: called by every thread right after the first CTA barrier of the transform, i.e. when all threads have consumed
// their first-stage inputs (row_step.cuh issues the next asynchronous bulk copy into the input staging buffer there).
struct NoHook { __device__ __forceinline__ void operator()() const {} };

template <typename T, int N, int DIR, int S, int NS, bool SYNC_LAST, class Load, class Store, class Hook>
__device__ __forceinline__ void fft_stage(int j0, cplx<T>* __restrict__ sm, const cplx<T>* __restrict__ tab,
                                          Load& load, Store& store, Hook& hook) {
  constexpr int R = fft_radix<N>(S);
  constexpr int NST = fft_nstages<N>();
  constexpr bool first = (S == 0), last = (S == NST - 1);
  constexpr int TPL = fft_tpl<N>();
  constexpr int NB = (N / R) / TPL;         // butterflies per thread: 16 / R
  cplx<T> v[NB][R];
  if constexpr (first) {
    // two-phase load: issue every global load of this thread first (all in flight together), then finish
    // (multipliers, packing).  Without this split ptxas interleaves loads with their dependent arithmetic.
    // Load::BATCHES = 2 splits the 16 slots into k < 8 and k >= 8 (two round trips, half the raw registers: for loaders
    // whose raw record is 32 bytes the single batch spilled, and a spill of a just-loaded value stalls on its load).
    constexpr int NBAT = Load::BATCHES;
    constexpr int SLOTS = NB * R;
#pragma unroll
    for (int bat = 0; bat < NBAT; ++bat) {
      if constexpr (Load::VEC == 4) {
        typename Load::raw_t raw[SLOTS / NBAT];
#pragma unroll
        for (int s = 0; s < SLOTS / NBAT; s += 4) load.issue(bat * (SLOTS / NBAT) + s, raw + s);
#pragma unroll
        for (int s = 0; s < SLOTS / NBAT; ++s) {
          const int k = bat * (SLOTS / NBAT) + s;
          v[k % NB][k / NB] = load.finish(j0 + k * TPL, k, raw[s]);
        }
      } else {
      decltype(load.issue(0, 0)) raw[SLOTS / NBAT];
#pragma unroll
      for (int s = 0; s < SLOTS / NBAT; ++s) {
        const int k = bat * (SLOTS / NBAT) + s;
        raw[s] = load.issue(j0 + k * TPL, k);
      }
#pragma unroll
      for (int s = 0; s < SLOTS / NBAT; ++s) {
        const int k = bat * (SLOTS / NBAT) + s;      // slot k = b + r NB  <->  v[b][r]
        v[k % NB][k / NB] = load.finish(j0 + k * TPL, k, raw[s]);
      }
      }
    }
#pragma unroll
    for (int b = 0; b < NB; ++b) dftR<R, DIR>(v[b]);
  } else {
    TwBase<R, T> tw[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      const int j = j0 + b * TPL;
      tw[b] = load_stage_twiddles<R, DIR>(tab + fft_tw_offset_rt(N, S) + (j & (NS - 1)), NS);
#pragma unroll
      for (int r = 0; r < R; ++r) v[b][r] = sm[fft_pad<N>(j + r * (N / R))];
    }
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      apply_stage_twiddles<R>(v[b], tw[b]);
      dftR<R, DIR>(v[b]);
    }
  }
  if (!last || SYNC_LAST) __syncthreads();     // every thread has finished reading this buffer
  if constexpr (first) hook();
  if constexpr (last && is_vec_store<Store>::value) {
    // last stage, vector store: slot k = b + r NB holds output index j0 + k TPL
#pragma unroll
    for (int k0 = 0; k0 < NB * R; k0 += 4) {
      cplx<T> t4[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) t4[i] = v[(k0 + i) % NB][(k0 + i) / NB];
      store.f(k0, t4);
    }
  } else {
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      const int j = j0 + b * TPL;
      const int k = j & (NS - 1);
      const int base = (j - k) * R + k;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const int o = base + r * NS;
        if constexpr (last) {
          if constexpr (!is_vec_store<Store>::value) store(o, b + r * NB, v[b][r]);   // o = j0 + k TPL, slot k = b + r NB
        } else sm[fft_pad<N>(o)] = v[b][r];
      }
    }
  }
  if constexpr (!last) {
    __syncthreads();
    fft_stage<T, N, DIR, S + 1, NS * R, SYNC_LAST>(j0, sm, tab, load, store, hook);
  }
}

template <typename T, int N, int DIR, bool SYNC_LAST, class Load, class Store, class Hook = NoHook>
__device__ __forceinline__ void fft_line(int j, cplx<T>* __restrict__ sm, const cplx<T>* __restrict__ tab,
                                         Load load, Store store, Hook hook = Hook()) {
  fft_stage<T, N, DIR, 0, 1, SYNC_LAST>(j, sm, tab, load, store, hook);
}

// ---------------------------------------------------------------------------------------
// "warp-local" plan for N = R1 x 16 x 16 (N = 4096, 2048, 1024: R1 = 16, 8, 4): the same Stockham stages, but the
// butterflies of stages 2 and 3 are assigned to threads so that the exchange BETWEEN them stays inside a half-warp:
//   stage 2 (radix 16, Ns = R1) butterfly j = k + R1 q writes the 16 positions  TPL q + k + R1 r,
//   stage 3 (radix 16, Ns = TPL) butterfly j'' = k + R1 r reads the 16 positions j'' + TPL q  (and writes the same),
// so the 16 producers {q} and the 16 consumers {r} of one k form a closed group.  Thread t of the line runs, in both
// stages, butterfly  wl_j(t) = (t >> 4) + R1 (t & 15)  (k = t >> 4, q or r = t & 15): a group is a half-warp, its 256
// positions are read in stage 2 by its own threads only, so the stage-2 -> stage-3 exchange needs a __syncwarp instead
// of two CTA barriers and the warps of a line drift apart (one warp's exchange overlaps another warp's arithmetic).
// Inside the group the element (q, r) is kept at position TPL q + k + R1 rot(r, q) (rot: fft_wl_rot below).  Only the stage-1 -> stage-2 exchange is
// CTA-wide.  Stage 1 is generic in its base index j0: j0 = t for inputs loaded in natural order (coalesced), j0 = wl_j(t)
// for inputs the thread already owns in registers.  Outputs: slot k of thread t is index wl_j(t) + k TPL.
// Twiddle tables (host: fill_stage_tables_wl): [15 powers][R1] for stage 2 (indexed by k = t >> 4: a broadcast per half-warp, so
// all 15 powers are read and none is derived), then [6 base powers][TPL] for stage 3 stored in THREAD order (entry t holds
// W_N^{wl_j(t) power}).  In fp64 the caller passes a copy of the table in SHARED memory: with 200 KB of dynamic shared memory the
// L1 is smaller than the table, every global twiddle load missed it (ncu, round 1: 0.06 % hits) and paid L2 latency in the
// middle of a stage; from shared memory the loads cost the same data-pipe wavefronts and 30 cycles.
// ---------------------------------------------------------------------------------------
// measured in k_row_step (B200, one row pair per CTA): the plan wins at N = 4096 (295 vs 316 us at C5); at N = 2048 the plain
// 16 x 16 x 8 plan is faster (141.9 vs 150.6 us at 2048 x 4096 fp64: the R1 = 8 first stage spills) and so is 16 x 8 x 8 at N = 1024
// (65.9 vs 74.4 us at 1024 x 4096 fp64): with one row pair per CTA several CTAs share an SM and hide each other's barriers
template <int N> __host__ __device__ constexpr bool fft_wl_supported() { return N == 4096; }
template <int N> __host__ __device__ constexpr int fft_wl_r1() { return N / 256; }
// stage 2 reads all 15 twiddle powers (fp64: 36 fewer DP instructions per butterfly) or 6 base powers and derives 9 (fp32: the
// shared-memory data pipe, not the FMA pipe, is the scarcer resource there)
template <typename T> __host__ __device__ constexpr bool fft_wl_stage2_all() { return sizeof(T) == 8; }
__host__ __device__ constexpr int fft_wl_r1_rt(int N) { return N / 256; }
__host__ __device__ constexpr int fft_wl_tw_elems_rt(int N) { return 15 * fft_wl_r1_rt(N) + 6 * (N / 16); }
// shared-memory index padding i + (i >> A) + (i >> B) and the in-group rotation, chosen per element size and N (searched
// exhaustively: every access of the plan - stage-1 writes from either base index, stage-2/3 reads and writes, the
// last-stage store - is then bank-conflict free for 16-byte (fp64) and 8-byte (fp32) elements).
template <typename T, int N> __host__ __device__ constexpr int fft_wl_pad_a() { return (sizeof(T) == 4 || N == 4096) ? 4 : 3; }
template <typename T, int N> __host__ __device__ constexpr int fft_wl_pad_b() { return 2 * fft_wl_pad_a<T, N>(); }
template <typename T, int N> __host__ __device__ constexpr int fft_wl_line_elems() {
  return N + (N >> fft_wl_pad_a<T, N>()) + (N >> fft_wl_pad_b<T, N>());
}
template <typename T, int N> __device__ __forceinline__ int fft_wl_pad(int i) {
  return i + (i >> fft_wl_pad_a<T, N>()) + (i >> fft_wl_pad_b<T, N>());
}
template <typename T, int N> __device__ __forceinline__ int fft_wl_rot(int r, int q) {
  return (sizeof(T) == 8 && N == 2048) ? (r ^ q) : r;
}
__host__ __device__ __forceinline__ int fft_wl_j_rt(int t, int r1) { return (t >> 4) + r1 * (t & 15); }
template <int N> __device__ __forceinline__ int fft_wl_j(int t) { return (t >> 4) + fft_wl_r1<N>() * (t & 15); }
template <typename T, int N, int DIR, bool SYNC_LAST, class Load, class Store, class Hook = NoHook>
__device__ __forceinline__ void fft_line_wl(int j0, int t, cplx<T>* __restrict__ sm, const cplx<T>* __restrict__ tabw,
                                            Load load, Store store, Hook hook = Hook()) {
  static_assert(fft_wl_supported<N>(), "warp-local plan: N = R1 x 16 x 16");
  constexpr int R1 = fft_wl_r1<N>(), TPL = N / 16, NB = 16 / R1;
  // ---- stage 1 (radix R1, Ns = 1, no twiddles) ----
  {
    cplx<T> v[NB][R1];
    constexpr int NBAT = Load::BATCHES, SLOTS = 16;
#pragma unroll
    for (int bat = 0; bat < NBAT; ++bat) {
      decltype(load.issue(0, 0)) raw[SLOTS / NBAT];
#pragma unroll
      for (int s = 0; s < SLOTS / NBAT; ++s) {
        const int k = bat * (SLOTS / NBAT) + s;
        raw[s] = load.issue(j0 + k * TPL, k);
      }
#pragma unroll
      for (int s = 0; s < SLOTS / NBAT; ++s) {
        const int k = bat * (SLOTS / NBAT) + s;      // slot k = b + r NB  <->  v[b][r]
        v[k % NB][k / NB] = load.finish(j0 + k * TPL, k, raw[s]);
      }
    }
#pragma unroll
    for (int b = 0; b < NB; ++b) dftR<R1, DIR>(v[b]);
    __syncthreads();                           // every thread has finished reading this buffer (previous transform)
    hook();
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      const int base = (j0 + b * TPL) * R1;
#pragma unroll
      for (int r = 0; r < R1; ++r) sm[fft_wl_pad<T, N>(base + r)] = v[b][r];
    }
    __syncthreads();
  }
  // ---- stages 2 and 3 (radix 16), exchange inside the half-warp ----
  const int kk = t >> 4, q = t & 15;
  const int j = kk + R1 * q;
  cplx<T> v[16];
#pragma unroll
  for (int r = 0; r < 16; ++r) v[r] = sm[fft_wl_pad<T, N>(j + r * TPL)];
  if constexpr (fft_wl_stage2_all<T>()) {
#pragma unroll
    for (int r = 1; r < 16; ++r) {             // stage-2 twiddles W_{16 R1}^{kk r}: all 15 powers, shared-memory broadcasts
      const cplx<T> w = tabw[(r - 1) * R1 + kk];
      v[r] = v[r] * (DIR < 0 ? w : conj(w));
    }
  } else {
    TwBase<16, T> b;                           // 6 base powers (rows 1, 2, 3, 4, 8, 12 of the table), the other 9 derived
#pragma unroll
    for (int i = 0; i < 6; ++i) { const cplx<T> w = tabw[(fft_tw_base_power(16, i) - 1) * R1 + kk]; b.w[i] = DIR < 0 ? w : conj(w); }
    apply_stage_twiddles<16>(v, b);
  }
  dft16<DIR>(v);
  __syncwarp();                                // the group's 256 positions have been read by its 16 threads
#pragma unroll
  for (int r = 0; r < 16; ++r) sm[fft_wl_pad<T, N>(TPL * q + kk + R1 * fft_wl_rot<T, N>(r, q))] = v[r];
  __syncwarp();
#pragma unroll
  for (int qq = 0; qq < 16; ++qq) v[qq] = sm[fft_wl_pad<T, N>(TPL * qq + kk + R1 * fft_wl_rot<T, N>(q, qq))];
  {
    TwBase<16, T> b;                           // stage-3 base powers from the shared-memory copy (thread order: conflict-free)
#pragma unroll
    for (int i = 0; i < 6; ++i) { const cplx<T> w = tabw[15 * R1 + i * TPL + t]; b.w[i] = DIR < 0 ? w : conj(w); }
    apply_stage_twiddles<16>(v, b);
  }
  dft16<DIR>(v);
  if (SYNC_LAST) __syncthreads();              // the store goes to shared memory: every group has finished reading it
#pragma unroll
  for (int r = 0; r < 16; ++r) store(j + r * TPL, r, v[r]);
}

}  // namespace ttsh
