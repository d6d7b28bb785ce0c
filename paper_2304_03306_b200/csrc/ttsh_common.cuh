// ttsh_common.cuh — shared device-side types of the B200 TTSH library (sm_100a only).
// Complex arithmetic, grid geometry, integer cutoff predicate, field-batch descriptors.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ttsh {

// ---------------------------------------------------------------------------------------
// complex scalar: layout-compatible with double2 / float2, naturally aligned for 64/128-bit LD/ST
// ---------------------------------------------------------------------------------------
template <typename T>
struct alignas(2 * sizeof(T)) cplx {
  T x, y;
};

template <typename T> __host__ __device__ __forceinline__ cplx<T> mk(T a, T b) { cplx<T> r; r.x = a; r.y = b; return r; }
template <typename T> __device__ __forceinline__ cplx<T> operator+(cplx<T> a, cplx<T> b) { return mk<T>(a.x + b.x, a.y + b.y); }
template <typename T> __device__ __forceinline__ cplx<T> operator-(cplx<T> a, cplx<T> b) { return mk<T>(a.x - b.x, a.y - b.y); }
template <typename T> __device__ __forceinline__ cplx<T> operator*(cplx<T> a, cplx<T> b) {
  return mk<T>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
template <typename T> __device__ __forceinline__ cplx<T> operator*(T s, cplx<T> a) { return mk<T>(s * a.x, s * a.y); }
template <typename T> __device__ __forceinline__ cplx<T> conj(cplx<T> a) { return mk<T>(a.x, -a.y); }
template <typename T> __device__ __forceinline__ cplx<T> mul_i(cplx<T> a) { return mk<T>(-a.y, a.x); }      // * (+i)
template <typename T> __device__ __forceinline__ cplx<T> mul_ni(cplx<T> a) { return mk<T>(a.y, -a.x); }     // * (-i)
// a * conj(b)
template <typename T> __device__ __forceinline__ cplx<T> mul_conj(cplx<T> a, cplx<T> b) {
  return mk<T>(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}

// ---------------------------------------------------------------------------------------
// programmatic dependent launch: the four kernels of a step are launched with the programmatic-stream-serialization
// attribute (engine.h: launch_pdl), so the next kernel's CTAs are scheduled while the last wave of the previous one drains
// and run their prologue (index arithmetic, twiddle loads, mbarrier set-up) early; pdl_wait() blocks until the previous grid
// has completed and its writes are visible, and must precede the first access to anything a predecessor writes.
// Both are no-ops in a kernel launched without the attribute.
// ---------------------------------------------------------------------------------------
#ifndef TTSH_PDL
#define TTSH_PDL 1
#endif
__device__ __forceinline__ void pdl_wait() {
#if TTSH_PDL
  asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
}
// Measured (B200): with the implicit trigger at kernel exit the attribute saves the launch latency at every kernel boundary
// (C5 fp64 425.4 -> 416.0 us per step, 256^2 21.4 -> 20.5 us); an explicit early trigger (TTSH_PDL_TRIGGER = 1: dependents
// become resident while the last wave still runs) was slower everywhere (C5 453 us, 1024^2 34.8 -> 46.5 us) and is off.
#ifndef TTSH_PDL_TRIGGER
#define TTSH_PDL_TRIGGER 0
#endif
__device__ __forceinline__ void pdl_trigger() {
#if TTSH_PDL && TTSH_PDL_TRIGGER
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
}

// ---------------------------------------------------------------------------------------
// grid geometry (host-filled, passed by value) and the HBM layouts
//
//   real fields       scalar[Ny][Nx], x contiguous.
//   retained modes    mx = 0..Wx-1 (Wx-1 = floor(num Nx / 2 den)), |my| <= My = floor(num Ny / 2 den): nothing outside
//                     is ever non-zero under the circular cutoff k^2 <= ((num/den) pi/dx)^2.
//                     Spectrum row q <-> my = q (q <= My) or q - Hy (q > My), Hy = 2 My + 1.
//   column tiles      the retained x-wavenumbers are grouped in NT tiles of CW adjacent columns (CW = the number of
//                     columns one CTA of the column pass transforms; a power of two).  Both complex arrays are
//                     TILE-MAJOR, so that a column CTA streams one contiguous block and never makes a strided access:
//   pruned spectrum   cplx[NT][Hy][CW]                      element (q, mx):  ((mx/CW) Hy + q) CW + mx%CW
//   intermediates     (x-spectral, y real).  A row-pass FFT packs the two same-parity rows y = 4a+p (A) and 4a+p+2 (B),
//                     row pair rp = 2a+p; (A, B) of one column are adjacent so that the row pass moves them with one
//                     32-byte (fp64) / 16-byte (fp32) access.  Two layouts, chosen so that every READ is contiguous
//                     and only fire-and-forget WRITES are scattered (in 2 CW-element pieces):
//     forward  (k_fwd_row writes, k_fwd_col reads)   cplx[NT][2][Ny/4][CW][2]   tile-major: the column CTA's block
//                     [Ny/2 rows of parity p][CW] is contiguous;  pair at  (((mx/CW) 2 + p) Ny/4 + a) 2 CW + 2 (mx%CW)
//     inverse  (k_inv_col writes, k_inv_row reads)   cplx[Ny/2][Wxp][2]         pair-row-major: the row CTA's 2 Wxp
//                     elements are contiguous;  pair at  (rp Wxp + mx) 2,   Wxp = NT CW
// ---------------------------------------------------------------------------------------
struct Geom {
  int Nx, Ny;
  int Wx;                  // retained x-wavenumbers
  int CW, cw_shift, NT;    // tile width (columns), log2, number of tiles = ceil(Wx / CW)
  int Wxp;                 // NT * CW: padded number of columns
  int My, Hy;
  int num, den;            // dealias fraction
  int cut_gx, cut_gy, cut_c;   // Nx / g, Ny / g, Nx Ny / g with g = min(Nx, Ny): the cutoff predicate with its common factor divided out
  double dkx, dky;         // 2 pi / (Nx dx), 2 pi / (Ny dx)   (Table I)
  double inv_sqrt_nx, inv_sqrt_ny;
};

__host__ __device__ __forceinline__ size_t spec_index(const Geom& g, int q, int mx) {
  return ((size_t)(mx >> g.cw_shift) * g.Hy + q) * g.CW + (mx & (g.CW - 1));
}
// forward intermediate: index of the (A, B) pair (rows 4a+p and 4a+p+2) of column mx; B is the next element
__host__ __device__ __forceinline__ size_t inter_pair_index(const Geom& g, int a, int p, int mx) {
  return ((((size_t)(mx >> g.cw_shift) * 2 + p) * (g.Ny >> 2) + a) * g.CW + (mx & (g.CW - 1))) * 2;
}

// permuted row layout of the internal real fields: element x = j + k TPL (the 16 points one thread owns are k = 0..15)
// is stored at ((k >> 2) TPL + j) 4 + (k & 3), so that a thread moves its points with 4 wide accesses (LDG/STG.256 in
// fp64) and a warp instruction still covers 1 KB of contiguous memory.  TPL = row length / 16.
__host__ __device__ __forceinline__ int perm_index(int x, int tpl) {
  const int j = x % tpl, k = x / tpl;
  return ((k >> 2) * tpl + j) * 4 + (k & 3);
}

// thread-order ("wl") permuted row layout of a real field: element x = wl_j(t) + k TPL at ((k >> 2) TPL + t) 4 + (k & 3)
__host__ __device__ __forceinline__ int perm_index_wl(int x, int tpl) {
  const int r1 = tpl / 16, jj = x % tpl, k = x / tpl;
  const int t = 16 * (jj % r1) + jj / r1;
  return ((k >> 2) * tpl + t) * 4 + (k & 3);
}

// strict '>' cutoff evaluated exactly in integers (reading R4):
//   k^2 > ((num/den) pi/dx)^2   <=>   4 den^2 ((mx Ny)^2 + (my Nx)^2) > num^2 (Nx Ny)^2
// Nx, Ny are powers of two, so the three products share the factor g = min(Nx, Ny), which is divided out (host, make_geom:
// cut_gx = Nx / g, cut_gy = Ny / g, cut_c = Nx Ny / g): with |mx| <= Nx/2, |my| <= Ny/2, max(Nx, Ny) <= 2^14 and den <= 64 both
// sides stay below 2^42, so nothing overflows int64 at any accepted size.
__host__ __device__ __forceinline__ bool is_cut(const Geom& g, int mx, int my, int num, int den) {
  const long long a = (long long)mx * g.cut_gy, b = (long long)my * g.cut_gx, c = g.cut_c;
  return 4LL * den * den * (a * a + b * b) > (long long)num * num * c * c;
}

// ---------------------------------------------------------------------------------------
// batched field descriptors: one launch transforms up to 5 fields (blockIdx.y selects the field)
// ---------------------------------------------------------------------------------------
enum SpecMode : int {     // multiplier applied to the spectrum while loading the inverse column pass
  SM_ONE = 0,             // x^                              (w^ -> w,  psi^ -> psi and, with -i k_x in the row pass, v_y)
  SM_IKY = 1,             // i k_y x^                        (Alg. 1 line 2)
  SM_IKY_MEANX = 2,       // i k_y psi^ = v^_x; the (0,0) entry is the mean flow v^_x(0)   (lines 8, 14)
  SM_LOWPASS4 = 3         // 1 inside the (1/4) pi/dx circle, else 0   (Alg. 2 lines 2-8)
};
enum RowMode : int {      // multiplier applied in x-spectral space by the inverse row pass
  RM_ONE = 0,
  RM_IKX = 1,             // i k_x            (d_x w)
  RM_NIKX_MEANY = 2,      // -i k_x psi~ = v~_y; the mx = 0 entry is the mean flow v^_y(0)/sqrt(Ny)  (lines 8, 14)
  RM_MODE_MASK = 0xff,
  RM_PERM = 0x100         // flag: the real rows of this field use the permuted internal layout (perm_index, fft_core.cuh)
};

struct FieldOp {
  const void* src;
  void* dst;
  int mode;
  int _pad;
};
struct Batch {
  FieldOp f[5];
};

// parameters of the model as the kernels need them (always double; cast inside)
struct Model {
  double lambda0, alpha, beta, Gamma0, Gamma2, gamma_v, gamma_w, dt;
};

}  // namespace ttsh
