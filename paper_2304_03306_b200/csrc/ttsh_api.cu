// ttsh_api.cu — the C ABI of include/ttsh.h: handle, argument validation, workspace carving, the step
// schedule of Algorithm 1 and its CUDA-graph replay.  No device memory is allocated here.
#include "../../include/ttsh.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "engine.h"
#include "fft_passes.cuh"

using namespace ttsh;
#define TTSH_STR2(x) #x
#define TTSH_STR(x) TTSH_STR2(x)

namespace {

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

inline bool pow2_in_range(int n) { return n >= 64 && n <= 16384 && (n & (n - 1)) == 0; }   // PAPER.md:271 (8192), :282 (16384)

struct Layout {
  size_t tabX, tabXw, tabY, tabS, K, K2, what, psihat, v0, diag_partial, diag_out, R[5], Tm[5], S[3], total;
};

Geom make_geom(int Nx, int Ny, double dx, int num, int den, size_t w) {
  Geom g;
  g.Nx = Nx; g.Ny = Ny;
  g.num = num; g.den = den;
  const int gmin = Nx < Ny ? Nx : Ny;
  g.cut_gx = Nx / gmin; g.cut_gy = Ny / gmin; g.cut_c = g.cut_gx * g.cut_gy * gmin;
  g.Wx = (int)((long long)num * Nx / (2LL * den)) + 1;
  g.CW = col_tile_width(Ny, (int)(2 * w));
  g.cw_shift = g.CW == 1 ? 0 : (g.CW == 2 ? 1 : (g.CW == 4 ? 2 : 3));
  g.NT = (g.Wx + g.CW - 1) / g.CW;
  g.Wxp = g.NT * g.CW;
  g.My = (int)((long long)num * Ny / (2LL * den));
  g.Hy = 2 * g.My + 1;
  const long double two_pi = 2.0L * acosl(-1.0L);
  g.dkx = (double)(two_pi / ((long double)Nx * (long double)dx));
  g.dky = (double)(two_pi / ((long double)Ny * (long double)dx));
  g.inv_sqrt_nx = (double)(1.0L / sqrtl((long double)Nx));
  g.inv_sqrt_ny = (double)(1.0L / sqrtl((long double)Ny));
  return g;
}

// The workspace is sized for the widest dealias fraction the ABI accepts (2/3), so that
// ttsh_workspace_bytes does not depend on the parameters.
Layout make_layout(int Nx, int Ny, size_t w) {
  const Geom g = make_geom(Nx, Ny, 1.0, 2, 3, w);
  const size_t P = (size_t)Nx * Ny, cw = 2 * w;
  const size_t inter = (size_t)g.NT * g.CW * Ny * cw, spec = (size_t)g.NT * g.CW * g.Hy * cw;
  Layout L;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
  L.tabX = take((size_t)Nx * cw);
  L.tabXw = take((size_t)Nx * cw);         // warp-local plan tables (fft_core.cuh), 6 (Nx/256 + Nx/16) entries; Nx = 16384: W_Nx^j, j < Nx/32
  L.tabY = take((size_t)Ny * cw);
  L.tabS = take((size_t)Ny * cw);
  L.K = take(P * w);
  L.K2 = take(P * w);                      // K in the thread-order row layout of the fused row-step kernel
  L.what = take(spec);
  L.psihat = take(spec);
  L.v0 = take(8 * sizeof(double));
  L.diag_partial = take((size_t)DIAG_BLOCKS * 8 * sizeof(double));
  L.diag_out = take(8 * sizeof(double));
  for (int i = 0; i < 5; ++i) L.R[i] = take(P * w);
  for (int i = 0; i < 5; ++i) L.Tm[i] = take(inter);
  for (int i = 0; i < 3; ++i) L.S[i] = take(spec);
  L.total = off;
  return L;
}

}  // namespace

struct ttsh_handle {
  int Nx, Ny;
  double dx, dt;
  ttsh_params p;
  ttsh_dtype dtype;
  Geom g;
  Model m;
  cudaStream_t stream;
  char* ws;
  void *tabX, *tabXw, *tabY, *tabS, *K, *K2, *what, *psihat, *R[5], *Tm[5], *S[3];
  double *v0, *diag_partial, *diag_out;
  bool initialized;
  double t;
  long long step;
  long long launches;
  int sticky;
  std::string err;
  cudaGraphExec_t graph_exec;      // one captured Euler step
  cudaGraphExec_t graph_exec_k;    // GRAPH_K captured Euler steps (grids up to 256^2: one graph launch costs as much as the step)
  bool graph_ok;
  int advection_form;
  int device;           // CUDA device of the workspace: every entry point must be called with it current
  int rs_slots, rs_slots_ens, rs_slots_tan;   // persistent grid of k_row_step on this device (single system / ensemble / tangent variant)
  bool row_step_ok;     // the fused row-step kernel supports this grid / dtype / dealias fraction
  bool row_step_wl;     // ... and runs the warp-local FFT plan (thread-order K copy, warp-local twiddle table)
  void* rs_tab;         // the twiddle table the fused row kernel of this grid reads (tabX, or tabXw for the warp-local / real-row variants)
  bool col_step_ok;     // the fused column kernel (col_step.cuh) applies: an Euler step is k_row_step + k_col_step
  bool inter_valid;     // ... and the inverse intermediates Tm[0], Tm[2], Tm[3] of the CURRENT state are at hand (k_col_step of the
                        //     previous step wrote them); cleared by everything that touches the state or the scratch arrays
  bool row_step_real;   // ... or the real-row variant (row_step_real.cuh: its own K order and table)
  bool real_rows;       // Nx = 16384: one real row per half-length transform (fft_rows_real.cuh); internal real fields in natural order
};

struct ttsh_psd {
  ttsh_handle* h;                      // borrowed
  std::vector<double> omegas, cs, sn;  // frequencies; phases of the current sample (host)
  void* acc;                           // cplx<T>[nfreq][Ny*Nx] in the caller's workspace
  size_t acc_bytes;
  double *partial, *out;
  long long nsamples;
};

struct ttsh_tangent {
  ttsh_handle* h;                      // borrowed
  int nvec;
  size_t stride;                       // bytes between the workspace blocks of consecutive vectors
  // block of vector 0 (vector i: + i * stride): dw^, dpsi^ (pruned tile-major spectra), dv^(0), and per-vector scratch:
  // dw | dv_x | dv_y in real space (permuted internal row layout), three intermediates, three spectra
  void *what, *psihat;
  double* v0;
  void *real[3], *inter[3], *spec[3];
  std::vector<bool> set;
  double *partial, *coef, *rdiag, *gram;
};
template <class P> static P* vec_ptr(const ttsh_tangent* s, P* p0, int i) {
  return reinterpret_cast<P*>(reinterpret_cast<char*>(p0) + (size_t)i * s->stride);
}

struct ttsh_ensemble {
  bool col_fused;                      // the step is k_row_step + k_col_step (small ensembles of grids with 128 <= Ny <= 1024), else 4 launches
  std::vector<ttsh_handle*> members;   // borrowed
  size_t mstride;                      // bytes between consecutive members' workspaces
  cudaGraphExec_t graph_exec;
  long long launches;
};

namespace {

#define TRY(h, call)                                                        \
  do {                                                                      \
    cudaError_t e_ = (call);                                                \
    if (e_ != cudaSuccess) return fail_cuda((h), e_, #call);                \
  } while (0)

// every pointer of a handle lives on one CUDA device (that of the workspace); the kernels' shared-memory opt-in and the
// persistent grids were set up for it.  Entry points refuse to run with another device current.
bool on_device(const ttsh_handle* h) {
  int dev = -1;
  return h->device < 0 || (cudaGetDevice(&dev) == cudaSuccess && dev == h->device);
}
#define CHECK_DEVICE(h) do { if (!on_device(h)) return TTSH_ERR_INVALID_ARG; } while (0)

int fail_cuda(ttsh_handle* h, cudaError_t e, const char* what) {
  if (h) {
    h->sticky = TTSH_ERR_CUDA;
    h->err = std::string(what) + ": " + cudaGetErrorString(e);
  }
  return TTSH_ERR_CUDA;
}

// forward-sign twiddle W_M^p = exp(-2 pi i p / M), evaluated in long double, exact on the axes
template <typename T> void put_twiddle(T* t, long long p, long long M) {
  p %= M;
  const long double two_pi = 2.0L * acosl(-1.0L);
  long double a = two_pi * (long double)p / (long double)M;
  long double c = cosl(a), s = -sinl(a);
  if (4 * p == M || 4 * p == 3 * M) c = 0.0L;
  if (p == 0 || 2 * p == M) s = 0.0L;
  t[0] = (T)c;
  t[1] = (T)s;
}
// per-stage tables of a length-N transform (layout: fft_core.cuh, fft_tw_offset_rt)
template <typename T> void fill_stage_tables(std::vector<unsigned char>& buf, int N) {
  buf.assign((size_t)(fft_tw_elems_rt(N) + 1) * 2 * sizeof(T), 0);
  T* t = reinterpret_cast<T*>(buf.data());
  int ns = fft_radix_rt(N, 0);
  for (int s = 1; s < fft_nstages_rt(N); ++s) {
    const int R = fft_radix_rt(N, s), off = fft_tw_offset_rt(N, s);
    for (int b = 0; b < fft_tw_nbase(R); ++b)
      for (int k = 0; k < ns; ++k)
        put_twiddle<T>(t + 2 * (size_t)(off + b * ns + k), (long long)k * fft_tw_base_power(R, b), (long long)ns * R);
    ns *= R;
  }
}
// tables of the warp-local plan N = R1 x 16 x 16 (fft_core.cuh, fft_line_wl): stage 2 [15 powers][R1], stage 3 [6 base powers][TPL] in thread order
template <typename T> void fill_stage_tables_wl(std::vector<unsigned char>& buf, int N) {
  const int R1 = fft_wl_r1_rt(N), TPL = N / 16;
  buf.assign((size_t)(fft_wl_tw_elems_rt(N) + 1) * 2 * sizeof(T), 0);
  T* t = reinterpret_cast<T*>(buf.data());
  for (int r = 1; r < 16; ++r)
    for (int k = 0; k < R1; ++k) put_twiddle<T>(t + 2 * (size_t)((r - 1) * R1 + k), (long long)k * r, 16LL * R1);
  for (int b = 0; b < 6; ++b)
    for (int th = 0; th < TPL; ++th)
      put_twiddle<T>(t + 2 * (size_t)(15 * R1 + b * TPL + th), (long long)fft_wl_j_rt(th, R1) * fft_tw_base_power(16, b), (long long)N);
}
// split twiddles of the column pass: W_Ny^p, p < Ny/2
template <typename T> void fill_split_table(std::vector<unsigned char>& buf, int Ny) {
  buf.assign((size_t)(Ny / 2) * 2 * sizeof(T), 0);
  T* t = reinterpret_cast<T*>(buf.data());
  for (int p = 0; p < Ny / 2; ++p) put_twiddle<T>(t + 2 * (size_t)p, p, Ny);
}

// ---- dtype dispatch helpers ---------------------------------------------------------------
#define DISPATCH(h, fn, ...) ((h)->dtype == TTSH_F64 ? fn<double>(__VA_ARGS__) : fn<float>(__VA_ARGS__))

Batch make_batch(std::initializer_list<FieldOp> ops) {
  Batch b;
  memset(&b, 0, sizeof(b));
  int i = 0;
  for (const FieldOp& o : ops) b.f[i++] = o;
  return b;
}
FieldOp op(const void* src, void* dst, int mode) { FieldOp o; o.src = src; o.dst = dst; o.mode = mode; o._pad = 0; return o; }

// inverse 2-D transforms of the state into real fields; any destination may be NULL
int enqueue_inverse(ttsh_handle* h, void* w, void* gx, void* gy, void* vx, void* vy, void* psi) {
  h->inter_valid = false;
  // column pass: which intermediates are needed
  const bool need_w = w || gx, need_gy = gy != nullptr, need_psi = vy || psi, need_vx = vx != nullptr;
  Batch cb; memset(&cb, 0, sizeof(cb));
  int nc = 0;
  if (need_w) cb.f[nc++] = op(h->what, h->Tm[0], SM_ONE);
  if (need_gy) cb.f[nc++] = op(h->what, h->Tm[1], SM_IKY);
  if (need_psi) cb.f[nc++] = op(h->psihat, h->Tm[2], SM_ONE);
  if (need_vx) cb.f[nc++] = op(h->psihat, h->Tm[3], SM_IKY_MEANX);
  if (nc == 0) return TTSH_OK;
  TRY(h, DISPATCH(h, launch_inv_col, h->g, cb, nc, h->tabY, h->tabS, h->v0, h->stream));
  h->launches++;
  // row pass; psi and v_y share the intermediate psi~, so psi (if requested) goes in a second launch slot
  Batch rb; memset(&rb, 0, sizeof(rb));
  int nr = 0;
  if (w) rb.f[nr++] = op(h->Tm[0], w, RM_ONE);
  if (gx) rb.f[nr++] = op(h->Tm[0], gx, RM_IKX);
  if (gy) rb.f[nr++] = op(h->Tm[1], gy, RM_ONE);
  if (vx) rb.f[nr++] = op(h->Tm[3], vx, RM_ONE);
  if (vy) rb.f[nr++] = op(h->Tm[2], vy, RM_NIKX_MEANY);
  if (nr) {
    TRY(h, DISPATCH(h, launch_inv_row, h->g, rb, nr, h->tabX, h->tabXw, h->v0, h->stream));
    h->launches++;
  }
  if (psi) {
    Batch pb = make_batch({op(h->Tm[2], psi, RM_ONE)});
    TRY(h, DISPATCH(h, launch_inv_row, h->g, pb, 1, h->tabX, h->tabXw, h->v0, h->stream));
    h->launches++;
  }
  return TTSH_OK;
}

// forward 2-D transforms of n real fields into pruned spectra S[0..n-1]
int enqueue_forward(ttsh_handle* h, int n, const void* const* src) {
  h->inter_valid = false;
  Batch rb; memset(&rb, 0, sizeof(rb));
  Batch cb; memset(&cb, 0, sizeof(cb));
  for (int i = 0; i < n; ++i) {
    rb.f[i] = op(src[i], h->Tm[i], 0);
    cb.f[i] = op(h->Tm[i], h->S[i], 0);
  }
  TRY(h, DISPATCH(h, launch_fwd_row, h->g, rb, n, h->tabX, h->tabXw, h->stream));
  TRY(h, DISPATCH(h, launch_fwd_col, h->g, cb, n, h->tabY, h->tabS, h->stream));
  h->launches += 2;
  return TTSH_OK;
}

int enqueue_stage(ttsh_handle* h, int stage) {
  switch (stage) {
    case TTSH_STAGE_INV_COL: {
      if (h->advection_form == TTSH_ADVECTION_CONSERVATIVE) {   // w, psi (-> v_y), i k_y psi (-> v_x)
        Batch cb = make_batch({op(h->what, h->Tm[0], SM_ONE), op(h->psihat, h->Tm[2], SM_ONE), op(h->psihat, h->Tm[3], SM_IKY_MEANX)});
        TRY(h, DISPATCH(h, launch_inv_col, h->g, cb, 3, h->tabY, h->tabS, h->v0, h->stream));
      } else {
        Batch cb = make_batch({op(h->what, h->Tm[0], SM_ONE), op(h->what, h->Tm[1], SM_IKY), op(h->psihat, h->Tm[2], SM_ONE),
                               op(h->psihat, h->Tm[3], SM_IKY_MEANX)});
        TRY(h, DISPATCH(h, launch_inv_col, h->g, cb, 4, h->tabY, h->tabS, h->v0, h->stream));
      }
      h->launches++;
      return TTSH_OK;
    }
    case TTSH_STAGE_INV_ROW: {
      if (h->advection_form == TTSH_ADVECTION_CONSERVATIVE) {
        Batch rb = make_batch({op(h->Tm[0], h->R[0], RM_ONE | RM_PERM), op(h->Tm[3], h->R[3], RM_ONE | RM_PERM),
                               op(h->Tm[2], h->R[4], RM_NIKX_MEANY | RM_PERM)});
        TRY(h, DISPATCH(h, launch_inv_row, h->g, rb, 3, h->tabX, h->tabXw, h->v0, h->stream));
      } else {
        Batch rb = make_batch({op(h->Tm[0], h->R[0], RM_ONE | RM_PERM), op(h->Tm[0], h->R[1], RM_IKX | RM_PERM),
                               op(h->Tm[1], h->R[2], RM_ONE | RM_PERM), op(h->Tm[3], h->R[3], RM_ONE | RM_PERM),
                               op(h->Tm[2], h->R[4], RM_NIKX_MEANY | RM_PERM)});
        TRY(h, DISPATCH(h, launch_inv_row, h->g, rb, 5, h->tabX, h->tabXw, h->v0, h->stream));
      }
      h->launches++;
      return TTSH_OK;
    }
    case TTSH_STAGE_REAL:
      if (h->advection_form == TTSH_ADVECTION_CONSERVATIVE)
        TRY(h, DISPATCH(h, launch_realspace_cons, h->g, h->m, h->R[3], h->R[4], h->K, h->R[0], h->R[1], h->R[2], h->stream));
      else
        TRY(h, DISPATCH(h, launch_realspace, h->g, h->m, h->R[3], h->R[4], h->K, h->R[0], h->R[1], h->R[2], h->stream));
      h->launches++;
      return TTSH_OK;
    case TTSH_STAGE_FWD_ROW: {
      Batch rb = make_batch({op(h->R[1], h->Tm[0], RM_PERM), op(h->R[2], h->Tm[1], RM_PERM), op(h->R[0], h->Tm[2], RM_PERM)});
      TRY(h, DISPATCH(h, launch_fwd_row, h->g, rb, 3, h->tabX, h->tabXw, h->stream));
      h->launches++;
      return TTSH_OK;
    }
    case TTSH_STAGE_FWD_COL: {
      Batch cb = make_batch({op(h->Tm[0], h->S[0], 0), op(h->Tm[1], h->S[1], 0), op(h->Tm[2], h->S[2], 0)});
      TRY(h, DISPATCH(h, launch_fwd_col, h->g, cb, 3, h->tabY, h->tabS, h->stream));
      h->launches++;
      return TTSH_OK;
    }
    case TTSH_STAGE_REAL_FWD_ROW:     // a3 + row half of a4 in one kernel (conservative form only)
      if (h->advection_form != TTSH_ADVECTION_CONSERVATIVE || h->real_rows) return TTSH_ERR_INVALID_ARG;
      TRY(h, DISPATCH(h, launch_fwd_row_fused, h->g, h->m, h->R[3], h->R[4], h->R[0], h->K, h->Tm[1], h->Tm[4], h->tabX, h->stream));
      h->launches++;
      return TTSH_OK;
    case TTSH_STAGE_FWD_COL_P2: {      // column pass of the two intermediates A~, B~ of TTSH_STAGE_REAL_FWD_ROW
      Batch cb = make_batch({op(h->Tm[1], h->S[0], 0), op(h->Tm[4], h->S[1], 0)});
      TRY(h, DISPATCH(h, launch_fwd_col, h->g, cb, 2, h->tabY, h->tabS, h->stream));
      h->launches++;
      return TTSH_OK;
    }
    case TTSH_STAGE_ROW_STEP:         // a2/a6 row pass + a3 + a4 row pass in one kernel (conservative form, 1/2 rule)
      if (h->advection_form != TTSH_ADVECTION_CONSERVATIVE || !h->row_step_ok) return TTSH_ERR_INVALID_ARG;
      TRY(h, DISPATCH(h, launch_row_step, h->g, h->m, h->Tm[0], h->Tm[3], h->Tm[2], (h->row_step_wl || h->row_step_real) ? h->K2 : h->K, h->Tm[1], h->Tm[4],
                      h->rs_tab, h->v0, h->stream, h->rs_slots));
      h->launches++;
      return TTSH_OK;
    case TTSH_STAGE_COL_STEP:         // a4 column pass + a5 + the column pass of a2 / a6 of the next step in one kernel
      if (h->advection_form != TTSH_ADVECTION_CONSERVATIVE || !h->col_step_ok) return TTSH_ERR_INVALID_ARG;
      TRY(h, DISPATCH(h, launch_col_step, h->g, h->m, h->Tm[1], h->Tm[4], h->what, h->psihat, h->v0, h->Tm[0], h->Tm[2], h->Tm[3], h->tabY,
                      h->tabS, h->stream));
      h->launches++;
      return TTSH_OK;
    case TTSH_STAGE_SPECTRAL_P2:
      TRY(h, DISPATCH(h, launch_spectral_p2, h->g, h->m, h->S[0], h->S[1], h->what, h->psihat, h->v0, h->stream));
      h->launches++;
      return TTSH_OK;
    case TTSH_STAGE_SPECTRAL:
      TRY(h, DISPATCH(h, launch_spectral, h->g, h->m, h->S[0], h->S[1], h->S[2], h->what, h->psihat, h->v0, h->stream));
      h->launches++;
      return TTSH_OK;
  }
  return TTSH_ERR_INVALID_ARG;
}

// one application of Algorithm 1.  The two inverse transforms of v (a6) are scheduled at the START of the
// step that consumes v, together with those of w and grad w: the state carried between steps is (w^, v^(0)).
int enqueue_step(ttsh_handle* h) {
  static const int fused[] = {TTSH_STAGE_INV_COL, TTSH_STAGE_INV_ROW, TTSH_STAGE_REAL_FWD_ROW, TTSH_STAGE_FWD_COL_P2,
                              TTSH_STAGE_SPECTRAL_P2};
  static const int rowstep[] = {TTSH_STAGE_INV_COL, TTSH_STAGE_ROW_STEP, TTSH_STAGE_FWD_COL_P2, TTSH_STAGE_SPECTRAL_P2};
  static const int plain[] = {TTSH_STAGE_INV_COL, TTSH_STAGE_INV_ROW, TTSH_STAGE_REAL, TTSH_STAGE_FWD_ROW, TTSH_STAGE_FWD_COL,
                              TTSH_STAGE_SPECTRAL};
  // conservative form: 4 launches where the fused row-step kernel applies, else 5 (fused real-space + forward row pass); the
  // literal form and Nx = 16384 (real-row passes, no fused row kernels) run the 6-launch sequence
  const bool f = h->advection_form == TTSH_ADVECTION_CONSERVATIVE && (!h->real_rows || h->row_step_real);
  if (f && h->col_step_ok) {      // two launches per step; the column pass of a2 / a6 only when its output is not at hand
    int rc = TTSH_OK;
    if (!h->inter_valid) rc = enqueue_stage(h, TTSH_STAGE_INV_COL);
    if (rc == TTSH_OK) rc = enqueue_stage(h, TTSH_STAGE_ROW_STEP);
    if (rc == TTSH_OK) rc = enqueue_stage(h, TTSH_STAGE_COL_STEP);
    h->inter_valid = rc == TTSH_OK;
    return rc;
  }
  const int* seq = f ? (h->row_step_ok ? rowstep : fused) : plain;
  const int n = f ? (h->row_step_ok ? 4 : 5) : 6;
  for (int i = 0; i < n; ++i) {
    int rc = enqueue_stage(h, seq[i]);
    if (rc != TTSH_OK) return rc;
  }
  return TTSH_OK;
}
inline int launches_per_step(const ttsh_handle* h) {
  const bool f = h->advection_form == TTSH_ADVECTION_CONSERVATIVE && (!h->real_rows || h->row_step_real);
  if (f && h->col_step_ok) return 2;
  return f ? (h->row_step_ok ? 4 : 5) : 6;
}

// natural <-> internal row layout of a real field (to_perm = 1: natural -> internal).  On real-row grids the internal layout IS
// the natural one.
int copy_real(ttsh_handle* h, const void* src, void* dst, int to_perm) {
  const size_t P = (size_t)h->Nx * h->Ny;
  if (h->real_rows) TRY(h, cudaMemcpyAsync(dst, src, P * (size_t)h->dtype, cudaMemcpyDeviceToDevice, h->stream));
  else TRY(h, DISPATCH(h, launch_permute, h->Nx, P, src, dst, to_perm, h->stream));
  h->launches++;
  return TTSH_OK;
}

int apply_mask_k(ttsh_handle* h, const void* mask, ttsh_mask_kind kind);
int apply_mask(ttsh_handle* h, const void* mask, ttsh_mask_kind kind) {
  int rc = apply_mask_k(h, mask, kind);
  if (rc != TTSH_OK || !(h->row_step_ok && (h->row_step_wl || h->row_step_real))) return rc;
  if (h->row_step_real) TRY(h, DISPATCH(h, launch_reperm_real, h->Nx, (size_t)h->Nx * h->Ny, h->K, h->K2, h->stream));
  else TRY(h, DISPATCH(h, launch_reperm_wl, h->Nx, (size_t)h->Nx * h->Ny, h->K, h->K2, h->stream));
  h->launches++;
  return TTSH_OK;
}
int apply_mask_k(ttsh_handle* h, const void* mask, ttsh_mask_kind kind) {
  const size_t P = (size_t)h->Nx * h->Ny;
  const size_t w = (size_t)h->dtype;
  if (!mask) {
    TRY(h, DISPATCH(h, launch_fill, P, h->K, 0.0, h->stream));
    h->launches++;
    return TTSH_OK;
  }
  if (kind == TTSH_MASK_PROCESSED) return copy_real(h, mask, h->K, 1);   // K is kept in the internal row layout
  // Algorithm 2: K = ( iDFT[ lowpass_{1/4}( DFT[K_naive] ) ] )^2
  TRY(h, DISPATCH(h, launch_mask_to_real, P, static_cast<const unsigned char*>(mask), h->R[0], h->stream));
  h->launches++;
  const void* src[1] = {h->R[0]};
  int rc = enqueue_forward(h, 1, src);
  if (rc != TTSH_OK) return rc;
  Batch cb = make_batch({op(h->S[0], h->Tm[0], SM_LOWPASS4)});
  TRY(h, DISPATCH(h, launch_inv_col, h->g, cb, 1, h->tabY, h->tabS, h->v0, h->stream));
  Batch rb = make_batch({op(h->Tm[0], h->R[0], RM_ONE | RM_PERM)});
  TRY(h, DISPATCH(h, launch_inv_row, h->g, rb, 1, h->tabX, h->tabXw, h->v0, h->stream));
  TRY(h, DISPATCH(h, launch_square, P, h->R[0], h->K, h->stream));
  h->launches += 3;
  return TTSH_OK;
}

}  // namespace

extern "C" {

size_t ttsh_workspace_bytes(int Nx, int Ny, ttsh_dtype t) {
  if (!pow2_in_range(Nx) || !pow2_in_range(Ny)) return 0;
  if (t != TTSH_F64 && t != TTSH_F32) return 0;
  return make_layout(Nx, Ny, (size_t)t).total;
}

int ttsh_create(ttsh_handle** out, int Nx, int Ny, double dx, double dt, const ttsh_params* p, ttsh_dtype t,
                const void* mask, ttsh_mask_kind kind, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!out) return TTSH_ERR_INVALID_ARG;
  *out = nullptr;
  if (!p || !workspace) return TTSH_ERR_INVALID_ARG;
  if (t != TTSH_F64 && t != TTSH_F32) return TTSH_ERR_INVALID_ARG;
  if (!(dx > 0.0) || !(dt > 0.0) || !(p->Gamma2 >= 0.0)) return TTSH_ERR_INVALID_ARG;
  if (!std::isfinite(dx) || !std::isfinite(dt)) return TTSH_ERR_INVALID_ARG;
  for (double v : {p->lambda0, p->alpha, p->beta, p->Gamma0, p->Gamma2, p->gamma_v, p->gamma_w})
    if (!std::isfinite(v)) return TTSH_ERR_INVALID_ARG;
  if (kind != TTSH_MASK_BINARY && kind != TTSH_MASK_PROCESSED) return TTSH_ERR_INVALID_ARG;
  if (p->dealias_num <= 0 || p->dealias_den <= 0) return TTSH_ERR_INVALID_ARG;
  if (4 * p->dealias_num < p->dealias_den || 3 * p->dealias_num > 2 * p->dealias_den) return TTSH_ERR_INVALID_ARG;
  if (p->dealias_den > 64) return TTSH_ERR_INVALID_ARG;
  if (!pow2_in_range(Nx) || !pow2_in_range(Ny)) return TTSH_ERR_UNSUPPORTED_SIZE;
  const Layout L = make_layout(Nx, Ny, (size_t)t);
  if (workspace_bytes < L.total) return TTSH_ERR_WORKSPACE_TOO_SMALL;
  if (reinterpret_cast<uintptr_t>(workspace) % ALIGN) return TTSH_ERR_INVALID_ARG;

  ttsh_handle* h = new (std::nothrow) ttsh_handle();
  if (!h) return TTSH_ERR_INVALID_ARG;
  h->Nx = Nx; h->Ny = Ny; h->dx = dx; h->dt = dt; h->p = *p; h->dtype = t;
  h->g = make_geom(Nx, Ny, dx, p->dealias_num, p->dealias_den, (size_t)t);
  h->m.lambda0 = p->lambda0; h->m.alpha = p->alpha; h->m.beta = p->beta; h->m.Gamma0 = p->Gamma0;
  h->m.Gamma2 = p->Gamma2; h->m.gamma_v = p->gamma_v; h->m.gamma_w = p->gamma_w; h->m.dt = dt;
  h->stream = static_cast<cudaStream_t>(cuda_stream);
  h->ws = static_cast<char*>(workspace);
  h->tabX = h->ws + L.tabX; h->tabXw = h->ws + L.tabXw; h->K2 = h->ws + L.K2; h->tabY = h->ws + L.tabY; h->tabS = h->ws + L.tabS; h->K = h->ws + L.K; h->what = h->ws + L.what; h->psihat = h->ws + L.psihat;
  h->v0 = reinterpret_cast<double*>(h->ws + L.v0);
  h->diag_partial = reinterpret_cast<double*>(h->ws + L.diag_partial);
  h->diag_out = reinterpret_cast<double*>(h->ws + L.diag_out);
  for (int i = 0; i < 5; ++i) h->R[i] = h->ws + L.R[i];
  for (int i = 0; i < 5; ++i) h->Tm[i] = h->ws + L.Tm[i];
  for (int i = 0; i < 3; ++i) h->S[i] = h->ws + L.S[i];
  h->initialized = false; h->t = 0.0; h->step = 0; h->launches = 0; h->sticky = 0;
  h->graph_exec = h->graph_exec_k = nullptr; h->graph_ok = false; h->advection_form = TTSH_ADVECTION_CONSERVATIVE;
  h->row_step_ok = h->dtype == TTSH_F64 ? row_step_supported<double>(h->g) : row_step_supported<float>(h->g);
  h->row_step_real = h->dtype == TTSH_F64 ? row_step_is_real<double>(h->g) : row_step_is_real<float>(h->g);
  h->row_step_wl = Nx == 4096;
  h->rs_tab = h->row_step_real ? (Nx == 16384 ? h->tabX : h->tabXw) : (h->row_step_wl ? h->tabXw : h->tabX);
  h->real_rows = Nx == 16384;
  h->rs_slots = h->rs_slots_ens = h->rs_slots_tan = 0;
  h->col_step_ok = h->row_step_ok && !h->real_rows &&
                   (h->dtype == TTSH_F64 ? col_step_supported<double>(h->g) : col_step_supported<float>(h->g));
  h->inter_valid = false;
  h->device = -1;
  *out = h;   // from here on errors are reported through the handle (caller destroys it)

  {   // the device of the workspace must be the current one
    int dev = -1;
    TRY(h, cudaGetDevice(&dev));
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, workspace) == cudaSuccess && at.type == cudaMemoryTypeDevice && at.device != dev) {
      h->err = "the workspace is not on the current CUDA device";
      h->sticky = TTSH_ERR_INVALID_ARG;
      return TTSH_ERR_INVALID_ARG;
    }
    (void)cudaGetLastError();
    h->device = dev;
  }
  std::vector<unsigned char> tx, ty, ts;
  const int Nrow = h->real_rows ? Nx / 2 : Nx;       // length of the complex row transform
  if (t == TTSH_F64) { fill_stage_tables<double>(tx, Nrow); fill_stage_tables<double>(ty, Ny / 2); fill_split_table<double>(ts, Ny); }
  else { fill_stage_tables<float>(tx, Nrow); fill_stage_tables<float>(ty, Ny / 2); fill_split_table<float>(ts, Ny); }
  if (h->real_rows) {      // W_Nx^j, j < Nx/32: the split / merge twiddles of the real-row passes
    std::vector<unsigned char> tr((size_t)(Nx / 32) * 2 * (size_t)t);
    for (int j = 0; j < Nx / 32; ++j) {
      if (t == TTSH_F64) put_twiddle<double>(reinterpret_cast<double*>(tr.data()) + 2 * (size_t)j, j, Nx);
      else put_twiddle<float>(reinterpret_cast<float*>(tr.data()) + 2 * (size_t)j, j, Nx);
    }
    TRY(h, cudaMemcpyAsync(h->tabXw, tr.data(), tr.size(), cudaMemcpyHostToDevice, h->stream));
    TRY(h, cudaStreamSynchronize(h->stream));
  }
  if (h->row_step_real && !h->real_rows) {     // warp-local tables of the half-length transform, then W_Nx^j, j < Nx/32
    std::vector<unsigned char> tw;
    const int off = DISPATCH(h, row_step_real_tabr, h->g);
    if (t == TTSH_F64) fill_stage_tables_wl<double>(tw, Nx / 2); else fill_stage_tables_wl<float>(tw, Nx / 2);
    tw.resize((size_t)(off + Nx / 32) * 2 * (size_t)t, 0);
    for (int j = 0; j < Nx / 32; ++j) {
      if (t == TTSH_F64) put_twiddle<double>(reinterpret_cast<double*>(tw.data()) + 2 * (size_t)(off + j), j, Nx);
      else put_twiddle<float>(reinterpret_cast<float*>(tw.data()) + 2 * (size_t)(off + j), j, Nx);
    }
    TRY(h, cudaMemcpyAsync(h->tabXw, tw.data(), tw.size(), cudaMemcpyHostToDevice, h->stream));
    TRY(h, cudaStreamSynchronize(h->stream));
  }
  if (h->row_step_wl) {
    std::vector<unsigned char> tw;
    if (t == TTSH_F64) fill_stage_tables_wl<double>(tw, Nx); else fill_stage_tables_wl<float>(tw, Nx);
    TRY(h, cudaMemcpyAsync(h->tabXw, tw.data(), tw.size(), cudaMemcpyHostToDevice, h->stream));
    TRY(h, cudaStreamSynchronize(h->stream));
  }
  TRY(h, cudaMemcpyAsync(h->tabX, tx.data(), tx.size(), cudaMemcpyHostToDevice, h->stream));
  std::vector<unsigned char> trx;
  if (h->row_step_real && h->real_rows) {      // Nx = 16384: the fused real-row kernel reads the plain tables of the half-length
                                               // transform (tabX) followed by W_Nx^j, j < Nx/32
    const int off = DISPATCH(h, row_step_real_tabr, h->g);
    trx.assign((size_t)(Nx / 32) * 2 * (size_t)t, 0);
    for (int j = 0; j < Nx / 32; ++j) {
      if (t == TTSH_F64) put_twiddle<double>(reinterpret_cast<double*>(trx.data()) + 2 * (size_t)j, j, Nx);
      else put_twiddle<float>(reinterpret_cast<float*>(trx.data()) + 2 * (size_t)j, j, Nx);
    }
    TRY(h, cudaMemcpyAsync(static_cast<char*>(h->tabX) + (size_t)off * 2 * (size_t)t, trx.data(), trx.size(), cudaMemcpyHostToDevice, h->stream));
  }
  TRY(h, cudaMemcpyAsync(h->tabY, ty.data(), ty.size(), cudaMemcpyHostToDevice, h->stream));
  TRY(h, cudaMemcpyAsync(h->tabS, ts.data(), ts.size(), cudaMemcpyHostToDevice, h->stream));
  TRY(h, cudaMemsetAsync(h->v0, 0, 8 * sizeof(double), h->stream));
  TRY(h, cudaStreamSynchronize(h->stream));   // the host tables go out of scope below
  TRY(h, DISPATCH(h, prepare_rows, h->g));
  TRY(h, DISPATCH(h, prepare_cols, h->g));
  if (h->row_step_ok) TRY(h, DISPATCH(h, prepare_row_step, h->g, &h->rs_slots, &h->rs_slots_ens, &h->rs_slots_tan));
  return apply_mask(h, mask, kind);
}

int ttsh_set_mask(ttsh_handle* h, const void* mask, ttsh_mask_kind kind) {
  if (!h) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (kind != TTSH_MASK_BINARY && kind != TTSH_MASK_PROCESSED) return TTSH_ERR_INVALID_ARG;
  return apply_mask(h, mask, kind);
}

int ttsh_set_velocity(ttsh_handle* h, const void* vx, const void* vy) {
  if (!h || !vx || !vy) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  const void* src[2] = {vx, vy};
  int rc = enqueue_forward(h, 2, src);
  if (rc != TTSH_OK) return rc;
  TRY(h, DISPATCH(h, launch_spectral_init, h->g, h->S[0], h->S[1], h->what, h->psihat, h->v0, h->stream));
  h->launches++;
  h->initialized = true;
  h->t = 0.0;
  h->step = 0;
  return TTSH_OK;
}

int ttsh_set_advection_form(ttsh_handle* h, int form) {
  if (!h || (form != TTSH_ADVECTION_CONSERVATIVE && form != TTSH_ADVECTION_LITERAL)) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (form != h->advection_form) {   // the captured steps no longer match
    if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
    if (h->graph_exec_k) cudaGraphExecDestroy(h->graph_exec_k);
    h->graph_exec = h->graph_exec_k = nullptr;
    h->graph_ok = false;
  }
  h->advection_form = form;
  h->inter_valid = false;
  return TTSH_OK;
}

int ttsh_step(ttsh_handle* h, int n) {
  if (!h || n < 0) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (!h->initialized) return TTSH_ERR_NOT_INITIALIZED;
  if (n == 0) return TTSH_OK;
  // Small grids are launch-latency bound: replay captured steps.  Up to 1024^2 one step per graph launch; up to 256^2, where the
  // four kernels of a step take about as long as a graph launch costs on the host, GRAPH_K steps per launch.  Large grids launch
  // directly.  Replays are bit-identical to direct launches (same kernels, same order).
  constexpr int GRAPH_K = 16;
  if (launches_per_step(h) == 2 && !h->inter_valid) {   // fused column kernel: the captured steps start at the row kernel
    int rc = enqueue_stage(h, TTSH_STAGE_INV_COL);
    if (rc != TTSH_OK) return rc;
    h->inter_valid = true;
  }
  const size_t P = (size_t)h->Nx * h->Ny;
  const bool use_graph = P <= (size_t)1024 * 1024 && n >= 4;
  const bool use_k = P <= (size_t)256 * 256 && n >= GRAPH_K;
  auto capture = [&](int steps, cudaGraphExec_t* out) -> int {
    // capture on a private stream (the caller's may be the legacy default stream, which cannot capture);
    // the instantiated graph is then replayed on the caller's stream.
    cudaGraph_t graph = nullptr;
    cudaStream_t cap = nullptr;
    const long long before = h->launches;
    TRY(h, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaStream_t user = h->stream;
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) { cudaStreamDestroy(cap); return fail_cuda(h, e, "cudaStreamBeginCapture"); }
    h->stream = cap;
    int rc = TTSH_OK;
    for (int i = 0; i < steps && rc == TTSH_OK; ++i) rc = enqueue_step(h);
    h->stream = user;
    e = cudaStreamEndCapture(cap, &graph);
    cudaStreamDestroy(cap);
    h->launches = before;
    if (rc != TTSH_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail_cuda(h, e, "cudaStreamEndCapture");
    e = cudaGraphInstantiate(out, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { *out = nullptr; return fail_cuda(h, e, "cudaGraphInstantiate"); }
    return TTSH_OK;
  };
  if (use_graph && !h->graph_ok) {
    int rc = capture(1, &h->graph_exec);
    if (rc != TTSH_OK) return rc;
    h->graph_ok = true;
  }
  if (use_k && !h->graph_exec_k) {
    int rc = capture(GRAPH_K, &h->graph_exec_k);
    if (rc != TTSH_OK) return rc;
  }
  int left = n;
  while (use_k && left >= GRAPH_K) {
    TRY(h, cudaGraphLaunch(h->graph_exec_k, h->stream));
    h->launches += (long long)GRAPH_K * launches_per_step(h);
    left -= GRAPH_K;
  }
  for (; left > 0; --left) {
    if (use_graph) {
      TRY(h, cudaGraphLaunch(h->graph_exec, h->stream));
      h->launches += launches_per_step(h);
    } else {
      int rc = enqueue_step(h);
      if (rc != TTSH_OK) return rc;
    }
  }
  h->t += (double)n * h->dt;
  h->step += n;
  return TTSH_OK;
}

int ttsh_get_fields(ttsh_handle* h, void* vx, void* vy, void* omega, void* psi) {
  if (!h) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (!h->initialized) return TTSH_ERR_NOT_INITIALIZED;
  return enqueue_inverse(h, omega, nullptr, nullptr, vx, vy, psi);
}

size_t ttsh_state_elems(const ttsh_handle* h) { return h ? (size_t)h->g.Wx * h->g.Hy : 0; }

int ttsh_get_state(ttsh_handle* h, void* w_hat, double* mean_flow) {
  if (!h || !w_hat || !mean_flow) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (!h->initialized) return TTSH_ERR_NOT_INITIALIZED;
  TRY(h, DISPATCH(h, launch_state_pack, h->g, h->what, w_hat, h->stream));
  h->launches++;
  TRY(h, cudaMemcpyAsync(mean_flow, h->v0, 2 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  TRY(h, cudaStreamSynchronize(h->stream));
  return TTSH_OK;
}

int ttsh_set_state(ttsh_handle* h, const void* w_hat, const double* mean_flow, double t, long long step) {
  if (!h || !w_hat || !mean_flow) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  h->inter_valid = false;
  TRY(h, DISPATCH(h, launch_state_unpack, h->g, w_hat, h->what, h->stream));
  h->launches++;
  TRY(h, cudaMemcpyAsync(h->v0, mean_flow, 2 * sizeof(double), cudaMemcpyHostToDevice, h->stream));
  TRY(h, DISPATCH(h, launch_psi_from_w, h->g, h->what, h->psihat, h->stream));
  h->launches++;
  TRY(h, cudaStreamSynchronize(h->stream));
  h->initialized = true;
  h->t = t;
  h->step = step;
  return TTSH_OK;
}

int ttsh_diagnostics(ttsh_handle* h, double cx, double cy, ttsh_diag* host_out) {
  if (!h || !host_out) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (!h->initialized) return TTSH_ERR_NOT_INITIALIZED;
  int rc = enqueue_inverse(h, h->R[0], nullptr, nullptr, h->R[3], h->R[4], nullptr);
  if (rc != TTSH_OK) return rc;
  TRY(h, DISPATCH(h, launch_diag, h->g, h->dx, cx, cy, h->R[3], h->R[4], h->R[0], h->diag_partial, h->diag_out, h->stream));
  h->launches += 2;
  double rec[8];
  TRY(h, cudaMemcpyAsync(rec, h->diag_out, sizeof(rec), cudaMemcpyDeviceToHost, h->stream));
  TRY(h, cudaStreamSynchronize(h->stream));
  const double P = (double)h->Nx * (double)h->Ny;
  ttsh_diag d;
  d.t = h->t; d.step = h->step;
  d.kinetic_energy = 0.5 * rec[0] / P;
  d.enstrophy = 0.5 * rec[1] / P;
  d.sum_speed = rec[2]; d.sum_abs_vtheta = rec[3];
  d.mean_vx = rec[4] / P; d.mean_vy = rec[5] / P;
  d.max_speed = rec[6];
  d.nonfinite = (long long)rec[7];
  if (rec[2] > 0.0) {
    const double two_over_pi = 2.0 / acos(-1.0);
    d.vortex_order = (rec[3] / rec[2] - two_over_pi) / (1.0 - two_over_pi);   // Eq. (11)
    d.polar_order = hypot(rec[4], rec[5]) / rec[2];
  } else {
    d.vortex_order = 0.0;
    d.polar_order = 0.0;
  }
  *host_out = d;
  return TTSH_OK;
}

int ttsh_dumbbell_order(ttsh_handle* h, double cxl, double cyl, double cxr, double cyr, double radius, ttsh_psi2* host_out) {
  if (!h || !host_out || !(radius >= 0.0) || !std::isfinite(radius)) return TTSH_ERR_INVALID_ARG;
  if (!std::isfinite(cxl) || !std::isfinite(cyl) || !std::isfinite(cxr) || !std::isfinite(cyr)) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (!h->initialized) return TTSH_ERR_NOT_INITIALIZED;
  int rc = enqueue_inverse(h, h->R[0], nullptr, nullptr, nullptr, nullptr, nullptr);
  if (rc != TTSH_OK) return rc;
  TRY(h, DISPATCH(h, launch_region_argmax, h->g, h->dx, cxl, cyl, cxr, cyr, radius, h->R[0], h->diag_partial, h->diag_out, h->stream));
  h->launches += 2;
  double rec[6];
  TRY(h, cudaMemcpyAsync(rec, h->diag_out, sizeof(rec), cudaMemcpyDeviceToHost, h->stream));
  TRY(h, cudaStreamSynchronize(h->stream));
  ttsh_psi2 d;
  d.index_left = (long long)rec[2]; d.index_right = (long long)rec[5];
  d.omega_left = d.index_left >= 0 ? rec[1] : 0.0;
  d.omega_right = d.index_right >= 0 ? rec[4] : 0.0;
  const double den = fabs(d.omega_left) + fabs(d.omega_right);
  d.psi2 = (den > 0.0 && d.index_left >= 0 && d.index_right >= 0) ? fabs(d.omega_left + d.omega_right) / den : 0.0;
  *host_out = d;
  return TTSH_OK;
}

// ---- streaming temporal PSD (Eq. 5) ------------------------------------------------------------------------
struct PsdLayout { size_t acc, partial, out, total; };
static PsdLayout psd_layout(int Nx, int Ny, size_t w, int nfreq) {
  PsdLayout L;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
  L.acc = take((size_t)nfreq * Nx * Ny * 2 * w);
  L.partial = take((size_t)nfreq * psd_blocks() * sizeof(double));
  L.out = take((size_t)nfreq * sizeof(double));
  L.total = off;
  return L;
}
size_t ttsh_psd_workspace_bytes(int Nx, int Ny, ttsh_dtype t, int nfreq) {
  if (!pow2_in_range(Nx) || !pow2_in_range(Ny) || (t != TTSH_F64 && t != TTSH_F32) || nfreq < 1 || nfreq > 1024) return 0;
  return psd_layout(Nx, Ny, (size_t)t, nfreq).total;
}
int ttsh_psd_create(ttsh_psd** out, ttsh_handle* h, const double* omegas, int nfreq, void* workspace, size_t workspace_bytes) {
  if (!out) return TTSH_ERR_INVALID_ARG;
  *out = nullptr;
  if (!h || !omegas || !workspace || nfreq < 1 || nfreq > 1024) return TTSH_ERR_INVALID_ARG;
  if (reinterpret_cast<uintptr_t>(workspace) % ALIGN) return TTSH_ERR_INVALID_ARG;
  for (int m = 0; m < nfreq; ++m) if (!std::isfinite(omegas[m])) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  const PsdLayout L = psd_layout(h->Nx, h->Ny, (size_t)h->dtype, nfreq);
  if (workspace_bytes < L.total) return TTSH_ERR_WORKSPACE_TOO_SMALL;
  ttsh_psd* s = new (std::nothrow) ttsh_psd();
  if (!s) return TTSH_ERR_INVALID_ARG;
  s->h = h;
  s->omegas.assign(omegas, omegas + nfreq);
  s->cs.resize(nfreq); s->sn.resize(nfreq);
  char* ws = static_cast<char*>(workspace);
  s->acc = ws + L.acc;
  s->acc_bytes = (size_t)nfreq * h->Nx * h->Ny * 2 * (size_t)h->dtype;
  s->partial = reinterpret_cast<double*>(ws + L.partial);
  s->out = reinterpret_cast<double*>(ws + L.out);
  s->nsamples = 0;
  *out = s;
  TRY(h, cudaMemsetAsync(s->acc, 0, s->acc_bytes, h->stream));
  return TTSH_OK;
}
int ttsh_psd_accumulate(ttsh_psd* s) {
  if (!s) return TTSH_ERR_INVALID_ARG;
  ttsh_handle* h = s->h;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (!h->initialized) return TTSH_ERR_NOT_INITIALIZED;
  int rc = enqueue_inverse(h, h->R[0], nullptr, nullptr, nullptr, nullptr, nullptr);     // w(., t)
  if (rc != TTSH_OK) return rc;
  const int nf = (int)s->omegas.size();
  for (int m = 0; m < nf; ++m) { s->cs[m] = cos(s->omegas[m] * h->t); s->sn[m] = -sin(s->omegas[m] * h->t); }
  TRY(h, DISPATCH(h, launch_psd_accumulate, (size_t)h->Nx * h->Ny, nf, s->cs.data(), s->sn.data(), h->R[0], s->acc, h->stream));
  h->launches += (nf + 63) / 64;
  s->nsamples++;
  return TTSH_OK;
}
int ttsh_psd_result(ttsh_psd* s, double* S_host, long long* nsamples_host) {
  if (!s || !S_host) return TTSH_ERR_INVALID_ARG;
  ttsh_handle* h = s->h;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  const int nf = (int)s->omegas.size();
  TRY(h, DISPATCH(h, launch_psd_power, (size_t)h->Nx * h->Ny, nf, s->acc, s->partial, s->out, h->stream));
  h->launches += 2;
  TRY(h, cudaMemcpyAsync(S_host, s->out, (size_t)nf * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  TRY(h, cudaStreamSynchronize(h->stream));
  const double P = (double)h->Nx * (double)h->Ny;
  for (int m = 0; m < nf; ++m) S_host[m] /= P;
  if (nsamples_host) *nsamples_host = s->nsamples;
  return TTSH_OK;
}
int ttsh_psd_reset(ttsh_psd* s) {
  if (!s) return TTSH_ERR_INVALID_ARG;
  if (s->h->sticky) return s->h->sticky;
  CHECK_DEVICE(s->h);
  TRY(s->h, cudaMemsetAsync(s->acc, 0, s->acc_bytes, s->h->stream));
  s->nsamples = 0;
  return TTSH_OK;
}
int ttsh_psd_destroy(ttsh_psd* s) {
  delete s;
  return TTSH_OK;
}

// ---- tangent-linear evolution and QR growth rates -----------------------------------------
// Every vector owns one block of the workspace — dw^, dpsi^, dv^(0), three real fields, three intermediates, three spectra —
// and the blocks lie at a uniform stride, so one launch of each kernel serves ALL vectors (the member dimension of the
// kernels, as in ttsh_ensemble_step): a tangent step costs 7 launches whatever nvec is.
struct TanLayout { size_t what, psihat, v0, real[3], inter[3], spec[3], vec_stride, vec, partial, coef, rdiag, gram, total; };
static TanLayout tan_layout(int Nx, int Ny, size_t w, int nvec) {
  const Geom g = make_geom(Nx, Ny, 1.0, 2, 3, w);
  const size_t cw = 2 * w, P = (size_t)Nx * Ny;
  const size_t spec = (size_t)g.NT * g.CW * g.Hy * cw, inter = (size_t)g.NT * g.CW * Ny * cw;
  TanLayout L;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
  L.what = take(spec); L.psihat = take(spec); L.v0 = take(8 * sizeof(double));
  for (int i = 0; i < 3; ++i) L.real[i] = take(P * w);
  for (int i = 0; i < 3; ++i) L.inter[i] = take(inter);
  for (int i = 0; i < 3; ++i) L.spec[i] = take(spec);
  L.vec_stride = off;
  off = 0;
  L.vec = take(L.vec_stride * nvec);
  L.partial = take((size_t)DIAG_BLOCKS * nvec * nvec * sizeof(double));
  L.coef = take((size_t)(nvec + 8) * sizeof(double));
  L.rdiag = take((size_t)nvec * sizeof(double));
  L.gram = take((size_t)2 * nvec * nvec * sizeof(double));     // Gram matrix, R^-1
  L.total = off;
  return L;
}
size_t ttsh_tangent_workspace_bytes(int Nx, int Ny, ttsh_dtype t, int nvec) {
  if (!pow2_in_range(Nx) || !pow2_in_range(Ny) || (t != TTSH_F64 && t != TTSH_F32) || nvec < 1 || nvec > 64) return 0;
  return tan_layout(Nx, Ny, (size_t)t, nvec).total;
}
int ttsh_tangent_create(ttsh_tangent** out, ttsh_handle* h, int nvec, void* workspace, size_t workspace_bytes) {
  if (!out) return TTSH_ERR_INVALID_ARG;
  *out = nullptr;
  if (!h || !workspace || nvec < 1 || nvec > 64) return TTSH_ERR_INVALID_ARG;
  if (reinterpret_cast<uintptr_t>(workspace) % ALIGN) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (h->advection_form != TTSH_ADVECTION_CONSERVATIVE) return TTSH_ERR_INVALID_ARG;
  const TanLayout L = tan_layout(h->Nx, h->Ny, (size_t)h->dtype, nvec);
  if (workspace_bytes < L.total) return TTSH_ERR_WORKSPACE_TOO_SMALL;
  ttsh_tangent* s = new (std::nothrow) ttsh_tangent();
  if (!s) return TTSH_ERR_INVALID_ARG;
  char* ws = static_cast<char*>(workspace);
  s->h = h;
  s->nvec = nvec;
  s->stride = L.vec_stride;
  s->set.assign(nvec, false);
  char* v = ws + L.vec;                     // block of vector 0; vector i is at + i * stride
  s->what = v + L.what; s->psihat = v + L.psihat; s->v0 = reinterpret_cast<double*>(v + L.v0);
  for (int i = 0; i < 3; ++i) { s->real[i] = v + L.real[i]; s->inter[i] = v + L.inter[i]; s->spec[i] = v + L.spec[i]; }
  s->partial = reinterpret_cast<double*>(ws + L.partial);
  s->coef = reinterpret_cast<double*>(ws + L.coef);
  s->rdiag = reinterpret_cast<double*>(ws + L.rdiag);
  s->gram = reinterpret_cast<double*>(ws + L.gram);
  *out = s;
  TRY(h, cudaMemsetAsync(ws + L.vec, 0, L.vec_stride * nvec, h->stream));
  return TTSH_OK;
}
int ttsh_tangent_set(ttsh_tangent* s, int i, const void* dvx, const void* dvy) {
  if (!s || i < 0 || i >= s->nvec || !dvx || !dvy) return TTSH_ERR_INVALID_ARG;
  ttsh_handle* h = s->h;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  const void* src[2] = {dvx, dvy};
  int rc = enqueue_forward(h, 2, src);
  if (rc != TTSH_OK) return rc;
  TRY(h, DISPATCH(h, launch_spectral_init, h->g, h->S[0], h->S[1], vec_ptr(s, s->what, i), vec_ptr(s, s->psihat, i), vec_ptr(s, s->v0, i), h->stream));
  h->launches++;
  s->set[i] = true;
  return TTSH_OK;
}
// inverse transforms of `count` vectors starting at vector `first` into dw, dvx, dvy (vector `first`'s buffers; the others
// at + stride): permuted internal row layout if perm, else natural; any destination may be NULL
static int tangent_inverse(ttsh_tangent* s, int first, int count, void* dw, void* dvx, void* dvy, bool perm, size_t dst_stride) {
  ttsh_handle* h = s->h;
  const int pf = perm ? RM_PERM : 0;
  Batch cb; memset(&cb, 0, sizeof(cb));
  Batch rb; memset(&rb, 0, sizeof(rb));
  void* what = vec_ptr(s, s->what, first);
  void* psihat = vec_ptr(s, s->psihat, first);
  double* v0 = vec_ptr(s, s->v0, first);
  void* t0 = vec_ptr(s, s->inter[0], first);
  void* t1 = vec_ptr(s, s->inter[1], first);
  void* t2 = vec_ptr(s, s->inter[2], first);
  int nc = 0, nr = 0;
  if (dw) { cb.f[nc++] = op(what, t0, SM_ONE); rb.f[nr++] = op(t0, dw, RM_ONE | pf); }
  if (dvy) { cb.f[nc++] = op(psihat, t1, SM_ONE); rb.f[nr++] = op(t1, dvy, RM_NIKX_MEANY | pf); }
  if (dvx) { cb.f[nc++] = op(psihat, t2, SM_IKY_MEANX); rb.f[nr++] = op(t2, dvx, RM_ONE | pf); }
  if (nc == 0) return TTSH_OK;
  TRY(h, DISPATCH(h, launch_inv_col, h->g, cb, nc, h->tabY, h->tabS, v0, h->stream, count, s->stride));
  if (count == 1 || dst_stride == s->stride) {
    TRY(h, DISPATCH(h, launch_inv_row, h->g, rb, nr, h->tabX, h->tabXw, v0, h->stream, count, s->stride));
  } else return TTSH_ERR_INVALID_ARG;
  h->launches += 2;
  return TTSH_OK;
}
int ttsh_tangent_step(ttsh_tangent* s, int n) {
  if (!s || n < 0) return TTSH_ERR_INVALID_ARG;
  ttsh_handle* h = s->h;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (!h->initialized) return TTSH_ERR_NOT_INITIALIZED;
  if (h->advection_form != TTSH_ADVECTION_CONSERVATIVE) return TTSH_ERR_INVALID_ARG;
  for (int i = 0; i < s->nvec; ++i) if (!s->set[i]) return TTSH_ERR_NOT_INITIALIZED;
  const int M = s->nvec;
  const size_t ms = s->stride;
  for (int it = 0; it < n; ++it) {
    // base state in real space (permuted internal layout): R[0] = w, R[3] = v_x, R[4] = v_y
    h->inter_valid = false;
    int rc = enqueue_stage(h, TTSH_STAGE_INV_COL);
    if (rc == TTSH_OK) rc = enqueue_stage(h, TTSH_STAGE_INV_ROW);
    if (rc != TTSH_OK) return rc;
    if (h->row_step_ok && h->rs_slots_tan > 0) {
      // all vectors at once, fused (row_step.cuh, TAN): inverse column pass of (dw^, dpsi^, i k_y dpsi^), then ONE kernel for the
      // inverse row transforms, the linearised lines 1-2 at the base state (R[0], R[3], R[4], K) and the forward row transforms
      // into dA~ = i k_x dGy~ + dS'~ and dB~ = dGx~ (parked in the vectors' real scratch), column pass, lines 3-16 (linear).
      Batch cb = make_batch({op(s->what, s->inter[0], SM_ONE), op(s->psihat, s->inter[1], SM_ONE), op(s->psihat, s->inter[2], SM_IKY_MEANX)});
      TRY(h, DISPATCH(h, launch_inv_col, h->g, cb, 3, h->tabY, h->tabS, s->v0, h->stream, M, ms));
      TRY(h, DISPATCH(h, launch_row_step_tan, h->g, h->m, s->inter[0], s->inter[2], s->inter[1], h->K, s->real[0], s->real[1], h->tabX, s->v0,
                      h->stream, M, ms, h->rs_slots_tan, h->R[0], h->R[3], h->R[4]));
      Batch fb = make_batch({op(s->real[0], s->spec[0], 0), op(s->real[1], s->spec[1], 0)});
      TRY(h, DISPATCH(h, launch_fwd_col, h->g, fb, 2, h->tabY, h->tabS, h->stream, M, ms));
      TRY(h, DISPATCH(h, launch_spectral_p2, h->g, h->m, s->spec[0], s->spec[1], s->what, s->psihat, s->v0, h->stream, M, ms));
      h->launches += 4;
    } else {
    // all vectors at once: dw, dv_x, dv_y -> linearised lines 1-2 in place -> three forward transforms -> lines 3-16
    rc = tangent_inverse(s, 0, M, s->real[0], s->real[1], s->real[2], true, ms);
    if (rc != TTSH_OK) return rc;
    TRY(h, DISPATCH(h, launch_realspace_tangent, h->g, h->m, h->R[3], h->R[4], h->R[0], h->K, s->real[1], s->real[2], s->real[0], h->stream, M, ms));
    Batch rb = make_batch({op(s->real[1], s->inter[0], RM_PERM), op(s->real[2], s->inter[1], RM_PERM), op(s->real[0], s->inter[2], RM_PERM)});
    TRY(h, DISPATCH(h, launch_fwd_row, h->g, rb, 3, h->tabX, h->tabXw, h->stream, M, ms));
    Batch cb = make_batch({op(s->inter[0], s->spec[0], 0), op(s->inter[1], s->spec[1], 0), op(s->inter[2], s->spec[2], 0)});
    TRY(h, DISPATCH(h, launch_fwd_col, h->g, cb, 3, h->tabY, h->tabS, h->stream, M, ms));
    // lines 3-16 are linear: the same spectral kernel on the perturbations' (dw^, dpsi^, dv^(0))
    TRY(h, DISPATCH(h, launch_spectral, h->g, h->m, s->spec[0], s->spec[1], s->spec[2], s->what, s->psihat, s->v0, h->stream, M, ms));
    h->launches += 4;
    }
    rc = ttsh_step(h, 1);
    if (rc != TTSH_OK) return rc;
  }
  return TTSH_OK;
}
// modified Gram-Schmidt on the device (the fallback of the blocked QR below): all coefficients stay on the device; row i of R in
// one batched launch per operation: r_ii = |q_i|, q_i /= r_ii, then r_ij = <q_i, q_j> and q_j -= r_ij q_i for all j > i together.
// Adds log r_ii to log_r_host.
static int tangent_mgs(ttsh_tangent* s, double* log_r_host) {
  ttsh_handle* h = s->h;
  for (int i = 0; i < s->nvec; ++i) {
    void* qi = vec_ptr(s, s->what, i);
    double* qi0 = vec_ptr(s, s->v0, i);
    TRY(h, DISPATCH(h, launch_spec_dot, h->g, qi, qi, qi0, qi0, 1, 0, i, s->partial, s->rdiag, s->coef, h->stream));
    TRY(h, DISPATCH(h, launch_spec_scale_axpy, h->g, s->coef, nullptr, qi, nullptr, qi0, 1, 0, h->stream));
    h->launches += 3;
    const int rest = s->nvec - i - 1;
    if (rest > 0) {
      void* qj = vec_ptr(s, s->what, i + 1);
      double* qj0 = vec_ptr(s, s->v0, i + 1);
      TRY(h, DISPATCH(h, launch_spec_dot, h->g, qi, qj, qi0, qj0, rest, s->stride, -1, s->partial, s->rdiag, s->coef, h->stream));
      TRY(h, DISPATCH(h, launch_spec_scale_axpy, h->g, s->coef, qi, qj, qi0, qj0, rest, s->stride, h->stream));
      h->launches += 3;
    }
  }
  for (int i = 0; i < s->nvec; ++i) {
    TRY(h, DISPATCH(h, launch_psi_from_w, h->g, vec_ptr(s, s->what, i), vec_ptr(s, s->psihat, i), h->stream));
    h->launches++;
  }
  std::vector<double> r(s->nvec);
  TRY(h, cudaMemcpyAsync(r.data(), s->rdiag, (size_t)s->nvec * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  TRY(h, cudaStreamSynchronize(h->stream));
  for (int i = 0; i < s->nvec; ++i) log_r_host[i] += log(r[i]);
  return TTSH_OK;
}

// QR of the current vectors, R_ii > 0.  Blocked: CholeskyQR2 — G = A^T A, R = chol(G) and R^-1 (one small block), A <- A R^-1,
// all on the device, twice (the second pass restores orthogonality to round-off; R = R2 R1, so log R_ii = log R1_ii + log R2_ii).  A
// Cholesky pivot below 1e-13 of its diagonal entry (vectors that are numerically dependent at the level where the Gram matrix
// loses them, cond(A) > ~3e6) sends the remaining work to modified Gram-Schmidt instead.
int ttsh_tangent_orthonormalize(ttsh_tangent* s, double* log_r_host) {
  if (!s || !log_r_host) return TTSH_ERR_INVALID_ARG;
  ttsh_handle* h = s->h;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  for (int i = 0; i < s->nvec; ++i) if (!s->set[i]) return TTSH_ERR_NOT_INITIALIZED;
  const int M = s->nvec;
  // device scratch: gram = G[M][M] | S[M][M]; rdiag = log R_ii accumulated over the two passes; coef[M + 1 ..] holds the flag
  double* Sdev = s->gram + (size_t)M * M;
  int* flag = reinterpret_cast<int*>(s->coef + M + 2);
  TRY(h, cudaMemsetAsync(s->rdiag, 0, (size_t)M * sizeof(double), h->stream));
  TRY(h, cudaMemsetAsync(flag, 0, sizeof(int), h->stream));
  for (int pass = 0; pass < 2; ++pass) {
    TRY(h, DISPATCH(h, launch_gram, h->g, s->what, s->v0, s->stride, M, s->partial, s->gram, h->stream));
    TRY(h, launch_chol_inv(M, s->gram, Sdev, s->rdiag, flag, h->stream));
    TRY(h, DISPATCH(h, launch_tri_apply, h->g, M, Sdev, s->what, s->psihat, s->v0, s->stride, h->stream));
    h->launches += 4;
  }
  int bad = 0;
  TRY(h, cudaMemcpyAsync(log_r_host, s->rdiag, (size_t)M * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  TRY(h, cudaMemcpyAsync(&bad, flag, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
  TRY(h, cudaStreamSynchronize(h->stream));
  if (bad) return tangent_mgs(s, log_r_host);      // adds its log r_ii to what a completed first pass recorded
  return TTSH_OK;
}
int ttsh_tangent_get_fields(ttsh_tangent* s, int i, void* dvx, void* dvy, void* domega) {
  if (!s || i < 0 || i >= s->nvec) return TTSH_ERR_INVALID_ARG;
  if (s->h->sticky) return s->h->sticky;
  CHECK_DEVICE(s->h);
  if (!s->set[i]) return TTSH_ERR_NOT_INITIALIZED;
  return tangent_inverse(s, i, 1, domega, dvx, dvy, false, 0);
}
int ttsh_tangent_destroy(ttsh_tangent* s) {
  delete s;
  return TTSH_OK;
}

// ---- ensembles -----------------------------------------------------------------------------------------------
int ttsh_ensemble_create(ttsh_ensemble** out, ttsh_handle* const* members, int count) {
  if (!out) return TTSH_ERR_INVALID_ARG;
  *out = nullptr;
  if (!members || count < 1 || count > 8192) return TTSH_ERR_INVALID_ARG;
  const ttsh_handle* h0 = members[0];
  if (!h0) return TTSH_ERR_INVALID_ARG;
  ptrdiff_t stride = 0;
  for (int b = 0; b < count; ++b) {
    const ttsh_handle* h = members[b];
    if (!h) return TTSH_ERR_INVALID_ARG;
    if (h->sticky) return h->sticky;
    if (h->Nx != h0->Nx || h->Ny != h0->Ny || h->dtype != h0->dtype || h->dx != h0->dx || h->dt != h0->dt ||
        h->stream != h0->stream || memcmp(&h->p, &h0->p, sizeof(ttsh_params)) != 0)
      return TTSH_ERR_INVALID_ARG;
    if (h->advection_form != TTSH_ADVECTION_CONSERVATIVE || !h->row_step_ok) return TTSH_ERR_INVALID_ARG;
    for (int a = 0; a < b; ++a) if (members[a] == h) return TTSH_ERR_INVALID_ARG;
    if (b == 1) stride = h->ws - h0->ws;
    if (b >= 1 && h->ws - h0->ws != (ptrdiff_t)b * stride) return TTSH_ERR_INVALID_ARG;
  }
  if (count > 1 && stride < (ptrdiff_t)make_layout(h0->Nx, h0->Ny, (size_t)h0->dtype).total) return TTSH_ERR_INVALID_ARG;
  ttsh_ensemble* e = new (std::nothrow) ttsh_ensemble();
  if (!e) return TTSH_ERR_INVALID_ARG;
  e->members.assign(members, members + count);
  e->mstride = count > 1 ? (size_t)stride : 0;
  e->graph_exec = nullptr;
  e->launches = 0;
  {   // k_col_step runs ONE CTA per tile and member: it shortens the dependency chain of a step, which is what binds a small ensemble,
      // but has less throughput than the separate column passes, which is what binds a large one (C3 x 16: 454 vs 395 us per step)
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    e->col_fused = h0->col_step_ok && (long long)count * h0->g.NT <= 8LL * sms;
  }
  *out = e;
  return TTSH_OK;
}

// the column pass of a2 / a6 for all members (stage 0 of a step)
static int ensemble_enqueue_inv_col(ttsh_ensemble* e, cudaStream_t stream) {
  ttsh_handle* h = e->members[0];
  Batch cb = make_batch({op(h->what, h->Tm[0], SM_ONE), op(h->psihat, h->Tm[2], SM_ONE), op(h->psihat, h->Tm[3], SM_IKY_MEANX)});
  TRY(h, DISPATCH(h, launch_inv_col, h->g, cb, 3, h->tabY, h->tabS, h->v0, stream, (int)e->members.size(), e->mstride));
  return TTSH_OK;
}
// one Euler step of all members.  With the fused column kernel (e->col_fused) the step is k_row_step + k_col_step and
// expects the members' inverse intermediates at hand (ttsh_ensemble_step sees to that); else the four launches of ttsh_step.
static int ensemble_enqueue_step(ttsh_ensemble* e, cudaStream_t stream) {
  ttsh_handle* h = e->members[0];
  const int B = (int)e->members.size();
  const size_t ms = e->mstride;
  if (!e->col_fused) { const int rc = ensemble_enqueue_inv_col(e, stream); if (rc != TTSH_OK) return rc; }
  TRY(h, DISPATCH(h, launch_row_step_ens, h->g, h->m, h->Tm[0], h->Tm[3], h->Tm[2], (h->row_step_wl || h->row_step_real) ? h->K2 : h->K, h->Tm[1], h->Tm[4],
                  h->rs_tab, h->v0, stream, B, ms, h->rs_slots_ens));
  if (e->col_fused) {
    TRY(h, DISPATCH(h, launch_col_step, h->g, h->m, h->Tm[1], h->Tm[4], h->what, h->psihat, h->v0, h->Tm[0], h->Tm[2], h->Tm[3], h->tabY, h->tabS,
                    stream, B, ms));
    return TTSH_OK;
  }
  Batch fb = make_batch({op(h->Tm[1], h->S[0], 0), op(h->Tm[4], h->S[1], 0)});
  TRY(h, DISPATCH(h, launch_fwd_col, h->g, fb, 2, h->tabY, h->tabS, stream, B, ms));
  TRY(h, DISPATCH(h, launch_spectral_p2, h->g, h->m, h->S[0], h->S[1], h->what, h->psihat, h->v0, stream, B, ms));
  return TTSH_OK;
}

int ttsh_ensemble_step(ttsh_ensemble* e, int n) {
  if (!e || n < 0) return TTSH_ERR_INVALID_ARG;
  ttsh_handle* h0 = e->members[0];
  for (ttsh_handle* h : e->members) {
    if (h->sticky) return h->sticky;
    CHECK_DEVICE(h);
    if (!h->initialized) return TTSH_ERR_NOT_INITIALIZED;
    if (h->advection_form != TTSH_ADVECTION_CONSERVATIVE) return TTSH_ERR_INVALID_ARG;
  }
  if (n == 0) return TTSH_OK;
  const int per_step = e->col_fused ? 2 : 4;
  if (e->col_fused) {     // the captured / enqueued steps start at the row kernel: make every member's intermediates valid first
    bool valid = true;
    for (ttsh_handle* h : e->members) valid = valid && h->inter_valid;
    if (!valid) {
      const int rc = ensemble_enqueue_inv_col(e, h0->stream);
      if (rc != TTSH_OK) return rc;
      e->launches += 1;
    }
  }
  for (ttsh_handle* h : e->members) h->inter_valid = e->col_fused;      // k_col_step leaves them valid for every member
  // a step of a small ensemble is launch-latency bound: replay one captured step (as ttsh_step does)
  const bool use_graph = (size_t)h0->Nx * h0->Ny * e->members.size() <= (size_t)4 * 1024 * 1024 && n >= 4;
  if (use_graph && !e->graph_exec) {
    cudaGraph_t graph = nullptr;
    cudaStream_t cap = nullptr;
    TRY(h0, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaError_t err = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (err != cudaSuccess) { cudaStreamDestroy(cap); return fail_cuda(h0, err, "cudaStreamBeginCapture"); }
    const int rc = ensemble_enqueue_step(e, cap);
    err = cudaStreamEndCapture(cap, &graph);
    cudaStreamDestroy(cap);
    if (rc != TTSH_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (err != cudaSuccess) return fail_cuda(h0, err, "cudaStreamEndCapture");
    err = cudaGraphInstantiate(&e->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (err != cudaSuccess) { e->graph_exec = nullptr; return fail_cuda(h0, err, "cudaGraphInstantiate"); }
  }
  for (int i = 0; i < n; ++i) {
    if (use_graph) TRY(h0, cudaGraphLaunch(e->graph_exec, h0->stream));
    else {
      const int rc = ensemble_enqueue_step(e, h0->stream);
      if (rc != TTSH_OK) return rc;
    }
    e->launches += per_step;
  }
  for (ttsh_handle* h : e->members) {
    h->t += (double)n * h->dt;
    h->step += n;
  }
  return TTSH_OK;
}

long long ttsh_ensemble_launch_count(const ttsh_ensemble* e) { return e ? e->launches : 0; }

int ttsh_ensemble_destroy(ttsh_ensemble* e) {
  if (!e) return TTSH_OK;
  if (e->graph_exec) cudaGraphExecDestroy(e->graph_exec);
  delete e;
  return TTSH_OK;
}

long long ttsh_launch_count(const ttsh_handle* h) { return h ? h->launches : 0; }

int ttsh_run_stage(ttsh_handle* h, int stage) {
  if (!h) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  if (!h->initialized) return TTSH_ERR_NOT_INITIALIZED;
  h->inter_valid = false;
  return enqueue_stage(h, stage);
}

int ttsh_debug_get_real(ttsh_handle* h, int which, void* dst) {
  if (!h || !dst || which < 0 || which > 5) return TTSH_ERR_INVALID_ARG;
  if (h->sticky) return h->sticky;
  CHECK_DEVICE(h);
  const void* src = which == 5 ? h->K : h->R[which];   // internal fields are in the internal row layout
  return copy_real(h, src, dst, 0);
}

int ttsh_destroy(ttsh_handle* h) {
  if (!h) return TTSH_OK;
  if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
  if (h->graph_exec_k) cudaGraphExecDestroy(h->graph_exec_k);
  delete h;
  return TTSH_OK;
}

const char* ttsh_strerror(int code) {
  switch (code) {
    case TTSH_OK: return "ok";
    case TTSH_ERR_INVALID_ARG: return "invalid argument";
    case TTSH_ERR_UNSUPPORTED_SIZE: return "unsupported grid size (Nx, Ny must be powers of two in [64, 16384])";
    case TTSH_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case TTSH_ERR_NOT_INITIALIZED: return "state not initialised (call ttsh_set_velocity first)";
    case TTSH_ERR_CUDA: return "CUDA error";
  }
  return "unknown error";
}

const char* ttsh_last_error(const ttsh_handle* h) { return h ? h->err.c_str() : ""; }

#ifndef TTSH_SOURCE_HASH
#define TTSH_SOURCE_HASH "unknown"
#endif
const char* ttsh_build_info(void) {
  return "ttsh sm_100a sources=" TTSH_SOURCE_HASH " cuda=" TTSH_STR(__CUDACC_VER_MAJOR__) "." TTSH_STR(__CUDACC_VER_MINOR__) " built " __DATE__ " " __TIME__;
}

}  // extern "C"
