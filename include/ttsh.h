/* ttsh.h — C ABI of the B200-native pseudospectral TTSH step.
 *
 * What it computes: one call of ttsh_step(h, n) applies n times Algorithm 1 of
 * S. Shiratani, K. A. Takeuchi, D. Nishiguchi, arXiv:2304.03306 ("PAPER.md" below; Appendix C,
 * PAPER.md:286-331) — the integrating-factor Euler step of the 2-D incompressible
 * Toner-Tu-Swift-Hohenberg equation in vorticity form with the damping-mask boundary terms
 * of Eq. (4) — on a periodic Nx x Ny grid.  ttsh_create runs Algorithm 2
 * (mask processing, Appendix D) on a binary mask.
 *
 * General TTSH form (BASELINE.json:north_star), with the paper's model as a preset:
 *     d_t v + lambda0 v.grad v = -grad p - (alpha + beta |v|^2) v + Gamma0 lap v - Gamma2 lap^2 v
 *     paper (Eq. 2):  lambda0 = lambda, beta = b, alpha = 1 - a, Gamma0 = -2, Gamma2 = 1
 *     linear symbol  sigma(k) = -alpha - Gamma0 k^2 - Gamma2 k^4   ( = a - (1-k^2)^2, Alg. 1 line 4, PAPER.md:295 )
 *
 * Conventions
 *   - real fields: row-major scalar[Ny][Nx], x contiguous; point (i, j) sits at (i*dx, j*dx);
 *     the DFT phase origin is index (0,0).  scalar = double (TTSH_F64) or float (TTSH_F32).
 *   - every pointer documented "DEVICE" must be device memory of the current CUDA device, 16-byte
 *     aligned; "HOST" pointers are ordinary host memory.  The library allocates NO device memory:
 *     the caller owns the mask, the workspace, all field buffers and the stream; they are borrowed
 *     for the duration of the enqueued (stream-ordered) work and the workspace must outlive the handle.
 *   - all functions return 0 (TTSH_OK) or a negative ttsh_status; they never throw, abort or print.
 *   - all work is enqueued on the stream given to ttsh_create; only ttsh_diagnostics synchronises.
 *   - a handle belongs to the CUDA device that was current in ttsh_create (the device of its workspace); every later call
 *     on it must be made with that device current, else it returns TTSH_ERR_INVALID_ARG.
 *   - there is no CPU fallback: without a CUDA device every compute call returns TTSH_ERR_CUDA.
 */
#ifndef TTSH_H_
#define TTSH_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ttsh_handle ttsh_handle;   /* opaque; host metadata + pointers into the workspace */

typedef enum {
  TTSH_OK = 0,
  TTSH_ERR_INVALID_ARG = -1,         /* NULL pointer, n < 0, dx <= 0, dt <= 0, Gamma2 < 0, non-finite parameter, bad dealias fraction, wrong device */
  TTSH_ERR_UNSUPPORTED_SIZE = -2,    /* Nx, Ny must be powers of two in [64, 16384]: the paper's grids are 8192^2 and
                                        16384^2 for Fig. 6(f); BASELINE.json's are 64 .. 4096 */
  TTSH_ERR_WORKSPACE_TOO_SMALL = -3,
  TTSH_ERR_NOT_INITIALIZED = -4,     /* ttsh_step / get_fields / diagnostics before ttsh_set_velocity */
  TTSH_ERR_CUDA = -5                 /* sticky; message via ttsh_last_error */
} ttsh_status;

/* Parameters of Eq. (2)/(4).  Paper preset (Table I :264-274): {9, 0.5, 1.6, -2, 1, 40, 4, 1, 2};
 * BASELINE.json configs: {3.5, -0.5, 0.5, -1, 1, 40, 4, 1, 2}. */
typedef struct {
  double lambda0;      /* advection strength                                   */
  double alpha;        /* linear damping (= 1 - a)                             */
  double beta;         /* cubic nonlinearity (= b)                             */
  double Gamma0;       /* coefficient of lap v  (negative = active)            */
  double Gamma2;       /* coefficient of -lap^2 v, must be >= 0                */
  double gamma_v;      /* velocity damping strength in the masked area, Eq. (4) */
  double gamma_w;      /* vorticity damping strength in the masked area, Eq. (4) */
  int dealias_num;     /* anti-aliasing cutoff |k| <= (num/den) * pi/dx, strict '>' removes; */
  int dealias_den;     /* the paper's 1/2 rule is {1, 2}; allowed: 1/4 <= num/den <= 2/3                         */
} ttsh_params;

typedef enum { TTSH_F64 = 8, TTSH_F32 = 4 } ttsh_dtype;

typedef enum {
  TTSH_MASK_BINARY = 0,      /* unsigned char[Ny*Nx], nonzero = masked (K_naive = 1); Algorithm 2 is run on it */
  TTSH_MASK_PROCESSED = 1    /* scalar[Ny*Nx], used as K(x) as given (caller guarantees K >= 0 and band-limited)           */
} ttsh_mask_kind;

/* Bytes of DEVICE workspace ttsh_create needs for this grid and dtype; 0 if the size is unsupported. */
size_t ttsh_workspace_bytes(int Nx, int Ny, ttsh_dtype t);

/* Creates a handle.  mask: DEVICE pointer (see ttsh_mask_kind) or NULL for no confinement (K == 0, the
 * unconfined periodic run).  workspace: DEVICE, >= ttsh_workspace_bytes, 256-byte aligned.  cuda_stream: a
 * cudaStream_t owned by the caller (NULL = the legacy default stream).  Enqueues Algorithm 2:
 * K = ( iDFT[ lowpass_{1/4}( DFT[K_naive] ) ] )^2.  The mask buffer may be released after the stream has
 * passed this call. */
int ttsh_create(ttsh_handle** out, int Nx, int Ny, double dx, double dt, const ttsh_params* p, ttsh_dtype t,
                const void* mask, ttsh_mask_kind kind, void* workspace, size_t workspace_bytes,
                void* cuda_stream);

/* Replaces K(x) on a live handle (state is kept: the hysteresis protocol of PAPER.md:143). */
int ttsh_set_mask(ttsh_handle* h, const void* mask, ttsh_mask_kind kind);

/* Sets the state from a real velocity field (DEVICE scalar[Ny*Nx] each): w^ = i k_x v^_y - i k_y v^_x, mean
 * flow v^(0) kept, then lines 5-16 of Algorithm 1 (cutoff, w^(0) = 0, Hermitian symmetrisation, stream-function
 * inversion), i.e. v0 is projected onto band-limited divergence-free fields.  Resets t and the step counter. */
int ttsh_set_velocity(ttsh_handle* h, const void* vx, const void* vy);

/* How the advection term of Algorithm 1 line 2 is evaluated:
 *   TTSH_ADVECTION_CONSERVATIVE (default)  lambda0 div(v w): the products v_x w, v_y w are formed in real space and the
 *        divergence is taken spectrally, folded into line 3 ( rhs^ = i k_x (rhs1_y - lambda0 v_x w)^ - i k_y (rhs1_x +
 *        lambda0 v_y w)^ + (-gamma_w K w)^ ).  div v = 0 holds exactly for the stream-function velocity and
 *        all products are alias-free on the retained band, so this equals the literal form up to round-off (measured
 *        <= 1e-15 relative per step) while needing 3 instead of 5 inverse transforms per step.
 *   TTSH_ADVECTION_LITERAL                 lambda0 v . iDFT[i k w^], exactly as line 2 is printed.
 * Both are tested against the CPU oracle, which always evaluates the literal form. */
typedef enum { TTSH_ADVECTION_CONSERVATIVE = 0, TTSH_ADVECTION_LITERAL = 1 } ttsh_advection_form;
int ttsh_set_advection_form(ttsh_handle* h, int form);

/* n >= 0 applications of Algorithm 1; asynchronous; t += n*dt. */
int ttsh_step(ttsh_handle* h, int n);

/* Writes the current fields into caller-owned DEVICE buffers scalar[Ny*Nx]; any pointer may be NULL.
 * v = iDFT[v^] (state), omega = iDFT[w^], psi = iDFT[w^/k^2] with psi^(0) = 0. */
int ttsh_get_fields(ttsh_handle* h, void* vx, void* vy, void* omega, void* psi);

/* Bit-exact checkpoint of the spectral state: w_hat is DEVICE complex-scalar[ttsh_state_elems] (interleaved re, im), the retained
 * modes of w^ (unitary DFT) in natural order [Hy][Wx]: element (q, m_x) at q Wx + m_x, with m_x = 0 .. Wx - 1,
 * Wx - 1 = floor(num Nx / (2 den)), and row q <-> m_y = q for q <= My, q - Hy above, My = floor(num Ny / (2 den)), Hy = 2 My + 1
 * (num/den = the dealias fraction: nothing outside this rectangle is ever non-zero under the cutoff of PAPER.md:301).
 * ttsh_state_elems = Wx Hy depends on Nx, Ny and the dealias fraction only — not on the tile widths this binary was built with —
 * so a checkpoint written by one build of the library restores in any other on a handle of the same grid, dtype and parameters;
 * there is no header in the buffer: the caller stores (Nx, Ny, dtype, num/den) beside it.  mean_flow is HOST double[2] = v^(0).
 * Both calls synchronise the stream. */
size_t ttsh_state_elems(const ttsh_handle* h);
int ttsh_get_state(ttsh_handle* h, void* w_hat, double* mean_flow);
int ttsh_set_state(ttsh_handle* h, const void* w_hat, const double* mean_flow, double t, long long step);

/* Diagnostics (sums over the ENTIRE grid; always double):
 *   kinetic_energy = (1/2P) sum |v|^2,  enstrophy = (1/2P) sum w^2,
 *   vortex_order   = Psi of Eq. (11), with e_theta the azimuthal unit vector about (cx, cy)
 *                    (physical units); the grid point with r = 0 contributes to the denominator only;
 *   polar_order    = |sum v| / sum |v|;   both orders are 0 when sum |v| = 0.
 * host_out: HOST.  Synchronises the stream.  Returns TTSH_OK also when nonfinite > 0 (advisory). */
typedef struct {
  double t;
  long long step;
  double kinetic_energy, enstrophy, vortex_order, polar_order;
  double sum_speed, sum_abs_vtheta, mean_vx, mean_vy, max_speed;
  long long nonfinite;
} ttsh_diag;
int ttsh_diagnostics(ttsh_handle* h, double cx, double cy, ttsh_diag* host_out);

/* The same diagnostics for a caller that cannot hand the library any device memory: no handle, no workspace, just the three
 * fields.  Meant for code that is given field pointers and nothing else (a monitoring hook called from inside another solver's
 * time loop), for processes whose framework allocator already owns all device memory so that a raw cudaMalloc would fail, and
 * for loops that cannot afford the device-wide synchronisation cudaMalloc / cudaFree imply.  This call allocates nothing and
 * frees nothing: its only scratch (one partial record per thread block, 592 x 8 doubles = 37,888 bytes) is a static
 * __device__ array inside the library, which every GPU that loads the library carries until the process exits.
 *   vx, vy, omega  DEVICE scalar[Ny*Nx] in (row-major, x contiguous; scalar per `t`); read only.
 *   cx, cy         centre of e_theta in physical units, as in ttsh_diagnostics.
 *   sums           DEVICE double[8] out, caller-owned: sum|v|^2, sum w^2, sum|v|, sum|e_theta.v|, sum v_x, sum v_y, max|v|,
 *                  number of non-finite values among v_x, v_y, omega.
 *   host_out       HOST or NULL.  NULL: the call only enqueues two kernels on cuda_stream and returns; read `sums` in stream
 *                  order.  Non-NULL: additionally copies `sums` back, synchronises the stream and fills *host_out like
 *                  ttsh_diagnostics does (t and step are 0: there is no handle to keep time).
 *   cuda_stream    cudaStream_t of the caller (NULL = the default stream).
 * Limits: 1 <= Nx, Ny <= 16384 (any integers, not only powers of two), i.e. at most TTSH_NOALLOC_MAX_POINTS grid points — the
 * library's own largest grid; the scratch does not grow with the grid.  Larger sizes return TTSH_ERR_UNSUPPORTED_SIZE, bad
 * pointers / dtype / dx TTSH_ERR_INVALID_ARG, a CUDA failure TTSH_ERR_CUDA; ttsh_diagnostics_noalloc_error() gives the text of
 * the last failure of this call on the calling thread ("" after a success).
 * Things to know about the shared static scratch:
 *   - the first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device current,
 *     which may also load the library's code onto that device).  Make that first call before any stream capture begins.
 *   - every call on a device uses the same array.  A call overwrites all of it before reading it, so nothing left behind by
 *     an earlier call (of any grid size or dtype) matters; but two calls whose kernels can run at the same time — different
 *     streams without an event between them — race on it and both results are undefined.  Serialise them.
 * The sums equal those of ttsh_diagnostics on the same fields (same arithmetic, same launch shape). */
#define TTSH_NOALLOC_MAX_POINTS (16384LL * 16384LL)
int ttsh_diagnostics_noalloc(int Nx, int Ny, double dx, ttsh_dtype t, const void* vx, const void* vy, const void* omega,
                             double cx, double cy, double* sums, ttsh_diag* host_out, void* cuda_stream);
const char* ttsh_diagnostics_noalloc_error(void);

/* Order parameter of the dumbbell geometry:
 *   Psi_2 = | w(x*_left) + w(x*_right) | / ( |w|(x*_left) + |w|(x*_right) ),   x*_side = argmax_side |w|,
 * "left"/"right" = the grid points within `radius` (the paper: D/2) of the centre of either cavity (physical units;
 * (i dx - cx)^2 + (j dx - cy)^2 <= radius^2, inclusive, plain non-periodic distance).  Ties in |w| go to the lowest linear
 * index j Nx + i.  psi2 = 0 when the denominator vanishes or a region holds no grid point (index -1).  1 = ferromagnetic
 * (same-sign vortices), 0 = antiferromagnetic.  host_out: HOST.  Synchronises the stream. */
typedef struct {
  double psi2;
  double omega_left, omega_right;        /* w at the two maximisers */
  long long index_left, index_right;     /* their linear indices j Nx + i */
} ttsh_psi2;
int ttsh_dumbbell_order(ttsh_handle* h, double cx_left, double cy_left, double cx_right, double cy_right, double radius,
                        ttsh_psi2* host_out);

/* Streaming temporal power spectral density of the vorticity field, Eq. (5):
 *   S(Omega) = (1/P) sum_x | sum_t w(x, t) exp(-i Omega t) |^2,   P = Nx Ny,
 * for a caller-chosen set of angular frequencies: one complex accumulator per grid point and frequency, updated by
 * ttsh_psd_accumulate with the handle's current field w(., t) (t = the handle's time), so no time series is ever stored.
 * omegas: HOST double[nfreq], 1 <= nfreq <= 1024.  workspace: DEVICE, >= ttsh_psd_workspace_bytes (about
 * nfreq x 2 fields), 256-byte aligned, owned by the caller, zeroed by create / reset (stream-ordered).  Accumulators have
 * the handle's scalar type; the sum over x is taken in double.  The accumulator borrows the handle: destroy it first. */
typedef struct ttsh_psd ttsh_psd;
size_t ttsh_psd_workspace_bytes(int Nx, int Ny, ttsh_dtype t, int nfreq);       /* 0 if unsupported */
int ttsh_psd_create(ttsh_psd** out, ttsh_handle* h, const double* omegas, int nfreq, void* workspace, size_t workspace_bytes);
int ttsh_psd_accumulate(ttsh_psd* s);                                           /* asynchronous */
int ttsh_psd_result(ttsh_psd* s, double* S_host, long long* nsamples_host);     /* S_host: HOST double[nfreq]; nsamples may be NULL; synchronises */
int ttsh_psd_reset(ttsh_psd* s);
int ttsh_psd_destroy(ttsh_psd* s);

/* Tangent-linear evolution and growth rates (Lyapunov exponents): nvec independent perturbations
 * (dw^, dv^(0)) of the state are carried along the trajectory by the Jacobian of Algorithm 1 at the current state (lines 1-2
 * differentiated, everything else is linear), and re-orthonormalised on request by a QR decomposition (CholeskyQR2 on the
 * device: Gram matrix, Cholesky factor, triangular solve, twice; modified Gram-Schmidt when the vectors are
 * numerically dependent) whose diagonal gives the growth: lambda_i = sum log R_ii / elapsed time.  The inner product is the Euclidean
 * one of the real vectors [dw(x) for all x ; dv^_x(0) ; dv^_y(0)] (unitary DFT normalisation of the mean flow).
 * workspace: DEVICE, >= ttsh_tangent_workspace_bytes, 256-byte aligned, owned by the caller.  1 <= nvec <= 64.  Requires
 * TTSH_ADVECTION_CONSERVATIVE.  The tangent object borrows the handle: destroy it first. */
typedef struct ttsh_tangent ttsh_tangent;
size_t ttsh_tangent_workspace_bytes(int Nx, int Ny, ttsh_dtype t, int nvec);     /* 0 if unsupported */
int ttsh_tangent_create(ttsh_tangent** out, ttsh_handle* h, int nvec, void* workspace, size_t workspace_bytes);
/* Sets perturbation i from a real velocity perturbation (DEVICE scalar[Ny*Nx] each) through the same (linear) projection
 * as ttsh_set_velocity. */
int ttsh_tangent_set(ttsh_tangent* s, int i, const void* dvx, const void* dvy);
/* n times: every perturbation through the Jacobian at the handle's current state, then one step of the handle itself
 * (so the handle advances by n steps).  Asynchronous.  TTSH_ERR_NOT_INITIALIZED unless the handle and all vectors are set. */
int ttsh_tangent_step(ttsh_tangent* s, int n);
/* QR of the current vectors: they are replaced by the orthonormal Q (R_ii > 0), log_r_host[i] = log R_ii (HOST double[nvec]).
 * Synchronises. */
int ttsh_tangent_orthonormalize(ttsh_tangent* s, double* log_r_host);
/* dv = (dvx, dvy) and dw of perturbation i into DEVICE scalar[Ny*Nx] buffers; any pointer may be NULL. */
int ttsh_tangent_get_fields(ttsh_tangent* s, int i, void* dvx, void* dvy, void* domega);
int ttsh_tangent_destroy(ttsh_tangent* s);

/* Ensembles: the paper's workload is sweeps of independent runs on one grid — disk radius R (Fig. 2), the
 * hysteresis branches, dumbbell separations — and on grids up to about 1024^2 one system
 * cannot fill a B200.  An ensemble advances `count` independent handles with ONE launch of each hot kernel per Euler step
 * (4 launches for all members together), every member computing exactly what ttsh_step computes for it: results are
 * bit-identical to stepping the members one by one.  On grids with 128 <= Ny <= 1024, where ttsh_step takes 2 launches
 * (TTSH_STAGE_COL_STEP), an ensemble does the same as long as count x (number of column tiles) <= 8 x (number of SMs); a larger
 * one is bound by throughput, keeps the 4 launches, and then agrees with ttsh_step to round-off instead of bit for bit.
 * Requirements (else TTSH_ERR_INVALID_ARG): count >= 1; all members have the same Nx, Ny, dtype, dx, dt, parameters and
 * stream, use TTSH_ADVECTION_CONSERVATIVE with the 1/2 rule on a grid the fused row kernel supports (Nx <= 8192 in fp64, Nx <= 16384 in fp32), and their workspaces lie at a uniform byte stride: workspace_b = workspace_0 + b * stride, stride >=
 * ttsh_workspace_bytes (carve them from one allocation).  Masks, states and step counters are per member; all other calls
 * (ttsh_set_velocity, ttsh_set_mask, ttsh_get_fields, ttsh_diagnostics, ...) keep working on the member handles.  The
 * ensemble borrows the members: destroy it before them. */
typedef struct ttsh_ensemble ttsh_ensemble;
int ttsh_ensemble_create(ttsh_ensemble** out, ttsh_handle* const* members, int count);
/* n >= 0 applications of Algorithm 1 to every member; asynchronous; every member's t and step counter advance.
 * TTSH_ERR_NOT_INITIALIZED if a member has no state yet. */
int ttsh_ensemble_step(ttsh_ensemble* e, int n);
long long ttsh_ensemble_launch_count(const ttsh_ensemble* e);
int ttsh_ensemble_destroy(ttsh_ensemble* e);

/* Number of kernel launches the library has enqueued for this handle so far (bench bookkeeping). */
long long ttsh_launch_count(const ttsh_handle* h);

/* Debug/bench entry points for the individual kernels of the hot path (used by the per-kernel parity
 * tests and the roofline measurement).  stage: one of TTSH_STAGE_*; runs that stage of a step once on the
 * current state, leaving its outputs in the workspace.  Returns TTSH_ERR_INVALID_ARG for an unknown stage. */
typedef enum {
  TTSH_STAGE_INV_COL = 0,   /* w^ -> y-transformed intermediates (a1+a2/a6 column pass)  */
  TTSH_STAGE_INV_ROW = 1,   /* intermediates -> omega, grad omega, v  (a2/a6 row pass)   */
  TTSH_STAGE_REAL = 2,      /* rhs1, rhs2 (a3)                                           */
  TTSH_STAGE_FWD_ROW = 3,   /* a4 row pass                                               */
  TTSH_STAGE_FWD_COL = 4,   /* a4 column pass                                            */
  TTSH_STAGE_SPECTRAL = 5,  /* a5                                                        */
  TTSH_STAGE_REAL_FWD_ROW = 6, /* a3 fused into the a4 row pass; emits A~ = i kx Gy~ + S'~ and B~ = Gx~ (conservative form)   */
  TTSH_STAGE_FWD_COL_P2 = 7,  /* a4 column pass of those two intermediates                                                    */
  TTSH_STAGE_SPECTRAL_P2 = 8, /* a5 from the two spectra: rhs^ = A^ - i ky B^                                                   */
  TTSH_STAGE_ROW_STEP = 9,    /* stages 1 + 6 in one kernel: w, v never leave the SM (1/2 rule; Nx = 8192, and 16384 in fp32: one real
                                 row per transform).  ttsh_step runs 0, 9, 7, 8 where supported, else 0, 1, 6, 7, 8 */
  TTSH_STAGE_COL_STEP = 10    /* stages 7 + 8 + stage 0 of the NEXT step in one kernel (Ny <= 1024, 1/2 rule): there ttsh_step runs
                                 9, 10 per Euler step, preceded by stage 0 once whenever the intermediates of the current state are
                                 not at hand (first step, or after any call that is not ttsh_step) */
} ttsh_stage;
int ttsh_run_stage(ttsh_handle* h, int stage);
/* Copies a workspace array out for inspection: which = 0..4 real scratch (omega|rhs2, g_x|rhs1_x, g_y|rhs1_y, v_x, v_y;
 * in the conservative form slots 1, 2 hold rhs1_x + lambda0 v_y w and rhs1_y - lambda0 v_x w and slot 0 holds
 * -gamma_w K w after TTSH_STAGE_REAL), 5 = K.  dst: DEVICE scalar[Ny*Nx]. */
int ttsh_debug_get_real(ttsh_handle* h, int which, void* dst);

int ttsh_destroy(ttsh_handle* h);

/* Measurement aid, not part of the method (the fp64 / fp32 ALU roof is not in MEASURED_PEAKS.json).  Enqueues ONE
 * kernel of `blocks` x 256 threads in which every thread runs 8 independent chains x <- x a + b for 16 x rounds fused multiply-adds
 * each, in registers: nothing but the FMA pipe limits it.  sink: DEVICE scalar[blocks * 256] out (thread i of block k writes the
 * sum of its chains, started at (i + 32 c) / 1024, c < 8, to sink[256 k + i]: with a = 1, b = 0 that is (8 i + 896) / 1024).
 * *flops_out (HOST, may be NULL) = 2 x 8 x 16 x rounds x 256 x blocks, the flops of the launch; the caller times it with events.
 * bench.py divides the two and reports the result as the peak of the ALU roofline. */
int ttsh_microbench_fma(ttsh_dtype t, int blocks, int rounds, double a, double b, void* sink, void* cuda_stream, double* flops_out);

/* "ttsh sm_100a sources=<first 16 hex digits of the SHA-256 of csrc/*.cu, *.cuh, *.h, include/ttsh.h, Makefile, concatenated in
 * sorted order> cuda=<nvcc version> built <date>": which sources this binary was compiled from (tests compare it with the tree). */
const char* ttsh_build_info(void);

const char* ttsh_strerror(int code);
const char* ttsh_last_error(const ttsh_handle* h);   /* "" if none */

#ifdef __cplusplus
}
#endif
#endif /* TTSH_H_ */
