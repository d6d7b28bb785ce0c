/* ttsh_oracle_c.c — "oracle-fft": the CPU oracle of oracle/ttsh_oracle.py restated in plain C with a textbook radix-2 FFT.
 *
 * THIS IS TEST INFRASTRUCTURE (and the honest CPU timing baseline of bench.py, the counterpart of the CPU curve of
 * Fig. 9).  It exists because the definition-oracle (explicit DFT-matrix products, O(N^3) per 2-D
 * transform) cannot follow 100 steps at 4096 x 4096 ("bootstrapped 100-step reference").  It is written
 * from the paper only and shares no code with the CUDA path:
 *
 *   Algorithm 1 (integration scheme)      PAPER.md:288-317, prose :319-331, Eq. (C1) :329
 *   Algorithm 2 (mask processing)
 *   unitary DFT
 *   vortex order parameter, Eq. (11)
 *
 * Same rules as the numpy oracle: fp64, FULL complex Ny x Nx spectra, no half-spectrum storage, no pruning, no fusion,
 * Algorithm 1 line by line in the paper's order; nabla -> +i k (reading R3), exact integer cutoff predicate (R4),
 * 1/sqrt(Nx Ny) normalisation (R10).  The only "fast" ingredient is the 1-D transform: an iterative radix-2
 * decimation-in-time FFT (bit reversal + log2 N butterfly passes, twiddles from a long-double table) applied to every row
 * and then every column, OpenMP over lines.  -ffp-contract=off: plain IEEE operations.
 *
 * Pins (tests/test_oracle_c.py, `-m "not gpu"`): locked to the definition-oracle (whole trajectories, K, diagnostics,
 * <= 1e-13) on square and non-square grids, plus the closed-form single-mode growth and the uniform fixed point run
 * through this code alone; line 12 (Hermitian average) on a caller-supplied non-Hermitian spectrum and the
 * non-finite count on one bad value per field, through the test-only ttsho_debug_* entries at the end of this file.  Whole chaotic trajectories of the paper: parity unpinned (as for the numpy oracle).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

typedef struct {
  int Nx, Ny;
  double dx, dt;
  double lambda0, alpha, beta, Gamma0, Gamma2, gamma_v, gamma_w;
  int num, den;
  double *kx, *ky;          /* signed wavenumbers (Table I) */
  cplx *twx, *twy;          /* W_N^k = exp(-2 pi i k / N), k < N/2 */
  double *K;                /* processed mask, Algorithm 2 */
  double *vx, *vy;          /* state: v(t) */
  cplx *w_hat;              /* state: w^(t) */
  cplx *s0, *s1, *s2, *s3;  /* scratch spectra */
  double t;
  long long nstep;
} ttsho;

/* ---- 1-D radix-2 FFT, in place.  sign = -1: forward e^{-i...}, +1: inverse.  No normalisation. ---- */
static void fft1(cplx* a, int N, const cplx* tw, int sign) {
  for (int i = 1, j = 0; i < N; ++i) {            /* bit-reversal permutation */
    int bit = N >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) { cplx t = a[i]; a[i] = a[j]; a[j] = t; }
  }
  for (int len = 2; len <= N; len <<= 1) {        /* butterflies: X[k] = E[k] + W_len^k O[k], X[k + len/2] = E[k] - W_len^k O[k] */
    const int half = len >> 1, stride = N / len;
    for (int i = 0; i < N; i += len)
      for (int k = 0; k < half; ++k) {
        cplx w = tw[k * stride];
        if (sign > 0) w = conj(w);
        const cplx u = a[i + k], v = a[i + k + half] * w;
        a[i + k] = u + v;
        a[i + k + half] = u - v;
      }
  }
}

static cplx* make_twiddles(int N) {
  cplx* tw = (cplx*)malloc(sizeof(cplx) * (size_t)(N / 2 > 0 ? N / 2 : 1));
  const long double two_pi = 2.0L * acosl(-1.0L);
  for (int k = 0; k < N / 2; ++k) {
    long double a = two_pi * (long double)k / (long double)N;
    long double c = cosl(a), s = -sinl(a);
    if (4 * k == N) c = 0.0L;
    if (k == 0) s = 0.0L;
    tw[k] = (double)c + (double)s * I;
  }
  return tw;
}

/* F[my][mx] = (Nx Ny)^-1/2 sum f[j][i] exp(sign 2 pi i (mx i/Nx + my j/Ny)): every row, then every column (R10) */
static void fft2(const ttsho* o, cplx* f, int sign) {
  const int Nx = o->Nx, Ny = o->Ny;
  const double sx = 1.0 / sqrt((double)Nx), sy = 1.0 / sqrt((double)Ny);
#pragma omp parallel for schedule(static)
  for (int j = 0; j < Ny; ++j) {
    cplx* row = f + (size_t)j * Nx;
    fft1(row, Nx, o->twx, sign);
    for (int i = 0; i < Nx; ++i) row[i] *= sx;
  }
  enum { CB = 32 };                               /* columns gathered CB at a time (cache lines), one FFT each */
#pragma omp parallel
  {
    cplx* buf = (cplx*)malloc(sizeof(cplx) * (size_t)Ny * CB);
#pragma omp for schedule(static)
    for (int i0 = 0; i0 < Nx; i0 += CB) {
      const int nb = Nx - i0 < CB ? Nx - i0 : CB;
      for (int j = 0; j < Ny; ++j)
        for (int c = 0; c < nb; ++c) buf[(size_t)c * Ny + j] = f[(size_t)j * Nx + i0 + c];
      for (int c = 0; c < nb; ++c) fft1(buf + (size_t)c * Ny, Ny, o->twy, sign);
      for (int j = 0; j < Ny; ++j)
        for (int c = 0; c < nb; ++c) f[(size_t)j * Nx + i0 + c] = buf[(size_t)c * Ny + j] * sy;
    }
    free(buf);
  }
}

static int signed_index(int m, int N) { return m <= N / 2 ? m : m - N; }   /* Nyquist taken as +N/2 (R8) */

/* strict cutoff k^2 > ((num/den) pi/dx)^2 in integers (R4) */
static int is_cut(const ttsho* o, int my, int mx, int num, int den) {
  const long long a = (long long)signed_index(mx, o->Nx) * o->Ny, b = (long long)signed_index(my, o->Ny) * o->Nx;
  const long long c = (long long)o->Nx * o->Ny;
  return (__int128)4 * den * den * ((__int128)a * a + (__int128)b * b) > (__int128)num * num * c * c;
}

/* ---- Algorithm 2: K = ( iDFT[ lowpass_{1/4}( DFT[K_naive] ) ] )^2 ---- */
static void process_mask(ttsho* o, const unsigned char* mask) {
  const int Nx = o->Nx, Ny = o->Ny;
  const size_t P = (size_t)Nx * Ny;
  cplx* Kh = o->s0;
  for (size_t p = 0; p < P; ++p) Kh[p] = mask[p] ? 1.0 : 0.0;
  fft2(o, Kh, -1);                                              /* line 1 */
#pragma omp parallel for schedule(static)
  for (int my = 0; my < Ny; ++my)
    for (int mx = 0; mx < Nx; ++mx)
      if (is_cut(o, my, mx, 1, 4)) Kh[(size_t)my * Nx + mx] = 0.0;   /* lines 2-8 */
  fft2(o, Kh, +1);
  for (size_t p = 0; p < P; ++p) { const double s = creal(Kh[p]); o->K[p] = s * s; }   /* line 9 */
}

/* ---- lines 5-16 of Algorithm 1 (reading R7).  In: w_naive (overwritten by w^_new), v0_new[2].
 *      Out: w^_new in wn, v^_x in vxh, v^_y in vyh. ---- */
static void post(const ttsho* o, cplx* wn, const double v0_new[2], cplx* vxh, cplx* vyh, cplx* tmp) {
  const int Nx = o->Nx, Ny = o->Ny;
  memcpy(tmp, wn, sizeof(cplx) * (size_t)Nx * Ny);
#pragma omp parallel for schedule(static)
  for (int my = 0; my < Ny; ++my)
    for (int mx = 0; mx < Nx; ++mx) {
      const size_t p = (size_t)my * Nx + mx;
      const size_t pm = (size_t)((Ny - my) % Ny) * Nx + (size_t)((Nx - mx) % Nx);          /* index of -k */
      cplx w = 0.5 * (tmp[p] + conj(tmp[pm]));                                             /* line 12 */
      const int zero = (mx == 0 && my == 0);
      if (zero || is_cut(o, my, mx, o->num, o->den)) w = 0.0;                              /* lines 7, 10 */
      const double kx = o->kx[mx], ky = o->ky[my];
      const double k2 = zero ? 1.0 : kx * kx + ky * ky;
      const cplx psi = w / k2;                                                             /* line 13 */
      wn[p] = w;
      vxh[p] = I * ky * psi;                                                               /* line 14 */
      vyh[p] = -I * kx * psi;
    }
  vxh[0] = v0_new[0];                                                                      /* line 8 */
  vyh[0] = v0_new[1];
}

static void velocity_from_hat(ttsho* o, cplx* vxh, cplx* vyh) {
  const size_t P = (size_t)o->Nx * o->Ny;
  fft2(o, vxh, +1);
  fft2(o, vyh, +1);
  for (size_t p = 0; p < P; ++p) { o->vx[p] = creal(vxh[p]); o->vy[p] = creal(vyh[p]); }
}

/* ---- exported C ABI (HOST pointers only) ---- */
ttsho* ttsho_create(int Nx, int Ny, double dx, double dt, const double* params7, int num, int den, const unsigned char* mask) {
  ttsho* o = (ttsho*)calloc(1, sizeof(ttsho));
  const size_t P = (size_t)Nx * Ny;
  o->Nx = Nx; o->Ny = Ny; o->dx = dx; o->dt = dt;
  o->lambda0 = params7[0]; o->alpha = params7[1]; o->beta = params7[2]; o->Gamma0 = params7[3]; o->Gamma2 = params7[4];
  o->gamma_v = params7[5]; o->gamma_w = params7[6];
  o->num = num; o->den = den;
  o->kx = (double*)malloc(sizeof(double) * Nx);
  o->ky = (double*)malloc(sizeof(double) * Ny);
  const double two_pi = 2.0 * acos(-1.0);
  for (int m = 0; m < Nx; ++m) o->kx[m] = (two_pi / (Nx * dx)) * (double)signed_index(m, Nx);
  for (int m = 0; m < Ny; ++m) o->ky[m] = (two_pi / (Ny * dx)) * (double)signed_index(m, Ny);
  o->twx = make_twiddles(Nx);
  o->twy = make_twiddles(Ny);
  o->K = (double*)calloc(P, sizeof(double));
  o->vx = (double*)calloc(P, sizeof(double));
  o->vy = (double*)calloc(P, sizeof(double));
  o->w_hat = (cplx*)calloc(P, sizeof(cplx));
  o->s0 = (cplx*)malloc(sizeof(cplx) * P); o->s1 = (cplx*)malloc(sizeof(cplx) * P);
  o->s2 = (cplx*)malloc(sizeof(cplx) * P); o->s3 = (cplx*)malloc(sizeof(cplx) * P);
  if (mask) process_mask(o, mask);
  return o;
}

void ttsho_destroy(ttsho* o) {
  if (!o) return;
  free(o->kx); free(o->ky); free(o->twx); free(o->twy); free(o->K); free(o->vx); free(o->vy); free(o->w_hat);
  free(o->s0); free(o->s1); free(o->s2); free(o->s3);
  free(o);
}

void ttsho_get_K(const ttsho* o, double* K) { memcpy(K, o->K, sizeof(double) * (size_t)o->Nx * o->Ny); }
void ttsho_set_K(ttsho* o, const double* K) { memcpy(o->K, K, sizeof(double) * (size_t)o->Nx * o->Ny); }

/* ttsh_set_velocity: w^ = i k_x v^_y - i k_y v^_x, mean flow kept, then lines 5-16 */
void ttsho_set_velocity(ttsho* o, const double* vx0, const double* vy0) {
  const int Nx = o->Nx, Ny = o->Ny;
  const size_t P = (size_t)Nx * Ny;
  cplx *vxh = o->s0, *vyh = o->s1;
  for (size_t p = 0; p < P; ++p) { vxh[p] = vx0[p]; vyh[p] = vy0[p]; }
  fft2(o, vxh, -1);
  fft2(o, vyh, -1);
  const double v0[2] = {creal(vxh[0]), creal(vyh[0])};
#pragma omp parallel for schedule(static)
  for (int my = 0; my < Ny; ++my)
    for (int mx = 0; mx < Nx; ++mx) {
      const size_t p = (size_t)my * Nx + mx;
      o->w_hat[p] = I * o->kx[mx] * vyh[p] - I * o->ky[my] * vxh[p];
    }
  post(o, o->w_hat, v0, vxh, vyh, o->s2);
  velocity_from_hat(o, vxh, vyh);
  o->t = 0.0;
  o->nstep = 0;
}

/* one application of Algorithm 1 */
static void step_once(ttsho* o) {
  const int Nx = o->Nx, Ny = o->Ny;
  const size_t P = (size_t)Nx * Ny;
  const double dt = o->dt;
  cplx *a = o->s0, *b = o->s1, *c = o->s2, *d = o->s3;
  /* line 2 inputs: w = iDFT[w^], grad w = iDFT[i k w^] */
#pragma omp parallel for schedule(static)
  for (int my = 0; my < Ny; ++my)
    for (int mx = 0; mx < Nx; ++mx) {
      const size_t p = (size_t)my * Nx + mx;
      a[p] = o->w_hat[p];
      b[p] = I * o->kx[mx] * o->w_hat[p];
      c[p] = I * o->ky[my] * o->w_hat[p];
    }
  fft2(o, a, +1); fft2(o, b, +1); fft2(o, c, +1);
  /* lines 1-2: rhs1 = -beta |v|^2 v - gamma_v K v ;  rhs2 = -lambda0 v . grad w - gamma_w K w */
  long double sx = 0.0L, sy = 0.0L;               /* sum_x (v + rhs1 dt) for line 8 */
  for (size_t p = 0; p < P; ++p) {
    const double vx = o->vx[p], vy = o->vy[p], K = o->K[p];
    const double w = creal(a[p]), gx = creal(b[p]), gy = creal(c[p]);
    const double s2 = vx * vx + vy * vy;
    const double r1x = -o->beta * s2 * vx - o->gamma_v * K * vx;
    const double r1y = -o->beta * s2 * vy - o->gamma_v * K * vy;
    const double r2 = -o->lambda0 * (vx * gx + vy * gy) - o->gamma_w * K * w;
    sx += (long double)(vx + dt * r1x);
    sy += (long double)(vy + dt * r1y);
    a[p] = r1x; b[p] = r1y; c[p] = r2;
  }
  fft2(o, a, -1); fft2(o, b, -1); fft2(o, c, -1);
  /* lines 3-4: rhs^ = i k_x rhs1_y^ - i k_y rhs1_x^ + rhs2^ ;  w^_naive = exp(sigma dt) (w^ + dt rhs^) */
#pragma omp parallel for schedule(static)
  for (int my = 0; my < Ny; ++my)
    for (int mx = 0; mx < Nx; ++mx) {
      const size_t p = (size_t)my * Nx + mx;
      const double kx = o->kx[mx], ky = o->ky[my];
      const double k2 = kx * kx + ky * ky;
      const double sigma = -o->alpha - o->Gamma0 * k2 - o->Gamma2 * k2 * k2;
      const cplx rhs = I * kx * b[p] - I * ky * a[p] + c[p];
      d[p] = exp(sigma * dt) * (o->w_hat[p] + dt * rhs);
    }
  /* line 8 / Eq. (C1): v^_new(0) = exp(sigma(0) dt) sum_x (v + rhs1 dt) / sqrt(N^2) */
  const double e0 = exp(-o->alpha * dt), rootP = sqrt((double)P);
  const double v0_new[2] = {e0 * (double)sx / rootP, e0 * (double)sy / rootP};
  memcpy(o->w_hat, d, sizeof(cplx) * P);
  post(o, o->w_hat, v0_new, a, b, c);
  velocity_from_hat(o, a, b);
  o->t += dt;
  o->nstep += 1;
}

void ttsho_step(ttsho* o, int n) { for (int i = 0; i < n; ++i) step_once(o); }

/* v (state), w = iDFT[w^], psi = iDFT[w^/k^2] with psi^(0) = 0; any pointer may be NULL */
void ttsho_get_fields(ttsho* o, double* vx, double* vy, double* w, double* psi) {
  const int Nx = o->Nx, Ny = o->Ny;
  const size_t P = (size_t)Nx * Ny;
  if (vx) memcpy(vx, o->vx, sizeof(double) * P);
  if (vy) memcpy(vy, o->vy, sizeof(double) * P);
  if (w) {
    memcpy(o->s0, o->w_hat, sizeof(cplx) * P);
    fft2(o, o->s0, +1);
    for (size_t p = 0; p < P; ++p) w[p] = creal(o->s0[p]);
  }
  if (psi) {
    for (int my = 0; my < Ny; ++my)
      for (int mx = 0; mx < Nx; ++mx) {
        const size_t p = (size_t)my * Nx + mx;
        const double k2 = o->kx[mx] * o->kx[mx] + o->ky[my] * o->ky[my];
        o->s0[p] = (mx == 0 && my == 0) ? 0.0 : o->w_hat[p] / k2;
      }
    fft2(o, o->s0, +1);
    for (size_t p = 0; p < P; ++p) psi[p] = creal(o->s0[p]);
  }
}

/* reading R13.  out[10]: kinetic_energy, enstrophy, vortex_order, polar_order, sum_speed, sum_abs_vtheta, mean_vx, mean_vy,
 * max_speed, nonfinite */
void ttsho_diagnostics(ttsho* o, double cx, double cy, double* out) {
  const int Nx = o->Nx, Ny = o->Ny;
  const size_t P = (size_t)Nx * Ny;
  memcpy(o->s0, o->w_hat, sizeof(cplx) * P);
  fft2(o, o->s0, +1);
  long double s_speed = 0, s_vth = 0, s_vx = 0, s_vy = 0, s_v2 = 0, s_w2 = 0;
  double vmax = 0.0;
  long long bad = 0;
  for (int j = 0; j < Ny; ++j)
    for (int i = 0; i < Nx; ++i) {
      const size_t p = (size_t)j * Nx + i;
      const double vx = o->vx[p], vy = o->vy[p], w = creal(o->s0[p]);
      const double x = i * o->dx - cx, y = j * o->dx - cy;
      const double r = sqrt(x * x + y * y);
      const double vth = r == 0.0 ? 0.0 : (-y * vx + x * vy) / r;         /* e_theta . v, Eq. (11) */
      const double sp = sqrt(vx * vx + vy * vy);
      s_speed += sp; s_vth += fabs(vth); s_vx += vx; s_vy += vy; s_v2 += vx * vx + vy * vy; s_w2 += w * w;
      if (sp > vmax) vmax = sp;
      bad += !isfinite(vx); bad += !isfinite(vy); bad += !isfinite(w);
    }
  const double two_over_pi = 2.0 / acos(-1.0);
  out[0] = 0.5 * (double)s_v2 / (double)P;
  out[1] = 0.5 * (double)s_w2 / (double)P;
  out[2] = s_speed > 0 ? ((double)s_vth / (double)s_speed - two_over_pi) / (1.0 - two_over_pi) : 0.0;
  out[3] = s_speed > 0 ? hypot((double)s_vx, (double)s_vy) / (double)s_speed : 0.0;
  out[4] = (double)s_speed; out[5] = (double)s_vth;
  out[6] = (double)s_vx / (double)P; out[7] = (double)s_vy / (double)P;
  out[8] = vmax; out[9] = (double)bad;
}

/* ---- test-only entries (tests/test_oracle_c.py); no arithmetic of their own ----
 * ttsho_debug_post: lines 5-16 of Algorithm 1 (`post` above) applied to a spectrum the CALLER supplies, so that
 * the Hermitian average of line 12 can be pinned with an input that is not the spectrum of a real field.
 * w_in, w_out, vxh_out, vyh_out: complex[Ny*Nx], interleaved (re, im); v0_new: the k = 0 velocity of line 8. */
void ttsho_debug_post(ttsho* o, const double* w_in, const double* v0_new, double* w_out, double* vxh_out, double* vyh_out) {
  const size_t P = (size_t)o->Nx * o->Ny;
  memcpy(o->s3, w_in, sizeof(cplx) * P);
  post(o, o->s3, v0_new, o->s0, o->s1, o->s2);
  memcpy(w_out, o->s3, sizeof(cplx) * P);
  memcpy(vxh_out, o->s0, sizeof(cplx) * P);
  memcpy(vyh_out, o->s1, sizeof(cplx) * P);
}

/* ttsho_debug_set_state: overwrites the raw state arrays (any pointer may be NULL), bypassing set_velocity's projection: the only
 * way to hand ttsho_diagnostics a non-finite value in a chosen field.  w_hat: complex[Ny*Nx] interleaved; vx, vy: double[Ny*Nx]. */
void ttsho_debug_set_state(ttsho* o, const double* w_hat, const double* vx, const double* vy) {
  const size_t P = (size_t)o->Nx * o->Ny;
  if (w_hat) memcpy(o->w_hat, w_hat, sizeof(cplx) * P);
  if (vx) memcpy(o->vx, vx, sizeof(double) * P);
  if (vy) memcpy(o->vy, vy, sizeof(double) * P);
}

double ttsho_time(const ttsho* o) { return o->t; }
long long ttsho_nstep(const ttsho* o) { return o->nstep; }
