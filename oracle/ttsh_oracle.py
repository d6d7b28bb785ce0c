"""Plain, slow, obviously-correct CPU oracle for one pseudospectral step of the 2-D
Toner-Tu-Swift-Hohenberg (TTSH) equation with the damping-mask boundary scheme.

THIS IS TEST INFRASTRUCTURE.  It is the reference the CUDA path is compared against.
It is written from the paper only (PAPER.md = arXiv:2304.03306, cited as PAPER.md:<line>):

* Algorithm 1 (integration scheme)      PAPER.md:288-317, prose :319-331, Eq. (C1) :329
* Algorithm 2 (mask processing scheme)  PAPER.md:337-361, prose :363-371
* unitary DFT / iDFT definition
* vortex order parameter, Eq. (11)
* stream function  lap(psi) = -omega, v = (d_y psi, -d_x psi)

Design rules (why it looks the way it does):
* fp64 everywhere; FULL complex Ny x Nx spectra, no half-spectrum storage, no pruning,
  no fusion, no re-ordering beyond what Algorithm 1 states.
* every transform is the DEFINITION of the DFT: a product with the explicit DFT matrix
  (a naive O(N^2) sum per line; numpy's matmul is the only library primitive used).
  ``transform="fft"`` swaps that single primitive for ``numpy.fft`` (pocketfft); that
  variant is locked to the matrix one by tests and is used only where the O(N^3) cost
  is prohibitive (4096^2 trajectories) and as the honest CPU timing baseline.
* derivative symbol: nabla -> +i k (readings R3 in DESIGN.md; Algorithm 1's own lines
  use iDFT[i k w], i k x rhs1, v_x = i k_y psi, which is consistent with the forward
  DFT sign e^{-ik.x} of PAPER.md:319).
* general TTSH form of BASELINE.json: sigma(k) = -alpha - Gamma0 k^2 - Gamma2 k^4; the
  paper's  a - (1-k^2)^2 is alpha=1-a, Gamma0=-2, Gamma2=1.

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``): brute-force 2-D DFT on 8x8/16x16/8x16,
Parseval, analytic derivatives, closed-form single-mode growth exp(sigma n dt), the
discrete uniform fixed point, the K=1 damping closed form, exact incompressibility,
Hermitian-symmetry repair, Algorithm-2 invariants, diagnostics of analytic fields.
Whole chaotic trajectories / regime boundaries of the paper: PARITY UNPINNED (they need
the paper's 8192^2 long runs).

Array conventions: real fields are ``f[j, i]`` (shape ``[Ny, Nx]``), point (i, j) sits at
x = (i*dx, j*dx); spectra are ``F[my, mx]`` in DFT index order m = 0..N-1.
"""
from __future__ import annotations

from dataclasses import dataclass
from functools import lru_cache

import numpy as np

__all__ = [
    "TTSHParams", "TTSHOracle", "PAPER_PRESET", "BASELINE_PRESET", "dft1", "dft2", "idft2",
    "dft2_brute", "signed_index", "wavenumbers", "cut_mask", "process_mask", "linear_symbol",
]


# --------------------------------------------------------------------------------------
# parameters
# --------------------------------------------------------------------------------------
@dataclass(frozen=True)
class TTSHParams:
    """General TTSH form:  d_t v + lambda0 v.grad v = -grad p - (alpha + beta |v|^2) v
    + Gamma0 lap v - Gamma2 lap^2 v   plus the damping terms of Eq. (4)."""
    lambda0: float
    alpha: float
    beta: float
    Gamma0: float
    Gamma2: float
    gamma_v: float = 40.0      # PAPER.md:61, Table I :269
    gamma_w: float = 4.0       # PAPER.md:61, Table I :270
    dealias_num: int = 1       # cutoff = (num/den) * pi/dx ; the paper's 1/2 rule
    dealias_den: int = 2


# paper: (a, b, lambda, gamma_v, gamma_w) = (0.5, 1.6, 9, 40, 4), and
# a v - (1 + lap)^2 v  =  -(1-a) v - 2 lap v - lap^2 v  =>  alpha = 1-a, Gamma0 = -2, Gamma2 = 1
PAPER_PRESET = TTSHParams(lambda0=9.0, alpha=0.5, beta=1.6, Gamma0=-2.0, Gamma2=1.0)
# BASELINE.json configs: lambda0=3.5, alpha=-0.5, beta=0.5, Gamma0=-1, Gamma2=1 (+ paper's gammas)
BASELINE_PRESET = TTSHParams(lambda0=3.5, alpha=-0.5, beta=0.5, Gamma0=-1.0, Gamma2=1.0)


# --------------------------------------------------------------------------------------
# DFT  (PAPER.md:319:  f^(k) = N^-1 sum_x f(x) e^{-ik.x}  for an N x N lattice, i.e. unitary)
# --------------------------------------------------------------------------------------
@lru_cache(maxsize=16)
def _dft_matrix(N: int, sign: int) -> np.ndarray:
    """W[m, j] = exp(sign * 2 pi i * m j / N) / sqrt(N).

    The phase is reduced exactly in integers ((m*j) mod N) and evaluated in extended
    precision before rounding to fp64, so every entry is correctly rounded."""
    m = np.arange(N, dtype=np.int64)
    r = (m[:, None] * m[None, :]) % N
    two_pi = 2 * np.arccos(np.longdouble(-1.0))
    ang = two_pi * r.astype(np.longdouble) / np.longdouble(N)
    W = np.empty((N, N), dtype=np.complex128)
    W.real = np.cos(ang).astype(np.float64)
    W.imag = (sign * np.sin(ang)).astype(np.float64)
    W /= np.sqrt(np.float64(N))
    W.setflags(write=False)
    return W


def dft1(line: np.ndarray, sign: int = -1) -> np.ndarray:
    """Naive O(N^2) unitary DFT of one line: out[m] = N^-1/2 sum_j in[j] exp(sign 2 pi i j m / N)."""
    line = np.asarray(line, dtype=np.complex128)
    return _dft_matrix(line.shape[0], sign) @ line


def _transform2(f: np.ndarray, sign: int, transform: str) -> np.ndarray:
    f = np.asarray(f, dtype=np.complex128)
    Ny, Nx = f.shape
    if transform == "matmul":
        # dft1 over every row (x), then over every column (y)
        return _dft_matrix(Ny, sign) @ (f @ _dft_matrix(Nx, sign).T)
    if transform == "fft":
        return np.fft.fft2(f, norm="ortho") if sign < 0 else np.fft.ifft2(f, norm="ortho")
    raise ValueError(transform)


def dft2(f, transform: str = "matmul") -> np.ndarray:
    """F[my, mx] = (Nx Ny)^-1/2 sum_{j,i} f[j,i] exp(-2 pi i (mx i/Nx + my j/Ny))   (R10)."""
    return _transform2(f, -1, transform)


def idft2(F, transform: str = "matmul") -> np.ndarray:
    """f[j, i] = (Nx Ny)^-1/2 sum_{my,mx} F[my,mx] exp(+2 pi i (mx i/Nx + my j/Ny))."""
    return _transform2(F, +1, transform)


def dft2_brute(f) -> np.ndarray:
    """The O(P^2) double sum, written out with python loops over output bins.  Tiny grids only."""
    f = np.asarray(f, dtype=np.complex128)
    Ny, Nx = f.shape
    j = np.arange(Ny)[:, None]
    i = np.arange(Nx)[None, :]
    out = np.zeros((Ny, Nx), dtype=np.complex128)
    for my in range(Ny):
        for mx in range(Nx):
            phase = -2.0 * np.pi * (((mx * i) % Nx) / Nx + ((my * j) % Ny) / Ny)
            out[my, mx] = np.sum(f * np.exp(1j * phase)) / np.sqrt(Nx * Ny)
    return out


# --------------------------------------------------------------------------------------
# wavenumbers and the cutoff predicate
# --------------------------------------------------------------------------------------
def signed_index(N: int) -> np.ndarray:
    """DFT index m=0..N-1 -> signed wavenumber index in (-N/2, N/2]  (Nyquist taken as +N/2, R8)."""
    m = np.arange(N, dtype=np.int64)
    return np.where(m <= N // 2, m, m - N)


def wavenumbers(Nx: int, Ny: int, dx: float):
    """k in [-pi/dx, pi/dx]^2 with spacing 2 pi / L  (Table I).  Returns kx[1,Nx], ky[Ny,1]."""
    kx = (2.0 * np.pi / (Nx * dx)) * signed_index(Nx).astype(np.float64)
    ky = (2.0 * np.pi / (Ny * dx)) * signed_index(Ny).astype(np.float64)
    return kx[None, :], ky[:, None]


def cut_mask(Nx: int, Ny: int, num: int, den: int) -> np.ndarray:
    """True where  k^2 > ((num/den) * pi/dx)^2  (strict), evaluated
    exactly in integers (reading R4):  4 den^2 ((mx Ny)^2 + (my Nx)^2) > num^2 (Nx Ny)^2."""
    mx = signed_index(Nx)
    my = signed_index(Ny)
    assert 4 * den * den * 2 * (Nx * Ny // 2) ** 2 < 2 ** 62, "integer overflow in cutoff predicate"
    lhs = 4 * den * den * ((mx * Ny)[None, :] ** 2 + (my * Nx)[:, None] ** 2)
    return lhs > num * num * (Nx * Ny) ** 2


def linear_symbol(k2: np.ndarray, p: TTSHParams) -> np.ndarray:
    """sigma(k) = -alpha - Gamma0 k^2 - Gamma2 k^4   ( = a - (1-k^2)^2 for the paper preset)."""
    return -p.alpha - p.Gamma0 * k2 - p.Gamma2 * k2 * k2


# --------------------------------------------------------------------------------------
# Algorithm 2
# --------------------------------------------------------------------------------------
def process_mask(K_naive: np.ndarray, transform: str = "matmul") -> np.ndarray:
    """K = ( iDFT[ lowpass_{1/4}( DFT[K_naive] ) ] )^2 ; no optional extra filtering."""
    K_naive = np.asarray(K_naive, dtype=np.float64)
    Ny, Nx = K_naive.shape
    Kh = dft2(K_naive, transform)                       # line 1
    Kh = np.where(cut_mask(Nx, Ny, 1, 4), 0.0, Kh)      # lines 2-8, cutoff (1/4) pi/dx
    s = idft2(Kh, transform).real                       # the spectrum is Hermitian; Im is round-off
    return s * s                                        # line 9


# --------------------------------------------------------------------------------------
# the oracle
# --------------------------------------------------------------------------------------
class TTSHOracle:
    """State (v(t), w^(t)) of Algorithm 1 and the operations of the C ABI
    (include/ttsh.h): create / set_velocity / step / get_fields / diagnostics."""

    def __init__(self, Nx: int, Ny: int, dx: float, dt: float, params: TTSHParams,
                 mask=None, mask_kind: str = "binary", transform: str = "matmul"):
        self.Nx, self.Ny, self.dx, self.dt, self.p = int(Nx), int(Ny), float(dx), float(dt), params
        self.transform = transform
        self.kx, self.ky = wavenumbers(Nx, Ny, dx)
        self.k2 = self.kx ** 2 + self.ky ** 2
        self.cut = cut_mask(Nx, Ny, params.dealias_num, params.dealias_den)
        self.is_zero = np.zeros((Ny, Nx), dtype=bool)
        self.is_zero[0, 0] = True
        if mask is None:
            self.K = np.zeros((Ny, Nx))                               # no confinement
        elif mask_kind == "binary":
            self.K = process_mask(np.asarray(mask) != 0, transform)   # Algorithm 2
        elif mask_kind == "processed":
            self.K = np.array(mask, dtype=np.float64)
        else:
            raise ValueError(mask_kind)
        self.v = None          # real, shape [2, Ny, Nx]  (v_x, v_y)
        self.w_hat = None      # complex, shape [Ny, Nx]
        self.t = 0.0
        self.nstep = 0

    # -- transforms ----------------------------------------------------------------
    def _dft(self, f):
        return dft2(f, self.transform)

    def _idft(self, F):
        return idft2(F, self.transform)

    @staticmethod
    def _conj_reflect(F: np.ndarray) -> np.ndarray:
        """G[k] = conj(F[-k])  (indices modulo N)."""
        G = np.conj(F)
        G = np.roll(G[::-1, ::-1], shift=(1, 1), axis=(0, 1))
        return G

    # -- lines 5-16 of Algorithm 1 (garbled block read as R7) --------
    def _post(self, w_naive: np.ndarray, v0_new: np.ndarray):
        """k = 0: w^ = 0, v^(0) = v0_new.  beyond the cutoff: everything 0.  otherwise Hermitian
        average (line 12), psi^ = w^/k^2 (line 13), v^ = (i k_y psi^, -i k_x psi^) (line 14)."""
        w_new = 0.5 * (w_naive + self._conj_reflect(w_naive))           # line 12
        w_new = np.where(self.cut | self.is_zero, 0.0, w_new)           # lines 7, 10
        k2_safe = np.where(self.is_zero, 1.0, self.k2)
        psi_hat = w_new / k2_safe                                       # line 13
        vx_hat = 1j * self.ky * psi_hat                                 # line 14
        vy_hat = -1j * self.kx * psi_hat
        vx_hat[0, 0] = v0_new[0]                                        # line 8
        vy_hat[0, 0] = v0_new[1]
        return w_new, psi_hat, vx_hat, vy_hat

    # -- ttsh_set_velocity -----------------------------------------------------------
    def set_velocity(self, vx0, vy0):
        """Initial condition / restart from a real field v0 (PAPER.md:87 'random initial state').
        w^ = i k_x v^_y - i k_y v^_x, mean flow v^(0) kept, then the post-processing of lines 5-16
        so that the state is band-limited and divergence-free before the first step (:321)."""
        vxh = self._dft(vx0)
        vyh = self._dft(vy0)
        w_hat = 1j * self.kx * vyh - 1j * self.ky * vxh
        v0 = np.array([vxh[0, 0], vyh[0, 0]])
        self.w_hat, _, vxh_new, vyh_new = self._post(w_hat, v0)
        self.v = np.stack([self._idft(vxh_new).real, self._idft(vyh_new).real])
        self.t = 0.0
        self.nstep = 0

    # -- lines 1-2 (real-space right-hand sides) -------------------------------------
    def rhs_real(self):
        """Returns (w, g_x, g_y, rhs1 [2,Ny,Nx], rhs2) of Algorithm 1 lines 1-2."""
        p = self.p
        v = self.v
        w = self._idft(self.w_hat).real
        gx = self._idft(1j * self.kx * self.w_hat).real
        gy = self._idft(1j * self.ky * self.w_hat).real
        speed2 = v[0] ** 2 + v[1] ** 2
        rhs1 = -p.beta * speed2 * v - p.gamma_v * self.K * v                     # line 1
        rhs2 = -p.lambda0 * (v[0] * gx + v[1] * gy) - p.gamma_w * self.K * w     # line 2
        return w, gx, gy, rhs1, rhs2

    # -- one application of Algorithm 1 ----------------------------------------------
    def _step_once(self):
        p, dt = self.p, self.dt
        P = self.Nx * self.Ny
        _, _, _, rhs1, rhs2 = self.rhs_real()
        rhs_hat = (1j * self.kx * self._dft(rhs1[1]) - 1j * self.ky * self._dft(rhs1[0])
                   + self._dft(rhs2))                                              # line 3
        sigma = linear_symbol(self.k2, p)
        w_naive = np.exp(sigma * dt) * (self.w_hat + dt * rhs_hat)                 # line 4
        # line 8 / Eq. (C1): v^_new(0) = exp(sigma(0) dt) * sum_x (v + rhs1 dt) / sqrt(N^2)
        v0_new = np.exp(-p.alpha * dt) * np.sum(self.v + dt * rhs1, axis=(1, 2)) / np.sqrt(P)
        self.w_hat, _, vxh, vyh = self._post(w_naive, v0_new)
        self.v = np.stack([self._idft(vxh).real, self._idft(vyh).real])            # output v(t+dt)
        self.t += dt
        self.nstep += 1

    def step(self, n: int = 1):
        if self.v is None:
            raise RuntimeError("set_velocity first")
        for _ in range(int(n)):
            self._step_once()

    # -- ttsh_get_fields ---------------------------------------------------------------
    def get_fields(self):
        """v (state), w = iDFT[w^], psi = iDFT[w^/k^2] with psi^(0) = 0."""
        w = self._idft(self.w_hat).real
        k2_safe = np.where(self.is_zero, 1.0, self.k2)
        psi = self._idft(np.where(self.is_zero, 0.0, self.w_hat / k2_safe)).real
        return self.v[0].copy(), self.v[1].copy(), w, psi

    # -- ttsh_diagnostics (reading R13) ----------------------------------------------
    def diagnostics(self, cx: float, cy: float) -> dict:
        """E = (1/2P) sum |v|^2, Z = (1/2P) sum w^2, vortex order Psi of Eq. (11) (
        the sums run over the entire grid, :143), polar order |sum v| / sum |v|.  e_theta is the
        azimuthal unit vector about (cx, cy); the point r = 0 contributes to the denominator only."""
        P = self.Nx * self.Ny
        vx, vy = self.v
        w = self._idft(self.w_hat).real
        x = (np.arange(self.Nx) * self.dx - cx)[None, :]
        y = (np.arange(self.Ny) * self.dx - cy)[:, None]
        r = np.sqrt(x * x + y * y)
        r_safe = np.where(r == 0.0, 1.0, r)
        vtheta = np.where(r == 0.0, 0.0, (-y * vx + x * vy) / r_safe)
        speed = np.sqrt(vx * vx + vy * vy)
        ld = np.longdouble
        sum_speed = float(np.sum(speed, dtype=ld))
        sum_abs_vtheta = float(np.sum(np.abs(vtheta), dtype=ld))
        sum_vx = float(np.sum(vx, dtype=ld))
        sum_vy = float(np.sum(vy, dtype=ld))
        sum_v2 = float(np.sum(vx * vx + vy * vy, dtype=ld))
        sum_w2 = float(np.sum(w * w, dtype=ld))
        if sum_speed > 0.0:
            two_over_pi = 2.0 / np.pi
            vortex = (sum_abs_vtheta / sum_speed - two_over_pi) / (1.0 - two_over_pi)   # Eq. (11)
            polar = float(np.hypot(sum_vx, sum_vy)) / sum_speed
        else:
            vortex, polar = 0.0, 0.0
        return dict(t=self.t, step=self.nstep,
                    kinetic_energy=0.5 * sum_v2 / P, enstrophy=0.5 * sum_w2 / P,
                    vortex_order=vortex, polar_order=polar,
                    sum_speed=sum_speed, sum_abs_vtheta=sum_abs_vtheta,
                    mean_vx=sum_vx / P, mean_vy=sum_vy / P,
                    max_speed=float(speed.max()),
                    nonfinite=int(np.count_nonzero(~np.isfinite(vx)) + np.count_nonzero(~np.isfinite(vy))
                                  + np.count_nonzero(~np.isfinite(w))))

    # -- ttsh_dumbbell_order ---------------------------------------------
    def dumbbell_order(self, centre_left, centre_right, radius: float) -> dict:
        """Psi_2 of the current vorticity field; see psi2_of_field."""
        w = self._idft(self.w_hat).real
        return psi2_of_field(w, self.dx, centre_left, centre_right, radius)


def psi2_of_field(w: np.ndarray, dx: float, centre_left, centre_right, radius: float) -> dict:
    """Order parameter of the dumbbell geometry:

        Psi_2 = | w(x*_left) + w(x*_right) | / ( |w|(x*_left) + |w|(x*_right) ),   x*_side = argmax_side |w|,

    "left"/"right" = the grid points within `radius` (the paper: D/2) of the centre of either cavity, i.e.
    (i dx - cx)^2 + (j dx - cy)^2 <= radius^2 (inclusive; plain, non-periodic distance; evaluated in fp64 without
    contraction).  Ties in |w| go to the lowest linear index j Nx + i; Psi_2 = 0 if the denominator is 0 or a region holds
    no grid point (index -1).  Written as the definition: one pass over the grid per side."""
    Ny, Nx = w.shape
    out = {}
    best = []
    for side, (cx, cy) in (("left", centre_left), ("right", centre_right)):
        bi, ba = -1, -1.0
        for j in range(Ny):
            yy = j * dx - cy
            for i in range(Nx):
                xx = i * dx - cx
                if xx * xx + yy * yy <= radius * radius:
                    a = abs(float(w[j, i]))
                    if a > ba:
                        ba, bi = a, j * Nx + i
        val = float(w[bi // Nx, bi % Nx]) if bi >= 0 else 0.0
        out["index_" + side] = bi
        out["omega_" + side] = val
        best.append(val)
    den = abs(best[0]) + abs(best[1])
    ok = den > 0.0 and out["index_left"] >= 0 and out["index_right"] >= 0
    out["psi2"] = abs(best[0] + best[1]) / den if ok else 0.0
    return out


def temporal_psd(series, times, omegas) -> np.ndarray:
    """Temporal power spectral density of the vorticity field, Eq. (5):

        S(Omega) = (1/P) sum_x | sum_t w(x, t) exp(-i Omega t) |^2 ,   P = number of grid points,

    for the samples series[n] = w(., times[n]) and every Omega in omegas.  Written as the definition (one complex
    accumulator per point and frequency); accumulation in fp64, the final sum over x in long double."""
    series = [np.asarray(f, dtype=np.float64) for f in series]
    P = series[0].size
    out = np.zeros(len(omegas))
    for m, Om in enumerate(omegas):
        acc = np.zeros(series[0].shape, dtype=np.complex128)
        for f, t in zip(series, times):
            acc += f * complex(np.cos(Om * t), -np.sin(Om * t))
        out[m] = float(np.sum(acc.real * acc.real + acc.imag * acc.imag, dtype=np.longdouble)) / P
    return out

