"""CPU oracle for the tangent-linear ("Lyapunov") extension of the TTSH step (TEST INFRASTRUCTURE).

PAPER.md:153-159: "we simulated the time evolution of independent perturbations delta-omega_i(x, t) along with omega(x, t)
and measured the exponential growth rates using the QR decomposition" (the standard method of its refs. [36, 37]).

The paper gives no formulas beyond that sentence, so the oracle is the definition written out:

* a perturbation is an element of the tangent space of the state (w^, v^(0)) of Algorithm 1: (dw^, dv^(0)), with the
  dependent real field dv = iDFT[(i k_y dpsi^, -i k_x dpsi^)], dpsi^ = dw^/k^2, dv^(0) at k = 0 (lines 13-14 are linear);
* one tangent step applies the Jacobian of one application of Algorithm 1 at the current base state,
  i.e. every line of `TTSHOracle._step_once` differentiated by hand (lines 1-2 are the only nonlinear ones);
* growth rates: after some steps the vectors are re-orthonormalised by a QR decomposition (numpy.linalg.qr, a library
  primitive) of the matrix whose columns are the real vectors [dw(x) for all x ; dv^_x(0) ; dv^_y(0)] (Euclidean inner product;
  by Parseval the same as the Hermitian inner product of the spectra); lambda_i = sum log|R_ii| / elapsed time.

Pinned in tests/test_oracle_pins.py against central finite differences of the NONLINEAR oracle step, the exact single-mode
growth exp(sigma(k) dt) about the zero state, and the Gram determinant.  Whole Lyapunov spectra of the paper's runs
(Fig. 6c-e) are parity unpinned: they need its long 8192^2 runs.
"""
from __future__ import annotations

import numpy as np

from .ttsh_oracle import TTSHOracle, linear_symbol


class TangentOracle:
    def __init__(self, base: TTSHOracle, nvec: int):
        self.base, self.nvec = base, int(nvec)
        self.dw_hat = [None] * self.nvec          # complex [Ny, Nx]
        self.dv = [None] * self.nvec              # real [2, Ny, Nx]
        self.dv0 = [None] * self.nvec             # real [2]: dv^_x(0), dv^_y(0) (unitary DFT normalisation)

    # -- same projection as ttsh_set_velocity (it is linear) ----------------------------
    def set(self, i: int, dvx0, dvy0):
        b = self.base
        vxh, vyh = b._dft(np.asarray(dvx0, dtype=np.float64)), b._dft(np.asarray(dvy0, dtype=np.float64))
        w_hat = 1j * b.kx * vyh - 1j * b.ky * vxh
        v0 = np.array([vxh[0, 0].real, vyh[0, 0].real])
        self._assign(i, w_hat, v0)

    def _assign(self, i, w_naive, v0):
        b = self.base
        w_new, _, vxh, vyh = b._post(w_naive, v0)
        self.dw_hat[i] = w_new
        self.dv[i] = np.stack([b._idft(vxh).real, b._idft(vyh).real])
        self.dv0[i] = np.array(v0, dtype=np.float64)

    # -- Jacobian of one application of Algorithm 1 at the base state, applied to vector i --
    def _tangent_once(self, i, base_fields):
        b, p, dt = self.base, self.base.p, self.base.dt
        P = b.Nx * b.Ny
        w, gx, gy = base_fields
        v, K = b.v, b.K
        dw_hat, dv = self.dw_hat[i], self.dv[i]
        dw = b._idft(dw_hat).real
        dgx = b._idft(1j * b.kx * dw_hat).real
        dgy = b._idft(1j * b.ky * dw_hat).real
        speed2 = v[0] ** 2 + v[1] ** 2
        vdv = v[0] * dv[0] + v[1] * dv[1]
        drhs1 = -p.beta * (2.0 * vdv * v + speed2 * dv) - p.gamma_v * K * dv                       # d(line 1)
        drhs2 = (-p.lambda0 * (dv[0] * gx + dv[1] * gy + v[0] * dgx + v[1] * dgy)
                 - p.gamma_w * K * dw)                                                               # d(line 2)
        drhs_hat = 1j * b.kx * b._dft(drhs1[1]) - 1j * b.ky * b._dft(drhs1[0]) + b._dft(drhs2)      # line 3 (linear)
        sigma = linear_symbol(b.k2, p)
        dw_naive = np.exp(sigma * dt) * (dw_hat + dt * drhs_hat)                                     # line 4 (linear)
        dv0_new = np.exp(-p.alpha * dt) * np.sum(dv + dt * drhs1, axis=(1, 2)) / np.sqrt(P)          # line 8 (linear)
        self._assign(i, dw_naive, dv0_new)

    def step(self, n: int = 1):
        """n times: every perturbation through the Jacobian at the base state of time t, then the base step."""
        b = self.base
        for _ in range(int(n)):
            w, gx, gy, _, _ = b.rhs_real()
            for i in range(self.nvec):
                self._tangent_once(i, (w, gx, gy))
            b.step(1)

    # -- QR re-orthonormalisation ----------------------------------------------------------
    def as_matrix(self) -> np.ndarray:
        b = self.base
        cols = [np.concatenate([b._idft(self.dw_hat[i]).real.ravel(), self.dv0[i]]) for i in range(self.nvec)]
        return np.stack(cols, axis=1)

    def orthonormalize(self) -> np.ndarray:
        """Returns log|R_ii| (i = 0..nvec-1) and replaces the vectors by the columns of Q (signs chosen so that R_ii > 0)."""
        b = self.base
        Q, R = np.linalg.qr(self.as_matrix())
        sgn = np.where(np.diag(R) < 0, -1.0, 1.0)
        Q = Q * sgn[None, :]
        P = b.Nx * b.Ny
        for i in range(self.nvec):
            dw = Q[:P, i].reshape(b.Ny, b.Nx)
            self._assign(i, b._dft(dw), Q[P:, i])
        return np.log(np.abs(np.diag(R)))

    def get_fields(self, i: int):
        return self.dv[i][0].copy(), self.dv[i][1].copy(), self.base._idft(self.dw_hat[i]).real
