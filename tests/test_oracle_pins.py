"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Each test is chosen so that a plausible mistake in oracle/ttsh_oracle.py (dropped term, wrong
sign or index, transposed operand, wrong normalisation) fails it.  Citations: PAPER.md lines.
"""
import os

import numpy as np
import pytest

from oracle import (BASELINE_PRESET, PAPER_PRESET, TTSHOracle, TTSHParams, cut_mask, dft1, dft2,
                    dft2_brute, idft2, linear_symbol, process_mask, signed_index, wavenumbers)
from paper_2304_03306_b200 import workloads

GOLD = os.path.join(os.path.dirname(__file__), "golden")
LIN = TTSHParams(lambda0=0.0, alpha=-0.5, beta=0.0, Gamma0=-1.0, Gamma2=1.0, gamma_v=0.0, gamma_w=0.0)


def rng(seed):
    return np.random.default_rng(seed)


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300)


# ---------------------------------------------------------------- DFT
@pytest.mark.parametrize("shape", [(8, 8), (16, 16), (8, 16), (16, 8)])
def test_dft2_matches_brute_force_double_sum(shape):
    f = rng(1).standard_normal(shape) + 1j * rng(2).standard_normal(shape)
    assert np.max(np.abs(dft2(f) - dft2_brute(f))) < 1e-14
    assert np.max(np.abs(dft2(f, "fft") - dft2_brute(f))) < 1e-14


def test_dft_roundtrip_parseval_delta_cosine():
    Ny, Nx = 32, 64
    f = rng(3).standard_normal((Ny, Nx))
    F = dft2(f)
    assert np.max(np.abs(idft2(F) - f)) < 1e-13
    assert abs(np.sum(np.abs(F) ** 2) - np.sum(f ** 2)) < 1e-10 * np.sum(f ** 2)      # unitary
    delta = np.zeros((Ny, Nx)); delta[0, 0] = 1.0
    assert np.max(np.abs(dft2(delta) - 1.0 / np.sqrt(Nx * Ny))) < 1e-15                # delta -> constant
    # a single cosine lands in exactly two bins with amplitude A*sqrt(P)/2, and x is the LAST axis
    A, mx, my = 0.7, 5, 3
    i = np.arange(Nx)[None, :]; j = np.arange(Ny)[:, None]
    c = A * np.cos(2 * np.pi * (mx * i / Nx + my * j / Ny))
    C = dft2(c)
    expect = np.zeros_like(C); expect[my, mx] = expect[-my, -mx] = A * np.sqrt(Nx * Ny) / 2
    assert np.max(np.abs(C - expect)) < 1e-12


def test_dft_forward_sign_is_minus():
    # f = exp(+i k x) must land in bin +m of the FORWARD transform (e^{-ikx} kernel)
    N, m = 16, 3
    f = np.exp(2j * np.pi * m * np.arange(N) / N)
    F = dft1(f, -1)
    assert abs(F[m] - np.sqrt(N)) < 1e-13 and np.sum(np.abs(F)) - abs(F[m]) < 1e-12


def test_fft_backend_locked_to_matrix_backend():
    f = rng(4).standard_normal((128, 64))
    assert rel(dft2(f, "fft"), dft2(f)) < 1e-14
    assert rel(idft2(dft2(f), "fft"), f) < 1e-14


# ---------------------------------------------------------------- wavenumbers, nabla -> +ik (R3)
def test_wavenumber_table_and_spectral_derivative():
    Nx, Ny, dx = 32, 16, 0.5
    kx, ky = wavenumbers(Nx, Ny, dx)
    assert kx.shape == (1, Nx) and ky.shape == (Ny, 1)
    assert abs(kx[0, 1] - 2 * np.pi / (Nx * dx)) < 1e-15                # dk = 2 pi / L
    assert abs(kx.max() - np.pi / dx) < 1e-13 and kx.min() > -np.pi / dx  # k in (-pi/dx, pi/dx]
    x = np.arange(Nx)[None, :] * dx; y = np.arange(Ny)[:, None] * dx
    qx, qy, ph = kx[0, 3], ky[2, 0], 0.4
    f = np.sin(qx * x + qy * y + ph)
    dfdx = idft2(1j * kx * dft2(f)).real
    dfdy = idft2(1j * ky * dft2(f)).real
    assert np.max(np.abs(dfdx - qx * np.cos(qx * x + qy * y + ph))) < 1e-12
    assert np.max(np.abs(dfdy - qy * np.cos(qx * x + qy * y + ph))) < 1e-12


def test_cutoff_predicate_is_strict_and_circular():
    Nx = Ny = 64
    cut = cut_mask(Nx, Ny, 1, 2)
    m = signed_index(Nx)
    assert not cut[0, 16] and not cut[16, 0] and not cut[0, -16]        # exactly on the circle: kept
    assert cut[1, 16] and cut[0, 17]                                    # just outside: cut
    assert cut[12, 12] and not cut[11, 11]                              # circular, not per-axis
    assert cut[Ny // 2, 0] and cut[0, Nx // 2]                          # Nyquist always removed (R8)
    frac = 1.0 - cut.mean()
    assert abs(frac - np.pi / 16) < 0.01                                # pi/16 of the modes retained
    # non-square: isotropic in physical k
    cut2 = cut_mask(128, 64, 1, 2)
    assert not cut2[0, 32] and cut2[0, 33] and not cut2[16, 0] and cut2[17, 0]
    assert np.array_equal(cut, cut_mask(Nx, Ny, 2, 4))
    _ = m


def test_advection_term_two_modes_analytic():
    # v from a stream function with one mode, w with another: v.grad(w) analytically vs spectrally
    N, dx = 32, 0.5
    kx, ky = wavenumbers(N, N, dx)
    x = np.arange(N)[None, :] * dx; y = np.arange(N)[:, None] * dx
    a1, a2 = kx[0, 2], ky[1, 0]
    b1, b2 = kx[0, 1], ky[3, 0]
    psi = np.cos(a1 * x + a2 * y)            # v = (d_y psi, -d_x psi)
    vx = -a2 * np.sin(a1 * x + a2 * y); vy = a1 * np.sin(a1 * x + a2 * y)
    w = np.sin(b1 * x + b2 * y)
    exact = (vx * b1 + vy * b2) * np.cos(b1 * x + b2 * y)
    Wh = dft2(w)
    spectral = vx * idft2(1j * kx * Wh).real + vy * idft2(1j * ky * Wh).real
    assert np.max(np.abs(spectral - exact)) < 1e-12
    # and the stream-function inversion reproduces that v from w_psi = -lap psi = (a1^2+a2^2) psi
    o = TTSHOracle(N, N, dx, 0.01, LIN)
    o.set_velocity(vx, vy)
    assert np.max(np.abs(o.v[0] - vx)) < 1e-13 and np.max(np.abs(o.v[1] - vy)) < 1e-13
    wv = o.get_fields()[2]
    assert np.max(np.abs(wv - (a1 * a1 + a2 * a2) * psi)) < 1e-12     # curl v = w = -lap psi
    psi_o = o.get_fields()[3]
    assert np.max(np.abs(psi_o - psi)) < 1e-12


# ---------------------------------------------------------------- golden: parameters the paper prints
def _gold():
    vals = {}
    with open(os.path.join(GOLD, "table1_params.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                vals[k] = float(v)
    return vals


def test_paper_preset_matches_table_I_and_algorithm_1_symbol():
    g = _gold()
    p = PAPER_PRESET
    assert p.lambda0 == g["lambda"] and p.beta == g["b"] and p.gamma_v == g["gamma_v"] and p.gamma_w == g["gamma_w"]
    assert p.alpha == 1.0 - g["a"]
    k2 = np.array([0.0, 1.0, 0.37, 2.5])
    assert np.allclose(linear_symbol(k2, p), g["a"] - (1.0 - k2) ** 2, atol=1e-15)
    assert linear_symbol(np.array(0.0), p) == g["sigma_at_k0"]
    assert linear_symbol(np.array(1.0), p) == g["sigma_at_k1"]
    for key, sgn in (("k_plus", +1), ("k_minus", -1)):
        k = g[key]
        assert abs(k - np.sqrt(1 + sgn * np.sqrt(g["a"]))) < 1e-15
        assert abs(linear_symbol(np.array(k * k), p)) < 1e-14
    assert (p.dealias_num, p.dealias_den) == (1, 2)


# ---------------------------------------------------------------- linear operator / integrating factor
@pytest.mark.parametrize("lam", [0.0, 3.5])
def test_single_mode_grows_exactly_like_exp_sigma_t(lam):
    # linear terms are integrated "separately and exactly by using the exponential multiplier".
    # v.grad(w) == 0 for a single mode, so this also holds with advection switched on.
    N, dx, dt, n = 32, 0.5, 0.01, 40
    p = TTSHParams(lambda0=lam, alpha=-0.5, beta=0.0, Gamma0=-1.0, Gamma2=1.0, gamma_v=0.0, gamma_w=0.0)
    kx, ky = wavenumbers(N, N, dx)
    mx, my = 3, 2
    qx, qy = kx[0, mx], ky[my, 0]
    x = np.arange(N)[None, :] * dx; y = np.arange(N)[:, None] * dx
    amp = 1e-3
    psi = amp * np.cos(qx * x + qy * y + 0.3)
    vx = -qy * amp * np.sin(qx * x + qy * y + 0.3); vy = qx * amp * np.sin(qx * x + qy * y + 0.3)
    o = TTSHOracle(N, N, dx, dt, p)
    o.set_velocity(vx, vy)
    w0 = o.get_fields()[2]
    o.step(n)
    k2 = qx * qx + qy * qy
    sigma = 0.5 + k2 - k2 * k2
    growth = np.exp(sigma * n * dt)
    assert rel(o.get_fields()[2], growth * w0) < 1e-13
    assert rel(o.v[0], growth * vx) < 1e-13
    assert abs(o.t - n * dt) < 1e-15 and o.nstep == n
    _ = psi


def test_mode_beyond_cutoff_vanishes_and_nyquist_removed():
    N, dx = 32, 0.5
    kx, ky = wavenumbers(N, N, dx)
    x = np.arange(N)[None, :] * dx; y = np.arange(N)[:, None] * dx
    o = TTSHOracle(N, N, dx, 0.01, LIN)
    q = kx[0, 9]                      # 9 > N/4 = 8: beyond the 1/2 cutoff
    o.set_velocity(np.zeros((N, N)), np.sin(q * x) + 0 * y)
    assert np.max(np.abs(o.v)) < 1e-14 and np.max(np.abs(o.w_hat)) < 1e-13
    q = kx[0, 8]                      # exactly on the circle: kept
    o.set_velocity(np.zeros((N, N)), np.sin(q * x) + 0 * y)
    assert rel(o.v[1], np.sin(q * x) + 0 * y) < 1e-13


def test_uniform_flow_fixed_point_closed_form():
    # K = 0, uniform v: w^ = 0 and line 8 gives the map v <- e^{-alpha dt}(v - dt beta |v|^2 v); its fixed
    # point is |v*| = sqrt((1 - e^{alpha dt}) / (beta dt))  ->  sqrt(-alpha/beta) as dt -> 0.
    N, dx, dt = 16, 0.5, 0.01
    p = BASELINE_PRESET
    vstar = np.sqrt((1.0 - np.exp(p.alpha * dt)) / (p.beta * dt))
    assert abs(vstar - 0.998751301107) < 1e-11
    assert abs(vstar - np.sqrt(-p.alpha / p.beta)) < abs(p.alpha) * dt / 4 + 1e-6
    o = TTSHOracle(N, N, dx, dt, p)
    th = 0.7
    o.set_velocity(np.full((N, N), vstar * np.cos(th)), np.full((N, N), vstar * np.sin(th)))
    o.step(100)
    assert np.max(np.abs(o.v[0] - vstar * np.cos(th))) < 5e-15
    assert np.max(np.abs(o.v[1] - vstar * np.sin(th))) < 5e-15
    assert np.max(np.abs(o.w_hat)) < 1e-13
    # one step from another amplitude follows the map exactly (catches a wrong sign of the cubic term)
    o.set_velocity(np.full((N, N), 0.9), np.zeros((N, N)))
    o.step(1)
    assert abs(o.v[0].mean() - np.exp(-p.alpha * dt) * (0.9 - dt * p.beta * 0.9 ** 3)) < 1e-15
    # relaxation to the fixed point
    o.step(2999)
    assert abs(np.hypot(o.v[0].mean(), o.v[1].mean()) - vstar) < 1e-6


def test_paper_preset_uniform_flow_decays():
    # alpha = 1 - a = 0.5 > 0: mean flow decays, rate (a-1) for small amplitude (Eq. C1 :329)
    N, dt = 16, 0.01
    o = TTSHOracle(N, N, 0.5, dt, PAPER_PRESET)
    o.set_velocity(np.full((N, N), 1e-6), np.zeros((N, N)))
    o.step(10)
    assert abs(o.v[0].mean() / 1e-6 - np.exp(-0.5 * 10 * dt)) < 1e-10


def test_damping_closed_form_K_equal_one():
    # K == 1, lambda0 = beta = 0: curl(K v) = w, so one step multiplies every retained mode by
    # e^{sigma dt}(1 - (gamma_v + gamma_w) dt) and the mean flow by e^{-alpha dt}(1 - gamma_v dt).
    N, dx, dt = 32, 0.5, 0.01
    p = TTSHParams(lambda0=0.0, alpha=-0.5, beta=0.0, Gamma0=-1.0, Gamma2=1.0, gamma_v=40.0, gamma_w=4.0)
    ones = np.ones((N, N), dtype=np.uint8)
    o = TTSHOracle(N, N, dx, dt, p, mask=ones, mask_kind="binary")
    assert np.max(np.abs(o.K - 1.0)) < 1e-13                   # all-ones mask passes Algorithm 2 unchanged
    vx, vy = workloads.gaussian_velocity(N, N, 11, 1.0)
    vx = vx + 0.3
    o.set_velocity(vx, vy)
    w_hat0 = o.w_hat.copy(); mean0 = o.v[0].mean()
    o.step(1)
    sigma = linear_symbol(o.k2, p)
    expect = np.exp(sigma * dt) * (1.0 - 44.0 * dt) * w_hat0
    assert rel(o.w_hat, expect) < 1e-13
    assert abs(o.v[0].mean() - np.exp(0.5 * dt) * (1 - 40.0 * dt) * mean0) < 1e-15


def test_euler_is_first_order_in_dt():
    N, dx = 32, 0.5
    mask = workloads.disk_mask(N, N, dx, 5.0)
    vx, vy = workloads.planewave_velocity(N, N, dx, 5, amplitude=0.5, nmodes=6, kmax=1.0)

    def run(dt, T=0.08):
        o = TTSHOracle(N, N, dx, dt, BASELINE_PRESET, mask=mask)
        o.set_velocity(vx, vy)
        o.step(int(round(T / dt)))
        return o.v.copy()

    ref = run(0.01 / 16)
    e1 = np.linalg.norm(run(0.01) - ref)
    e2 = np.linalg.norm(run(0.005) - ref)
    assert 1.7 < e1 / e2 < 2.4


# ---------------------------------------------------------------- stream function, Hermitian repair
def _developed_state(N=32, steps=3, amp=0.8):
    dx = 0.5
    mask = workloads.disk_mask(N, N, dx, 5.0)
    vx, vy = workloads.gaussian_velocity(N, N, 21, amp, mask)
    o = TTSHOracle(N, N, dx, 0.01, BASELINE_PRESET, mask=mask)
    o.set_velocity(vx, vy)
    o.step(steps)
    return o


def test_velocity_is_divergence_free_and_curl_is_omega():
    o = _developed_state()
    vxh, vyh, wh = dft2(o.v[0]), dft2(o.v[1]), o.w_hat
    div = o.kx * vxh + o.ky * vyh
    assert np.max(np.abs(div)) < 1e-14 * max(1.0, np.max(np.abs(vxh)))
    curl = 1j * o.kx * vyh - 1j * o.ky * vxh
    assert np.max(np.abs(curl - wh)) < 1e-13 * np.max(np.abs(wh))
    assert abs(wh[0, 0]) == 0.0 and abs(o.get_fields()[2].sum()) < 1e-11   # w^(0) = 0
    assert np.max(np.abs(wh[o.cut])) == 0.0 and np.max(np.abs(vxh[o.cut])) < 1e-14
    assert np.max(np.abs(wh - np.conj(np.roll(wh[::-1, ::-1], (1, 1), (0, 1))))) < 1e-15


def test_hermitian_average_removes_injected_antihermitian_part():
    o = _developed_state(steps=1)
    good = o.w_hat.copy()
    bad = good.copy()
    bad[3, 5] += 0.25j; bad[0, 7] += 0.1 + 0.2j; bad[4, 0] -= 0.3j         # breaks w^(k) = w^(-k)*
    w_new, _, vxh, vyh = o._post(bad, np.zeros(2))
    refl = np.conj(np.roll(w_new[::-1, ::-1], (1, 1), (0, 1)))
    assert np.max(np.abs(w_new - refl)) < 1e-16
    assert np.max(np.abs(idft2(w_new).imag)) < 1e-15 and np.max(np.abs(idft2(vxh).imag)) < 1e-15
    assert abs(w_new[3, 5] - (good[3, 5] + 0.125j)) < 1e-15                # exactly the average of line 12


# ---------------------------------------------------------------- Algorithm 2
def test_mask_processing_invariants():
    N, dx = 64, 0.5
    Kn = workloads.disk_mask(N, N, dx, 12.0)
    K = process_mask(Kn)
    assert K.min() >= 0.0                                                   # squared => K >= 0
    Kh = dft2(K)
    assert np.max(np.abs(Kh[cut_mask(N, N, 1, 2)])) < 1e-13 * np.abs(Kh).max()   # obeys the 1/2 rule
    assert abs(dft2(Kn.astype(float))[0, 0].real - Kn.sum() / N) < 1e-10     # K^_naive(0) = #masked / sqrt(P)
    s = np.sqrt(K)
    assert 0.95 < s.max() < 1.2                                             # Gibbs overshoot range (Fig. 1c)
    assert K[N // 2, N // 2] < 1e-2 and K[0, 0] > 0.8                       # ~0 inside, ~1 outside
    assert np.max(np.abs(process_mask(np.zeros((N, N))))) == 0.0
    assert np.max(np.abs(process_mask(np.ones((N, N))) - 1.0)) < 1e-13
    assert rel(process_mask(Kn, "fft"), K) < 1e-13
    # dumbbell = AND of two circle masks: inside either circle is unmasked
    D = workloads.dumbbell_mask(128, 64, 0.5, 10.0, 12.0)
    assert D[32, 64] == 0 and D[32, 64 - 12 - 18] == 0 and D[32, 64 + 12 + 18] == 0 and D[32, 64 + 12 + 21] == 1
    assert D[32 + 15, 64] == 0 and D[32 + 16, 64] == 1 and D[0, 0] == 1     # waist half-height sqrt(R^2-(d/2)^2) = 8 = 16 pts (>= R is masked)


def test_confinement_keeps_the_flow_small_deep_inside_the_wall():
    cfg = workloads.CONFIGS["C1"]
    mask = cfg.mask()
    vx, vy = cfg.initial_velocity(mask)
    o = TTSHOracle(cfg.Nx, cfg.Ny, cfg.dx, cfg.dt, BASELINE_PRESET, mask=mask, transform="fft")
    o.set_velocity(vx, vy)
    o.step(100)
    i = np.arange(cfg.Nx)[None, :] - cfg.Nx // 2; j = np.arange(cfg.Ny)[:, None] - cfg.Ny // 2
    r = np.hypot(i, j) * cfg.dx
    speed = np.hypot(o.v[0], o.v[1])
    assert speed[r > cfg.R + 4.0].max() < 1e-2 * speed[r < cfg.R - 2.0].max()


# ---------------------------------------------------------------- diagnostics (Eq. 11; R13)
def test_vortex_order_parameter_limits_and_parseval():
    N, dx = 64, 0.5
    o = TTSHOracle(N, N, dx, 0.01, BASELINE_PRESET)
    cx = cy = (N // 2) * dx
    x = np.arange(N)[None, :] * dx - cx; y = np.arange(N)[:, None] * dx - cy
    r = np.hypot(x, y); rs = np.where(r == 0, 1.0, r)
    o.w_hat = np.zeros((N, N), complex)
    o.v = np.stack([-y / rs * np.exp(-r), x / rs * np.exp(-r)])               # purely azimuthal
    d = o.diagnostics(cx, cy)
    assert abs(d["vortex_order"] - 1.0) < 1e-12                               # "Psi = 1 if completely azimuthal"
    o.v = np.stack([x / rs * np.exp(-r), y / rs * np.exp(-r)])                # purely radial
    d = o.diagnostics(cx, cy)
    assert abs(d["vortex_order"] + (2 / np.pi) / (1 - 2 / np.pi)) < 1e-12
    o.v = np.stack([np.full((N, N), 0.3), np.full((N, N), -0.4)])             # uniform
    d = o.diagnostics(cx, cy)
    assert abs(d["polar_order"] - 1.0) < 1e-13 and abs(d["kinetic_energy"] - 0.125) < 1e-15
    assert abs(d["mean_vx"] - 0.3) < 1e-15 and abs(d["max_speed"] - 0.5) < 1e-15
    # disordered field: Psi ~ 0 ("Psi = 0 if completely disordered")
    g = rng(5)
    th = g.uniform(0, 2 * np.pi, (N, N))
    o.v = np.stack([np.cos(th), np.sin(th)])
    assert abs(o.diagnostics(cx, cy)["vortex_order"]) < 0.05
    # Parseval on a developed state
    s = _developed_state()
    d = s.diagnostics(8.0, 8.0)
    P = s.Nx * s.Ny
    vxh, vyh = dft2(s.v[0]), dft2(s.v[1])
    assert abs(d["kinetic_energy"] - 0.5 * np.sum(np.abs(vxh) ** 2 + np.abs(vyh) ** 2) / P) < 1e-14
    assert abs(d["enstrophy"] - 0.5 * np.sum(np.abs(s.w_hat) ** 2) / P) < 1e-13
    assert d["nonfinite"] == 0
    o.v = np.zeros((2, N, N))
    d0 = o.diagnostics(cx, cy)
    assert d0["vortex_order"] == 0.0 and d0["polar_order"] == 0.0


def test_diagnostics_centre_on_a_non_square_grid_and_both_mean_components():
    """Eq. (11) about a centre with cx != cy on a non-square grid: a field that is azimuthal about
    (cx, cy) gives Psi = 1 only about that centre (a swapped or transposed centre does not); mean_vx and mean_vy are
    distinct numbers; max_speed and the sums follow the closed forms of a hand-built field."""
    Nx, Ny, dx = 96, 48, 0.5
    o = TTSHOracle(Nx, Ny, dx, 0.01, BASELINE_PRESET)
    cx, cy = 30 * dx, 11 * dx                                               # grid points, cx != cy, neither the box centre
    x = np.arange(Nx)[None, :] * dx - cx; y = np.arange(Ny)[:, None] * dx - cy
    r = np.hypot(x, y); rs = np.where(r == 0, 1.0, r)
    o.w_hat = np.zeros((Ny, Nx), complex)
    o.v = np.stack([-y / rs * np.exp(-0.3 * r), x / rs * np.exp(-0.3 * r)])   # azimuthal about (cx, cy)
    assert abs(o.diagnostics(cx, cy)["vortex_order"] - 1.0) < 1e-12
    assert o.diagnostics(cy, cx)["vortex_order"] < 0.9                       # swapped coordinates: not the centre
    assert o.diagnostics(cx, cy + 4.0)["vortex_order"] < 0.99 and o.diagnostics(cx + 4.0, cy)["vortex_order"] < 0.99
    # uniform flow with different components: both means, polar order, energy
    o.v = np.stack([np.full((Ny, Nx), 0.3), np.full((Ny, Nx), -0.4)])
    d = o.diagnostics(cx, cy)
    assert abs(d["mean_vx"] - 0.3) < 1e-15 and abs(d["mean_vy"] + 0.4) < 1e-15
    assert abs(d["polar_order"] - 1.0) < 1e-13 and abs(d["sum_speed"] - 0.5 * Nx * Ny) < 1e-9
    # uniform flow (u, 0): |e_theta . v| = |u| |y| / r, summed by hand about (cx, cy)
    o.v = np.stack([np.full((Ny, Nx), 0.7), np.zeros((Ny, Nx))])
    want = 0.7 * np.sum(np.where(r == 0, 0.0, np.abs(y) / rs))
    d = o.diagnostics(cx, cy)
    assert abs(d["sum_abs_vtheta"] - want) < 1e-10 * want
    want_t = 0.7 * np.sum(np.where(r == 0, 0.0, np.abs(x) / rs))            # (0, u): |x| / r instead
    o.v = np.stack([np.zeros((Ny, Nx)), np.full((Ny, Nx), 0.7)])
    assert abs(o.diagnostics(cx, cy)["sum_abs_vtheta"] - want_t) < 1e-10 * want_t and abs(want - want_t) > 1e-3 * want


def test_nonfinite_counts_every_field():
    """`nonfinite` counts the non-finite entries of v_x, v_y AND w (reading R13): one bad value in each, separately."""
    N, dx = 16, 0.5
    for which, bad in (("vx", np.nan), ("vy", np.inf), ("w", np.nan)):
        o = TTSHOracle(N, N, dx, 0.01, LIN)
        o.w_hat = np.zeros((N, N), complex)
        o.v = np.zeros((2, N, N))
        if which == "vx":
            o.v[0, 3, 5] = bad
        elif which == "vy":
            o.v[1, 7, 2] = bad
        else:
            o.w_hat[0, 0] = bad                                              # w = iDFT[w^]: every point non-finite
        want = N * N if which == "w" else 1
        with np.errstate(all="ignore"):
            assert o.diagnostics(4.0, 4.0)["nonfinite"] == want, which


def test_rhs_terms_signs_on_a_hand_computable_field():
    # uniform v = (u, 0), w = A sin(qx x): rhs1 = -beta u^3 - gamma_v K u ; rhs2 = -lambda0 u A qx cos(qx x) - gamma_w K w
    N, dx = 16, 0.5
    p = BASELINE_PRESET
    Kf = 0.25 + 0.1 * np.cos(2 * np.pi * np.arange(N) / N)[None, :] * np.ones((N, 1))
    o = TTSHOracle(N, N, dx, 0.01, p, mask=Kf, mask_kind="processed")
    kx, _ = wavenumbers(N, N, dx)
    x = np.arange(N)[None, :] * dx + 0 * np.arange(N)[:, None]
    q, A, u = kx[0, 2], 0.7, 0.6
    o.v = np.stack([np.full((N, N), u), np.zeros((N, N))])
    o.w_hat = dft2(A * np.sin(q * x))
    w, gx, gy, rhs1, rhs2 = o.rhs_real()
    assert np.max(np.abs(rhs1[0] - (-p.beta * u ** 3 - p.gamma_v * Kf * u))) < 1e-14
    assert np.max(np.abs(rhs1[1])) == 0.0
    assert np.max(np.abs(rhs2 - (-p.lambda0 * u * A * q * np.cos(q * x) - p.gamma_w * Kf * A * np.sin(q * x)))) < 1e-13
    assert np.max(np.abs(gy)) < 1e-14


# ---------------------------------------------------------------- Psi_2 of the dumbbell geometry
def _two_vortices(Nx, Ny, dx, cl, cr, al, ar, width=3.0):
    x = np.arange(Nx)[None, :] * dx
    y = np.arange(Ny)[:, None] * dx
    g = lambda c: np.exp(-((x - c[0]) ** 2 + (y - c[1]) ** 2) / (2 * width ** 2))
    return al * g(cl) + ar * g(cr)


def test_psi2_ferromagnetic_antiferromagnetic_and_closed_form():
    """'By construction, Psi_2 = 1 for the ferromagnetic flow and 0 for the antiferromagnetic one'; for peak
    vorticities a and -b the definition gives |a - b| / (a + b)."""
    from oracle import psi2_of_field
    Nx, Ny, dx = 96, 48, 0.5
    cl, cr = (14.0, 12.0), (34.0, 12.0)            # grid points (28, 24) and (68, 24)
    r = 6.0
    d = psi2_of_field(_two_vortices(Nx, Ny, dx, cl, cr, 2.0, 0.7), dx, cl, cr, r)
    assert d["psi2"] == 1.0 and d["index_left"] == 24 * Nx + 28 and d["index_right"] == 24 * Nx + 68
    d = psi2_of_field(_two_vortices(Nx, Ny, dx, cl, cr, -1.5, -1.5), dx, cl, cr, r)
    assert d["psi2"] == 1.0
    d = psi2_of_field(_two_vortices(Nx, Ny, dx, cl, cr, 1.25, -1.25), dx, cl, cr, r)
    assert d["psi2"] == 0.0
    a, b = 2.0, 0.5
    w = _two_vortices(Nx, Ny, dx, cl, cr, a, -b)
    d = psi2_of_field(w, dx, cl, cr, r)
    wl, wr = w[24, 28], w[24, 68]                   # the peaks (each Gaussian leaks ~1e-10 into the other cavity)
    assert d["omega_left"] == wl and d["omega_right"] == wr
    assert abs(d["psi2"] - (a - b) / (a + b)) < 1e-8 and d["psi2"] == abs(wl + wr) / (abs(wl) + abs(wr))


def test_psi2_region_ties_and_degenerate_cases():
    from oracle import psi2_of_field
    Nx, Ny, dx = 40, 32, 0.5
    cl, cr = (5.0, 8.0), (14.0, 8.0)
    # a larger peak OUTSIDE both regions is ignored
    w = _two_vortices(Nx, Ny, dx, cl, cr, 1.0, 1.0, width=1.0)
    w[2, 2] = 50.0
    w[31, 39] = -80.0
    d = psi2_of_field(w, dx, cl, cr, 3.0)
    assert d["index_left"] == 16 * Nx + 10 and d["index_right"] == 16 * Nx + 28 and d["psi2"] == 1.0
    # the region is inclusive (<=) and uses the plain distance: radius 1.0 about a grid point holds exactly 13 points at dx = 0.5
    ones = np.ones((Ny, Nx))
    marked = np.zeros((Ny, Nx))
    for j in range(Ny):
        for i in range(Nx):
            if (i * dx - 5.0) ** 2 + (j * dx - 8.0) ** 2 <= 1.0:
                marked[j, i] = 1.0
    assert marked.sum() == 13
    # ties in |w| -> lowest linear index j Nx + i: the topmost point of the disk, (x, y) = (5.0, 7.0) -> (i, j) = (10, 14)
    d = psi2_of_field(ones, dx, cl, cr, 1.0)
    assert d["index_left"] == 14 * Nx + 10 and d["index_right"] == 14 * Nx + 28 and d["psi2"] == 1.0
    # sign does not break a tie in |w|
    w = ones.copy(); w[14, 10] = -1.0
    assert psi2_of_field(w, dx, cl, cr, 1.0)["index_left"] == 14 * Nx + 10
    assert psi2_of_field(w, dx, cl, cr, 1.0)["psi2"] == 0.0
    # zero field, and a region without grid points
    assert psi2_of_field(np.zeros((Ny, Nx)), dx, cl, cr, 1.0)["psi2"] == 0.0
    d = psi2_of_field(ones, dx, (5.25, 8.25), cr, 0.1)
    assert d["index_left"] == -1 and d["psi2"] == 0.0


def test_psi2_of_the_oracle_state_uses_the_real_vorticity():
    """TTSHOracle.dumbbell_order = psi2_of_field(iDFT[w^]): a two-vortex initial condition in a dumbbell keeps its signs."""
    Nx, Ny, dx = 64, 32, 0.5
    mask = workloads.dumbbell_mask(Nx, Ny, dx, 6.0, 9.0)
    cl, cr = ((Nx // 2) * dx - 4.5, (Ny // 2) * dx), ((Nx // 2) * dx + 4.5, (Ny // 2) * dx)
    x = np.arange(Nx)[None, :] * dx
    y = np.arange(Ny)[:, None] * dx
    def vortex(c, s):   # solid-body-like swirl with Gaussian envelope
        e = np.exp(-((x - c[0]) ** 2 + (y - c[1]) ** 2) / 8.0)
        return -s * (y - c[1]) * e, s * (x - c[0]) * e
    for sl, sr, expect in ((1.0, 1.0, 1.0), (1.0, -1.0, 0.0)):
        vxl, vyl = vortex(cl, sl); vxr, vyr = vortex(cr, sr)
        o = TTSHOracle(Nx, Ny, dx, 0.01, BASELINE_PRESET, mask=mask)
        o.set_velocity(vxl + vxr, vyl + vyr)
        d = o.dumbbell_order(cl, cr, 4.5)
        assert abs(d["psi2"] - expect) < 1e-6
        w = o.get_fields()[2]
        assert d["omega_left"] == w.flat[d["index_left"]] and d["omega_right"] == w.flat[d["index_right"]]


# ---------------------------------------------------------------- temporal PSD, Eq. (5)
def test_temporal_psd_closed_forms_and_library_special_case():
    from oracle import temporal_psd
    rng = np.random.default_rng(5)
    Ny, Nx, n, dt = 6, 8, 64, 0.25
    times = [k * dt for k in range(n)]
    a = rng.standard_normal((Ny, Nx))
    b = rng.standard_normal((Ny, Nx))
    base = 2 * np.pi / (n * dt)                         # DFT frequencies of the sampling window
    # (i) w(x, t) = a(x) cos(3 base t) + b(x) sin(3 base t) over whole periods: all the power sits at +-3 base,
    #     S = (n/2)^2 mean(a^2 + b^2); orthogonal DFT frequencies carry nothing
    series = [a * np.cos(3 * base * t) + b * np.sin(3 * base * t) for t in times]
    S = temporal_psd(series, times, [3 * base, -3 * base, 2 * base, 5 * base, 0.0])
    want = (n / 2) ** 2 * np.mean(a * a + b * b)
    assert abs(S[0] - want) < 1e-10 * want and abs(S[1] - want) < 1e-10 * want
    assert max(S[2], S[3], S[4]) < 1e-20 * want
    # (ii) a constant field: S(0) = n^2 mean(w^2)
    S = temporal_psd([a] * n, times, [0.0])
    assert abs(S[0] - n * n * np.mean(a * a)) < 1e-12 * S[0]
    # (iii) on the DFT frequencies the inner sum is numpy's FFT over the time axis (a shifted time origin only rotates
    #       the phase), and (iv) Parseval: sum_m S(Omega_m) = n sum_t mean(w(t)^2)
    series = [rng.standard_normal((Ny, Nx)) for _ in range(n)]
    t0 = 3.7
    S = temporal_psd(series, [t0 + t for t in times], [m * base for m in range(n)])
    F = np.fft.fft(np.stack(series), axis=0)
    assert np.allclose(S, np.mean(np.abs(F) ** 2, axis=(1, 2)), rtol=1e-11, atol=0)
    assert abs(S.sum() - n * sum(np.mean(f * f) for f in series)) < 1e-11 * S.sum()
    # (v) for a real series S(-W) = S(+W) exactly (the accumulators are complex conjugates of each other), so the sign of the
    #     exponent in Eq. (5) is not observable in S; what is observable is that HALF the power of a real cosine sits at +W
    W = 7 * base
    S = temporal_psd([a * np.cos(W * t) for t in times], times, [W, -W])
    assert S[0] == S[1] and abs(S[0] - (n / 2) ** 2 * np.mean(a * a)) < 1e-10 * S[0]
    # a non-DFT frequency against the explicit double sum on one point
    Om = 1.2345
    one = [np.full((1, 1), np.sin(0.9 * t) + 0.3) for t in times]
    ref = abs(sum((np.sin(0.9 * t) + 0.3) * np.exp(-1j * Om * t) for t in times)) ** 2
    assert abs(temporal_psd(one, times, [Om])[0] - ref) < 1e-12 * ref



# ---------------------------------------------------------------- tangent-linear step and QR growth rates
def _o1_state(Nx, Ny, dx, seed, amp=1.0):
    return workloads.planewave_velocity(Nx, Ny, dx, seed, amplitude=amp, nmodes=10)


def test_tangent_step_is_the_derivative_of_the_nonlinear_step():
    """Central finite differences of the NONLINEAR oracle (which the tangent code does not call for its arithmetic):
    (Phi^n(s + eps d) - Phi^n(s - eps d)) / 2 eps = J_n d + O(eps^2).  O(1) base state inside a disk, so that the cubic,
    advection and both damping terms all contribute; n = 1 and n = 3 (composition along the moving base state)."""
    from oracle.tangent import TangentOracle
    Nx, Ny, dx, dt = 32, 64, 0.5, 0.01
    mask = workloads.disk_mask(Nx, Ny, dx, 6.0)
    v0 = _o1_state(Nx, Ny, dx, 11)
    d0 = _o1_state(Nx, Ny, dx, 12, amp=0.7)
    d0 = (d0[0] + 0.3, d0[1] - 0.2)                       # with a mean-flow component (line 8 of Algorithm 1)
    eps = 1e-5
    for n in (1, 3):
        plus = TTSHOracle(Nx, Ny, dx, dt, BASELINE_PRESET, mask=mask)
        minus = TTSHOracle(Nx, Ny, dx, dt, BASELINE_PRESET, mask=mask)
        plus.set_velocity(v0[0] + eps * d0[0], v0[1] + eps * d0[1]); plus.step(n)
        minus.set_velocity(v0[0] - eps * d0[0], v0[1] - eps * d0[1]); minus.step(n)
        fd = [(a - b) / (2 * eps) for a, b in zip(plus.get_fields()[:3], minus.get_fields()[:3])]
        base = TTSHOracle(Nx, Ny, dx, dt, BASELINE_PRESET, mask=mask)
        base.set_velocity(*v0)
        tan = TangentOracle(base, 1)
        tan.set(0, *d0)
        tan.step(n)
        got = tan.get_fields(0)
        for f, g in zip(fd, got):
            assert np.linalg.norm(f - g) <= 1e-8 * np.linalg.norm(f), np.linalg.norm(f - g) / np.linalg.norm(f)
        assert base.nstep == n                              # the tangent step advances the base trajectory too
    # a dropped term must be visible at this tolerance: the advection part alone is far larger than 1e-8
    assert BASELINE_PRESET.lambda0 * dt > 1e-3


def test_tangent_about_the_zero_state_is_the_linear_operator():
    """Base state 0, no mask: the Jacobian is exp(sigma(k) dt) per mode (Alg. 1 line 4), so a single-mode perturbation
    grows by exactly exp(sigma(k) n dt) and its growth rate from the QR diagonal is sigma(k)."""
    from oracle.tangent import TangentOracle
    Nx = Ny = 32
    dx, dt, n = 0.5, 0.01, 7
    base = TTSHOracle(Nx, Ny, dx, dt, BASELINE_PRESET)
    z = np.zeros((Ny, Nx))
    base.set_velocity(z, z)
    x = np.arange(Nx)[None, :] * dx
    y = np.arange(Ny)[:, None] * dx
    kx, ky = 2 * np.pi * 2 / (Nx * dx), 2 * np.pi * 1 / (Ny * dx)          # retained mode (2, 1)
    ph = kx * x + ky * y
    dvx, dvy = ky * np.cos(ph), -kx * np.cos(ph)                            # divergence-free single mode
    tan = TangentOracle(base, 2)
    tan.set(0, dvx, dvy)
    tan.set(1, np.ones((Ny, Nx)), z)                                        # pure mean flow: grows by exp(-alpha dt)
    tan.orthonormalize()
    tan.step(n)
    logr = tan.orthonormalize()
    k2 = kx * kx + ky * ky
    p = BASELINE_PRESET
    sigma = -p.alpha - p.Gamma0 * k2 - p.Gamma2 * k2 * k2
    assert abs(logr[0] / (n * dt) - sigma) < 1e-10
    assert abs(logr[1] / (n * dt) - (-p.alpha)) < 1e-10


def test_tangent_qr_orthonormalises_and_measures_the_volume():
    from oracle.tangent import TangentOracle
    Nx, Ny, dx, dt = 32, 32, 0.5, 0.01
    mask = workloads.disk_mask(Nx, Ny, dx, 5.0)
    base = TTSHOracle(Nx, Ny, dx, dt, BASELINE_PRESET, mask=mask)
    base.set_velocity(*_o1_state(Nx, Ny, dx, 21))
    tan = TangentOracle(base, 3)
    for i in range(3):
        tan.set(i, *_o1_state(Nx, Ny, dx, 30 + i))
    A = tan.as_matrix()
    logr = tan.orthonormalize()
    sign, logdet = np.linalg.slogdet(A.T @ A)
    assert sign > 0 and abs(2 * logr.sum() - logdet) < 1e-9                 # prod R_ii^2 = det(Gram)
    Q = tan.as_matrix()
    assert np.allclose(Q.T @ Q, np.eye(3), atol=1e-12)                      # and the stored states reproduce Q
    # sign convention R_ii > 0: q_i has a positive component along a_i (Gram-Schmidt's choice), and A = Q R with the
    # upper-triangular R = Q^T A whose diagonal is exp(logr)
    R = Q.T @ A
    assert np.all(np.diag(R) > 0) and np.allclose(np.diag(R), np.exp(logr), rtol=1e-10)
    assert np.allclose(np.tril(R, -1), 0.0, atol=1e-9 * np.abs(R).max()) and np.allclose(Q @ R, A, atol=1e-9 * np.abs(A).max())
    assert abs(Q[:, 0] @ A[:, 0] - np.linalg.norm(A[:, 0])) < 1e-10 * np.linalg.norm(A[:, 0])   # q_0 = +a_0 / |a_0|
    assert np.allclose(tan.orthonormalize(), 0.0, atol=1e-12)               # idempotent: R = I
