"""Pins of oracle/ttsh_oracle_c.c ("oracle-fft": Algorithm 1/2 restated in plain C with a radix-2 FFT; no GPU).

It is (i) locked to the definition-oracle (explicit DFT-matrix products, oracle/ttsh_oracle.py) on whole trajectories, the
processed mask and the diagnostics, on square and non-square grids and for both parameter sets, and (ii) run alone through the
closed forms that pin the definition-oracle itself (single-mode growth exp(sigma n dt); the discrete uniform
fixed point; the K = 1 damping closed form), so that a mistake in the C code cannot hide behind a matching mistake elsewhere."""
import numpy as np
import pytest

from oracle import BASELINE_PRESET, PAPER_PRESET, TTSHOracle, TTSHParams
from oracle.c_oracle import TTSHOracleC
from paper_2304_03306_b200 import workloads


def rel(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def maxrel(a, b):
    return float(np.max(np.abs(np.asarray(a) - np.asarray(b))) / max(np.max(np.abs(b)), 1e-300))


CASES = [
    ("64x64 disk baseline", 64, 64, BASELINE_PRESET, "disk", 1.0),
    ("64x64 disk paper", 64, 64, PAPER_PRESET, "disk", 1.0),
    ("128x32 dumbbell", 128, 32, BASELINE_PRESET, "dumbbell", 1.0),
    ("32x128 disk noise", 32, 128, BASELINE_PRESET, "disk", 1e-2),
]


@pytest.mark.parametrize("name,Nx,Ny,p,geom,amp", CASES)
def test_c_oracle_locked_to_the_definition_oracle(name, Nx, Ny, p, geom, amp):
    dx, dt = 0.5, 0.01
    R = 0.3 * min(Nx, Ny) * dx
    mask = workloads.disk_mask(Nx, Ny, dx, R) if geom == "disk" else workloads.dumbbell_mask(Nx, Ny, dx, 5.0, 7.0)
    if amp < 0.1:
        vel = workloads.gaussian_velocity(Nx, Ny, workloads.SEED0 + 11, amp, mask)
    else:
        vel = workloads.planewave_velocity(Nx, Ny, dx, workloads.SEED0 + 11, amplitude=amp, nmodes=10)
    vel = (vel[0] + 0.2, vel[1] - 0.1)                                   # non-zero mean flow (line 8)
    o = TTSHOracle(Nx, Ny, dx, dt, p, mask=mask)
    c = TTSHOracleC(Nx, Ny, dx, dt, p, mask=mask)
    assert maxrel(c.K, o.K) <= 1e-13                                      # Algorithm 2
    o.set_velocity(*vel); c.set_velocity(*vel)
    for n in (0, 1, 20):
        o.step(n - o.nstep); c.step(n - c.nstep)
        fo, fc = o.get_fields(), c.get_fields()
        assert rel(np.stack(fc[:2]), np.stack(fo[:2])) <= 1e-13 and maxrel(np.stack(fc[:2]), np.stack(fo[:2])) <= 1e-12, (name, n)
        # psi^ = w^/k^2 amplifies the round-off of the low-k modes (white-noise start: psi is dominated by them): 1e-12
        assert rel(fc[2], fo[2]) <= 1e-13 and rel(fc[3], fo[3]) <= 1e-12, (name, n)
    cx, cy = (Nx // 2 - 3) * dx, (Ny // 2 + 2) * dx                       # cx != cy
    do, dc = o.diagnostics(cx, cy), c.diagnostics(cx, cy)
    for k in ("kinetic_energy", "enstrophy", "sum_speed", "sum_abs_vtheta", "max_speed"):
        assert abs(dc[k] - do[k]) <= 1e-12 * abs(do[k]), k
    for k in ("mean_vx", "mean_vy", "vortex_order", "polar_order"):
        assert abs(dc[k] - do[k]) <= 1e-12, k
    assert dc["nonfinite"] == 0 and dc["step"] == 20 and abs(dc["t"] - 0.2) < 1e-12


def test_c_oracle_other_dealias_fraction_and_processed_mask():
    from dataclasses import replace
    Nx, Ny, dx, dt = 64, 32, 0.5, 0.01
    p = replace(BASELINE_PRESET, dealias_num=2, dealias_den=3)
    K = 0.5 + 0.5 * np.cos(2 * np.pi * np.arange(Nx) / Nx)[None, :] * np.ones((Ny, 1))
    vel = workloads.planewave_velocity(Nx, Ny, dx, 5, amplitude=1.0, nmodes=6)
    o = TTSHOracle(Nx, Ny, dx, dt, p, mask=K, mask_kind="processed")
    c = TTSHOracleC(Nx, Ny, dx, dt, p, mask=K, mask_kind="processed")
    o.set_velocity(*vel); c.set_velocity(*vel)
    o.step(5); c.step(5)
    assert rel(c.get_fields()[2], o.get_fields()[2]) <= 1e-13


@pytest.mark.parametrize("lam", [0.0, 3.5])
def test_c_oracle_single_mode_closed_form(lam):
    """One retained Fourier mode, beta = gamma = 0: w(x, n dt) = exp(sigma(k) n dt) w(x, 0) exactly, also with
    advection switched on (v . grad w == 0 for a single mode)."""
    N, dx, dt, n = 64, 0.5, 0.01, 50
    p = TTSHParams(lambda0=lam, alpha=-0.5, beta=0.0, Gamma0=-1.0, Gamma2=1.0, gamma_v=0.0, gamma_w=0.0)
    k = 2 * np.pi * np.array([5, 3]) / (N * dx)
    x = np.arange(N)[None, :] * dx; y = np.arange(N)[:, None] * dx
    ph = k[0] * x + k[1] * y + 0.7
    vx0, vy0 = -k[1] * 1e-3 * np.sin(ph), k[0] * 1e-3 * np.sin(ph)
    c = TTSHOracleC(N, N, dx, dt, p)
    c.set_velocity(vx0, vy0)
    c.step(n)
    k2 = float(k @ k)
    g = np.exp((0.5 + k2 - k2 * k2) * n * dt)
    vx, vy, w, psi = c.get_fields()
    assert rel(vx, g * vx0) < 1e-12 and rel(vy, g * vy0) < 1e-12
    assert rel(w, g * 1e-3 * k2 * np.cos(ph)) < 1e-12 and rel(psi, g * 1e-3 * np.cos(ph)) < 1e-12
    # a mode beyond the 1/2 cutoff vanishes
    kc = 2 * np.pi * np.array([20, 0]) / (N * dx)
    c.set_velocity(0 * x + 0 * y, np.cos(kc[0] * x) + 0 * y)
    assert np.max(np.abs(c.get_fields()[1])) < 1e-14


def test_c_oracle_uniform_fixed_point_and_damping_closed_form():
    N, dx, dt = 32, 0.5, 0.01
    p = BASELINE_PRESET
    vstar = np.sqrt((1.0 - np.exp(p.alpha * dt)) / (p.beta * dt))        # discrete fixed point, -> sqrt(-alpha/beta) = 1
    assert abs(vstar - 0.998751301107) < 1e-11
    c = TTSHOracleC(N, N, dx, dt, p)
    c.set_velocity(np.full((N, N), 0.6 * vstar), np.full((N, N), 0.8 * vstar))
    c.step(100)
    vx, vy, w, _ = c.get_fields()
    assert np.max(np.abs(vx - 0.6 * vstar)) < 1e-13 and np.max(np.abs(vy - 0.8 * vstar)) < 1e-13 and np.max(np.abs(w)) < 1e-14
    # K == 1 (all-ones mask through Algorithm 2), lambda0 = beta = 0: one step multiplies the mean flow by
    # exp(-alpha dt) (1 - gamma_v dt) and every mode of w by exp(sigma dt) (1 - (gamma_v + gamma_w) dt)
    q = TTSHParams(lambda0=0.0, alpha=-0.5, beta=0.0, Gamma0=-1.0, Gamma2=1.0, gamma_v=40.0, gamma_w=4.0)
    c = TTSHOracleC(N, N, dx, dt, q, mask=np.ones((N, N), dtype=np.uint8))
    assert np.max(np.abs(c.K - 1.0)) < 1e-13
    k = 2 * np.pi * np.array([2, 1]) / (N * dx)
    x = np.arange(N)[None, :] * dx; y = np.arange(N)[:, None] * dx
    ph = k[0] * x + k[1] * y
    c.set_velocity(0.3 - k[1] * np.sin(ph), k[0] * np.sin(ph))
    c.step(1)
    vx, vy, w, _ = c.get_fields()
    k2 = float(k @ k)
    gw = np.exp((0.5 + k2 - k2 * k2) * dt) * (1 - 44.0 * dt)
    assert rel(w, gw * k2 * np.cos(ph)) < 1e-12
    assert abs(vx.mean() - 0.3 * np.exp(0.5 * dt) * (1 - 40.0 * dt)) < 1e-14


def test_c_hermitian_average_removes_injected_antihermitian_part():
    """Line 12 of Algorithm 1, w^(k) = 1/2 {w^(k) + w^(-k)*}, in the C restatement: its trajectories only ever
    feed it spectra of real fields, which are Hermitian already, so the line is pinned here on a spectrum that is not."""
    from oracle import idft2
    N, dx = 32, 0.5
    mask = workloads.disk_mask(N, N, dx, 5.0)
    vel = workloads.gaussian_velocity(N, N, 21, 0.8, mask)
    o = TTSHOracle(N, N, dx, 0.01, BASELINE_PRESET, mask=mask)
    c = TTSHOracleC(N, N, dx, 0.01, BASELINE_PRESET, mask=mask)
    o.set_velocity(*vel); o.step(1)
    good = o.w_hat.copy()
    bad = good.copy()
    bad[3, 5] += 0.25j; bad[0, 7] += 0.1 + 0.2j; bad[4, 0] -= 0.3j         # breaks w^(k) = w^(-k)*
    v0 = np.array([0.3, -0.2])
    w_new, vxh, vyh = c.debug_post(bad, v0)
    refl = np.conj(np.roll(w_new[::-1, ::-1], (1, 1), (0, 1)))
    assert np.max(np.abs(w_new - refl)) < 1e-16                            # Hermitian after the step
    assert np.max(np.abs(idft2(w_new).imag)) < 1e-15 and np.max(np.abs(idft2(vxh).imag)) < 1e-15
    assert abs(w_new[3, 5] - (good[3, 5] + 0.125j)) < 1e-15                # exactly the average of line 12
    assert abs(w_new[N - 3, N - 5] - np.conj(good[3, 5] + 0.125j)) < 1e-15  # and its mirror image at -k
    assert abs(w_new[0, 7] - (good[0, 7] + 0.05 + 0.1j)) < 1e-15 and abs(w_new[4, 0] - (good[4, 0] - 0.15j)) < 1e-15
    assert w_new[0, 0] == 0 and vxh[0, 0] == v0[0] and vyh[0, 0] == v0[1]  # lines 7-8
    # the same lines of the definition-oracle on the same input
    ow, _, ovx, ovy = o._post(bad, v0)
    assert np.max(np.abs(w_new - ow)) < 1e-15 and np.max(np.abs(vxh - ovx)) < 1e-15 and np.max(np.abs(vyh - ovy)) < 1e-15
    c.close()


def test_c_nonfinite_counts_every_field():
    """`nonfinite` counts the non-finite entries of v_x, v_y AND w (reading R13): one bad value in each, separately."""
    N, dx = 16, 0.5
    lin = TTSHParams(lambda0=0.0, alpha=-0.5, beta=0.0, Gamma0=-1.0, Gamma2=1.0, gamma_v=0.0, gamma_w=0.0)
    for which, bad in (("vx", np.nan), ("vy", np.inf), ("w", np.nan)):
        c = TTSHOracleC(N, N, dx, 0.01, lin)
        w_hat = np.zeros((N, N), complex); vx = np.zeros((N, N)); vy = np.zeros((N, N))
        if which == "vx":
            vx[3, 5] = bad
        elif which == "vy":
            vy[7, 2] = bad
        else:
            w_hat[0, 0] = bad                                              # w = iDFT[w^]: every point non-finite
        c.debug_set_state(w_hat, vx, vy)
        assert c.diagnostics(4.0, 4.0)["nonfinite"] == (N * N if which == "w" else 1), which
        c.close()
