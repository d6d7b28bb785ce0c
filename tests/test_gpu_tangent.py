"""GPU parity of the tangent-linear step and the QR growth rates against
oracle/tangent.py: perturbation fields element by element, log R_ii of the re-orthonormalisation, and the exact growth
about the zero state."""
import numpy as np
import pytest

from oracle import BASELINE_PRESET, TTSHOracle
from oracle.tangent import TangentOracle
from paper_2304_03306_b200 import workloads

pytestmark = pytest.mark.gpu

TOL_1, TOL_N = 1e-12, 1e-9


@pytest.fixture(scope="module")
def ttsh():
    import __graft_entry__ as ge
    ge.build()
    from paper_2304_03306_b200 import ttsh as t
    return t


def rel(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def setup(ttsh, Nx, Ny, nvec, dtype="f64", R=None, base_amp=1.0, transform="matmul"):
    dx, dt = 0.5, 0.01
    mask = workloads.disk_mask(Nx, Ny, dx, R if R is not None else 0.3 * min(Nx, Ny) * dx)
    v0 = workloads.planewave_velocity(Nx, Ny, dx, workloads.SEED0 + 40, amplitude=base_amp, nmodes=12)
    s = ttsh.Solver(Nx, Ny, dx, dt, ttsh.baseline_params(), dtype, mask=mask)
    o = TTSHOracle(Nx, Ny, dx, dt, BASELINE_PRESET, mask=mask, transform=transform)
    if dtype == "f32":
        v0 = tuple(a.astype(np.float32).astype(np.float64) for a in v0)
    s.set_velocity(*v0); o.set_velocity(*v0)
    tg, to = ttsh.Tangent(s, nvec), TangentOracle(o, nvec)
    for i in range(nvec):
        d = workloads.planewave_velocity(Nx, Ny, dx, workloads.SEED0 + 50 + i, amplitude=0.5 + 0.25 * i, nmodes=8)
        d = (d[0] + 0.1 * (i + 1), d[1] - 0.05 * i)          # with a mean-flow component
        if dtype == "f32":
            d = tuple(a.astype(np.float32).astype(np.float64) for a in d)
        tg.set(i, *d); to.set(i, *d)
    return s, o, tg, to


MAXABS_FACTOR = 10.0   # max|a - b| <= MAXABS_FACTOR * tol * max|b| (tests/test_gpu_parity.py)


def compare_vectors(tg, to, tol, what):
    for i in range(to.nvec):
        g = [t.cpu().numpy().astype(np.float64) for t in tg.get_fields(i)]
        r = to.get_fields(i)
        ev, ew = rel(np.stack(g[:2]), np.stack(r[:2])), rel(g[2], r[2])
        assert ev <= tol and ew <= tol, f"{what}: vector {i}: dv {ev:.3e} dw {ew:.3e} > {tol:g}"
        # pointwise bound beside the norm, as compare_state of test_gpu_parity.py: a few wrong points cannot hide in the L2 norm
        mv = np.max(np.abs(np.stack(g[:2]) - np.stack(r[:2]))) / np.max(np.abs(np.stack(r[:2])))
        mw = np.max(np.abs(g[2] - r[2])) / np.max(np.abs(r[2]))
        assert mv <= MAXABS_FACTOR * tol and mw <= MAXABS_FACTOR * tol, f"{what}: vector {i}: max dv {mv:.3e} dw {mw:.3e} > {MAXABS_FACTOR * tol:g}"


@pytest.mark.parametrize("Nx,Ny", [(64, 64), (128, 64), (64, 256)])
def test_tangent_steps_match_oracle(ttsh, Nx, Ny):
    s, o, tg, to = setup(ttsh, Nx, Ny, 3)
    compare_vectors(tg, to, TOL_1, "after set")
    tg.step(1); to.step(1)
    compare_vectors(tg, to, TOL_1, "1 step")
    tg.step(19); to.step(19)
    compare_vectors(tg, to, TOL_N, "20 steps")
    # the base trajectory advanced by the same 20 steps
    gv = [t.cpu().numpy() for t in s.get_fields()]
    ov = o.get_fields()
    assert rel(np.stack(gv[:2]), np.stack(ov[:2])) <= TOL_N and s.diagnostics()["step"] == 20
    tg.close(); s.close()


def test_tangent_at_the_size_bench_times(ttsh):
    """256 x 256 with 8 vectors (the configuration bench.py's Lyapunov line times), 1 and 20 steps, then one QR."""
    s, o, tg, to = setup(ttsh, 256, 256, 8, R=30.0)
    tg.step(1); to.step(1)
    compare_vectors(tg, to, TOL_1, "256^2 1 step")
    tg.step(19); to.step(19)
    compare_vectors(tg, to, TOL_N, "256^2 20 steps")
    lg, lo = np.asarray(tg.orthonormalize()), to.orthonormalize()
    assert np.allclose(lg, lo, rtol=0, atol=1e-9), lg - lo
    compare_vectors(tg, to, 1e-8, "256^2 after QR")
    tg.close(); s.close()


def test_tangent_at_1024_with_4_vectors(ttsh):
    """1024 x 1024 with 4 vectors (the other size DESIGN.md quotes): the fused tangent row kernel with one row pair per CTA, 1 and 5
    steps and one QR against the oracle with its FFT backend (locked to the matrix backend by the CPU pins)."""
    s, o, tg, to = setup(ttsh, 1024, 1024, 4, R=160.0, transform="fft")
    tg.step(1); to.step(1)
    compare_vectors(tg, to, TOL_1, "1024^2 1 step")
    tg.step(4); to.step(4)
    compare_vectors(tg, to, TOL_N, "1024^2 5 steps")
    lg, lo = np.asarray(tg.orthonormalize()), to.orthonormalize()
    assert np.allclose(lg, lo, rtol=0, atol=1e-9), lg - lo
    tg.close(); s.close()


def test_qr_growth_rates_match_oracle(ttsh):
    """Three cycles of (5 tangent steps, QR): log R_ii and the re-orthonormalised vectors agree with the oracle's
    numpy.linalg.qr (the device runs modified Gram-Schmidt: same R up to rounding for well-conditioned vectors)."""
    Nx = Ny = 64
    s, o, tg, to = setup(ttsh, Nx, Ny, 4)
    lg, lo = tg.orthonormalize(), to.orthonormalize()
    assert np.allclose(lg, lo, rtol=0, atol=1e-10)
    compare_vectors(tg, to, 1e-10, "after first QR")
    acc_g, acc_o = np.zeros(4), np.zeros(4)
    for cyc in range(3):
        tg.step(5); to.step(5)
        lg, lo = np.asarray(tg.orthonormalize()), to.orthonormalize()
        assert np.allclose(lg, lo, rtol=0, atol=1e-9), (cyc, lg - lo)
        acc_g += lg; acc_o += lo
    compare_vectors(tg, to, 1e-8, "after 3 cycles")
    # the vectors the device holds are orthonormal in the documented inner product
    P = Nx * Ny
    cols = []
    for i in range(4):
        dvx, dvy, dw = [t.cpu().numpy() for t in tg.get_fields(i)]
        cols.append(np.concatenate([dw.ravel(), [dvx.sum() / np.sqrt(P), dvy.sum() / np.sqrt(P)]]))
    A = np.stack(cols, axis=1)
    assert np.allclose(A.T @ A, np.eye(4), atol=1e-10)
    lam_g, lam_o = acc_g / (15 * 0.01), acc_o / (15 * 0.01)
    assert np.allclose(lam_g, lam_o, atol=1e-6)
    tg.close(); s.close()


@pytest.mark.parametrize("eps,tol", [(1e-4, 1e-9), (1e-8, 1e-6)])
def test_qr_of_nearly_parallel_vectors(ttsh, eps, tol):
    """An ill-conditioned set: vector 1 = vector 0 + eps * (something else).  eps = 1e-4 (cond ~ 1e4) goes through the blocked
    CholeskyQR2; eps = 1e-8 trips its pivot test and falls back to modified Gram-Schmidt on the device.  log R_ii against
    numpy's Householder QR (the oracle), where Gram-Schmidt and Householder differ most."""
    Nx = Ny = 64
    dx, dt = 0.5, 0.01
    s = ttsh.Solver(Nx, Ny, dx, dt, ttsh.baseline_params(), "f64")
    o = TTSHOracle(Nx, Ny, dx, dt, BASELINE_PRESET)
    z = np.zeros((Ny, Nx))
    s.set_velocity(z, z); o.set_velocity(z, z)
    tg, to = ttsh.Tangent(s, 3), TangentOracle(o, 3)
    a = workloads.planewave_velocity(Nx, Ny, dx, 3, amplitude=1.0, nmodes=6)
    b = workloads.planewave_velocity(Nx, Ny, dx, 4, amplitude=1.0, nmodes=6)
    c = workloads.planewave_velocity(Nx, Ny, dx, 5, amplitude=0.5, nmodes=6)
    vecs = [a, (a[0] + eps * b[0], a[1] + eps * b[1]), (c[0] + 0.3, c[1])]
    for i, v in enumerate(vecs):
        tg.set(i, *v); to.set(i, *v)
    lg, lo = np.asarray(tg.orthonormalize()), to.orthonormalize()
    assert np.allclose(lg, lo, rtol=0, atol=tol), lg - lo
    assert lo[1] - lo[0] < np.log(eps) + 2.0               # R_11 / R_00 really is of order eps
    # the device's vectors are orthonormal afterwards
    P = Nx * Ny
    cols = []
    for i in range(3):
        dvx, dvy, dw = [t.cpu().numpy() for t in tg.get_fields(i)]
        cols.append(np.concatenate([dw.ravel(), [dvx.sum() / np.sqrt(P), dvy.sum() / np.sqrt(P)]]))
    A = np.stack(cols, axis=1)
    assert np.allclose(A.T @ A, np.eye(3), atol=1e-6 if eps < 1e-6 else 1e-10)   # one pass of Gram-Schmidt loses eps_mach * cond
    tg.close(); s.close()


def test_growth_about_the_zero_state_is_sigma_of_k(ttsh):
    """Base state 0, no mask: the tangent map is exp(sigma(k) dt) per mode (Alg. 1 line 4): closed form on the GPU too."""
    Nx = Ny = 64
    dx, dt, n = 0.5, 0.01, 12
    s = ttsh.Solver(Nx, Ny, dx, dt, ttsh.baseline_params(), "f64")
    z = np.zeros((Ny, Nx))
    s.set_velocity(z, z)
    x = np.arange(Nx)[None, :] * dx
    y = np.arange(Ny)[:, None] * dx
    p = BASELINE_PRESET
    modes = [(3, 2), (1, -4)]
    tg = ttsh.Tangent(s, 3)
    sig = []
    for i, (mx, my) in enumerate(modes):
        kx, ky = 2 * np.pi * mx / (Nx * dx), 2 * np.pi * my / (Ny * dx)
        ph = kx * x + ky * y
        tg.set(i, ky * np.cos(ph), -kx * np.cos(ph))
        k2 = kx * kx + ky * ky
        sig.append(-p.alpha - p.Gamma0 * k2 - p.Gamma2 * k2 * k2)
    tg.set(2, np.ones((Ny, Nx)), z)                  # pure mean flow: exp(-alpha dt)
    sig.append(-p.alpha)
    tg.orthonormalize()
    tg.step(n)
    logr = np.asarray(tg.orthonormalize())
    assert np.allclose(logr / (n * dt), sig, rtol=0, atol=1e-10), logr / (n * dt) - np.asarray(sig)
    tg.close(); s.close()


def test_tangent_fp32_and_argument_validation(ttsh):
    s, o, tg, to = setup(ttsh, 128, 64, 2, dtype="f32")
    tg.step(1); to.step(1)
    compare_vectors(tg, to, 1e-5, "fp32 1 step")
    lg, lo = tg.orthonormalize(), to.orthonormalize()
    assert np.allclose(lg, lo, atol=1e-5)
    INV = ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_tangent_step(tg.s, -1) == INV
    assert ttsh.ttsh_tangent_set(tg.s, 2, 1, 1) == INV and ttsh.ttsh_tangent_set(tg.s, 0, 0, 0) == INV
    assert ttsh.ttsh_tangent_get_fields(tg.s, 5) == INV
    s2 = ttsh.Solver(64, 64, 0.5, 0.01, ttsh.baseline_params(), "f64")
    t2 = ttsh.Tangent(s2, 2)
    assert ttsh.ttsh_tangent_step(t2.s, 1) == ttsh.TTSH_ERR_NOT_INITIALIZED        # handle has no state
    z = np.zeros((64, 64))
    s2.set_velocity(z, z)
    assert ttsh.ttsh_tangent_step(t2.s, 1) == ttsh.TTSH_ERR_NOT_INITIALIZED        # vectors not set
    assert ttsh.ttsh_tangent_orthonormalize(t2.s, 2)[0] == ttsh.TTSH_ERR_NOT_INITIALIZED
    s2.set_advection_form(ttsh.TTSH_ADVECTION_LITERAL)
    t2.set(0, z + 1.0, z); t2.set(1, z, z + 1.0)
    assert ttsh.ttsh_tangent_step(t2.s, 1) == INV                                  # conservative form only
    t2.close(); s2.close(); tg.close(); s.close()
