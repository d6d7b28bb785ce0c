"""ttsh_diagnostics_noalloc against ttsh_diagnostics (GPU).

Why the entry point exists: everything else in the library needs a workspace that the caller allocates.  A caller that
only receives pointers to v_x, v_y, omega (a hook inside somebody else's time loop), or that runs where a raw cudaMalloc
fails (the framework's allocator holds all device memory) or is too costly (it synchronises the whole device), has no
workspace to give.  For them the reduction's scratch is a static array inside the library, shared by every call on a GPU
(include/ttsh.h).  What this file checks is what such a caller relies on:

  * the numbers are those of the handle-based ttsh_diagnostics on the same fields, within the tolerance the diagnostics
    parity tests use (1e-10 relative on the raw sums, reading R13 of DESIGN.md);
  * that holds for two calls in a row, the second on a different state, and for a small fp32 grid right after a larger
    fp64 one: whatever the earlier call left in the static array must not reach the later result;
  * the call really allocates no device memory; sizes beyond the stated maximum are refused with a message.

This file is named test_zz_* so that pytest collects it last (`pytest --collect-only -q tests`): under `-x` a failure here
cannot hide another test.  It passes in a fresh process on its own and after the rest of the suite: the per-device set-up
(looking up the static array's address) happens inside the first call, whenever that is."""
import ctypes as C

import pytest

from paper_2304_03306_b200 import workloads

pytestmark = pytest.mark.gpu

TOL_DIAG = 1e-10     # tests/test_gpu_parity.py


@pytest.fixture(scope="module")
def ttsh():
    import __graft_entry__ as ge
    ge.build()
    from paper_2304_03306_b200 import ttsh as t
    return t


def noalloc_diag(ttsh, s, fields, sums, cx, cy):
    """One call of the entry point on the solver's stream; fields = (vx, vy, omega) device tensors."""
    vx, vy, w = fields
    with s._ctx():
        rc, d = ttsh.ttsh_diagnostics_noalloc(s.Nx, s.Ny, s.dx, s.dtype_code, vx.data_ptr(), vy.data_ptr(), w.data_ptr(),
                                              cx, cy, sums.data_ptr(), s.stream.cuda_stream)
    assert rc == ttsh.TTSH_OK, ttsh.ttsh_diagnostics_noalloc_error()
    return d.as_dict()


def assert_same_diagnostics(d, ref, Nx, Ny, what):
    for key in ("sum_speed", "sum_abs_vtheta", "kinetic_energy", "enstrophy", "max_speed"):
        assert abs(d[key] - ref[key]) <= TOL_DIAG * abs(ref[key]), (what, key, d[key], ref[key])
    for key in ("mean_vx", "mean_vy"):
        assert abs(d[key] - ref[key]) * Nx * Ny <= TOL_DIAG * ref["sum_speed"], (what, key, d[key], ref[key])
    for key in ("vortex_order", "polar_order"):
        assert abs(d[key] - ref[key]) <= TOL_DIAG, (what, key, d[key], ref[key])
    assert d["nonfinite"] == ref["nonfinite"], what


def make_solver(ttsh, Nx, Ny, dtype, nsteps):
    dx = 0.5
    mask = workloads.disk_mask(Nx, Ny, dx, 0.3 * min(Nx, Ny) * dx)
    vel = workloads.planewave_velocity(Nx, Ny, dx, workloads.SEED0, amplitude=1.0)      # O(1) field: every sum is far from 0
    s = ttsh.Solver(Nx, Ny, dx, 0.01, ttsh.baseline_params(), dtype, mask=mask)
    s.set_velocity(*vel)
    s.step(nsteps)
    return s


def test_noalloc_diagnostics_match_the_handle_path_on_two_calls_in_a_row(ttsh):
    import torch
    Nx, Ny = 512, 256                       # 131072 points = 512 chunks of 256 threads: 80 of the 592 blocks find no work at all
    s = make_solver(ttsh, Nx, Ny, "f64", 3)
    cx, cy = 0.37 * Nx * s.dx, 0.61 * Ny * s.dx          # off-centre, off-grid: e_theta has no symmetry to hide behind
    with s._ctx():
        sums = torch.empty(8, dtype=torch.float64, device=s.device)

    # first call (on a fresh process this is also the one that does the per-device set-up)
    vx, vy, w, _ = s.get_fields(psi=False)
    ref1 = s.diagnostics(cx, cy)
    d1 = noalloc_diag(ttsh, s, (vx, vy, w), sums, cx, cy)
    assert_same_diagnostics(d1, ref1, Nx, Ny, "first call")
    raw1 = sums.cpu().numpy().copy()
    assert raw1[2] == d1["sum_speed"] and raw1[6] == d1["max_speed"] and raw1[0] == 2.0 * Nx * Ny * d1["kinetic_energy"]

    # second call straight after it, on another state: the array still holds the first call's records when it starts
    s.step(7)
    vx2, vy2, w2, _ = s.get_fields(psi=False)
    ref2 = s.diagnostics(cx, cy)
    free_before = torch.cuda.mem_get_info(s.device)[0]
    d2 = noalloc_diag(ttsh, s, (vx2, vy2, w2), sums, cx, cy)
    free_after = torch.cuda.mem_get_info(s.device)[0]
    assert_same_diagnostics(d2, ref2, Nx, Ny, "second call")
    assert d2["sum_speed"] != d1["sum_speed"]            # the states differ, so a stale result would show
    assert free_after == free_before, "the call changed the amount of free device memory"

    # the first state again: same input, same bits, whatever ran in between
    d1b = noalloc_diag(ttsh, s, (vx, vy, w), sums, cx, cy)
    assert d1b == d1
    s.close()


def test_noalloc_small_fp32_grid_right_after_a_larger_one(ttsh):
    """64 x 64 in fp32 gives work to 16 of the 592 blocks; the other records were last written by the larger grid of the
    call before and must come out as zeros, not as leftovers.  Also counts non-finite values like the handle path."""
    import torch
    big = make_solver(ttsh, 512, 256, "f64", 1)
    with big._ctx():
        sums = torch.empty(8, dtype=torch.float64, device=big.device)
    vx, vy, w, _ = big.get_fields(psi=False)
    cxb, cyb = 128 * big.dx, 64 * big.dx
    assert_same_diagnostics(noalloc_diag(ttsh, big, (vx, vy, w), sums, cxb, cyb), big.diagnostics(cxb, cyb), 512, 256, "512 x 256")

    small = make_solver(ttsh, 64, 64, "f32", 2)
    vx, vy, w, _ = small.get_fields(psi=False)
    cx, cy = 32 * small.dx, 32 * small.dx
    with small._ctx():
        small.stream.wait_stream(big.stream)             # the two solvers own different streams: keep the calls apart on the GPU
    d = noalloc_diag(ttsh, small, (vx, vy, w), sums, cx, cy)
    assert_same_diagnostics(d, small.diagnostics(cx, cy), 64, 64, "64 x 64 fp32 after 512 x 256")

    with small._ctx():
        vx[5, 7] = float("nan"); vy[0, 0] = float("inf"); w[63, 63] = float("-inf")
    assert noalloc_diag(ttsh, small, (vx, vy, w), sums, cx, cy)["nonfinite"] == 3
    big.close(); small.close()


def test_noalloc_asynchronous_form_and_argument_checks(ttsh):
    import torch
    s = make_solver(ttsh, 128, 64, "f64", 1)
    vx, vy, w, _ = s.get_fields(psi=False)
    cx, cy = 64 * s.dx, 32 * s.dx
    ref = s.diagnostics(cx, cy)
    with s._ctx():
        sums = torch.full((8,), -1.0, dtype=torch.float64, device=s.device)
        rc, d = ttsh.ttsh_diagnostics_noalloc(128, 64, s.dx, s.dtype_code, vx.data_ptr(), vy.data_ptr(), w.data_ptr(), cx, cy,
                                              sums.data_ptr(), s.stream.cuda_stream, read_back=False)
        assert rc == ttsh.TTSH_OK and d is None
        raw = sums.cpu().numpy()                         # stream-ordered copy on the same stream
    assert abs(raw[2] - ref["sum_speed"]) <= TOL_DIAG * ref["sum_speed"]
    assert abs(raw[0] - 2 * 128 * 64 * ref["kinetic_energy"]) <= TOL_DIAG * raw[0] and raw[7] == 0.0

    args = dict(Nx=128, Ny=64, dx=s.dx, dtype=s.dtype_code, vx_ptr=vx.data_ptr(), vy_ptr=vy.data_ptr(), omega_ptr=w.data_ptr(),
                cx=cx, cy=cy, sums_ptr=sums.data_ptr(), stream_ptr=s.stream.cuda_stream)
    with s._ctx():
        rc, _ = ttsh.ttsh_diagnostics_noalloc(**{**args, "Nx": 16385})
        assert rc == ttsh.TTSH_ERR_UNSUPPORTED_SIZE
        msg = ttsh.ttsh_diagnostics_noalloc_error()
        assert "16385" in msg and "maximum" in msg and str(ttsh.TTSH_NOALLOC_MAX_POINTS) in msg
        for bad in ({"Ny": 0}, {"dx": 0.0}, {"dtype": 2}, {"vx_ptr": 0}, {"sums_ptr": 0}, {"cx": float("nan")}):
            rc, _ = ttsh.ttsh_diagnostics_noalloc(**{**args, **bad})
            assert rc == ttsh.TTSH_ERR_INVALID_ARG and ttsh.ttsh_diagnostics_noalloc_error() != "", bad
        rc, _ = ttsh.ttsh_diagnostics_noalloc(**args)
        assert rc == ttsh.TTSH_OK and ttsh.ttsh_diagnostics_noalloc_error() == ""
    assert C.sizeof(ttsh.ttsh_diag) == 12 * 8
    s.close()
