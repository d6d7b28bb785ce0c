"""One small run of every kernel family ("the smem FFT kernels are the race risk"), collected as a `gpu` test:

3 steps of C1 (64 x 64 fp64, the CUDA-graph-free path), 3 steps of a 256 x 128 fp32 system (both advection forms), a 2-member
ensemble, a 2-vector tangent step with one QR, one PSD accumulation, the dumbbell order parameter, get_fields and diagnostics,
and one step at 4096 x 64 (the warp-local row plan with asynchronous bulk copies).  The test asserts that every number that comes
back is finite and that a second run gives the same numbers bit for bit (a race in a shared-memory exchange would show as a
run-to-run difference).  `python tests/test_gpu_all_kernels_smoke.py` runs the same thing stand-alone and prints the checksums:
that is the command to put under compute-sanitizer (one tool per run) on a pool where the tool is open (this one refuses it)."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2304_03306_b200 import ttsh, workloads  # noqa: E402


def main():
    out = []
    cfg = workloads.CONFIGS["C1"]
    mask = cfg.mask()
    s = ttsh.Solver(cfg.Nx, cfg.Ny, cfg.dx, cfg.dt, ttsh.baseline_params(), "f64", mask=mask)
    s.set_velocity(*cfg.initial_velocity(mask, amplitude=1.0))
    s.step(3)
    out.append(float(s.get_fields()[2].abs().sum()))
    tg = ttsh.Tangent(s, 2)
    for i in range(2):
        tg.set(i, *workloads.gaussian_velocity(cfg.Nx, cfg.Ny, 77 + i, 1.0))
    tg.step(1)
    out.extend(tg.orthonormalize())
    psd = ttsh.TemporalPSD(s, [0.0, 0.5, 1.0])
    psd.accumulate()
    out.extend(psd.result()[0])
    out.append(s.dumbbell_order((12.0, 16.0), (20.0, 16.0), 4.0)["psi2"])
    out.append(s.diagnostics()["kinetic_energy"])
    s.close()

    mask = workloads.dumbbell_mask(256, 128, 0.5, 20.0, 30.0)
    s = ttsh.Solver(256, 128, 0.5, 0.01, ttsh.baseline_params(), "f32", mask=mask)
    s.set_velocity(*workloads.planewave_velocity(256, 128, 0.5, 5, amplitude=1.0))
    s.step(2)
    s.set_advection_form(ttsh.TTSH_ADVECTION_LITERAL)
    s.step(1)
    out.append(s.diagnostics()["enstrophy"])
    s.close()

    masks = [workloads.disk_mask(64, 64, 0.5, r) for r in (10.0, 12.0)]
    ens = ttsh.Ensemble(2, 64, 64, 0.5, 0.01, ttsh.baseline_params(), "f64", masks=masks)
    for i, m in enumerate(ens.members):
        m.set_velocity(*workloads.gaussian_velocity(64, 64, 5 + i, 1e-2, masks[i]))
    ens.step(3)
    out.append(ens.members[1].diagnostics()["kinetic_energy"])
    ens.close()

    mask = workloads.disk_mask(4096, 64, 0.5, 12.0)
    s = ttsh.Solver(4096, 64, 0.5, 0.01, ttsh.baseline_params(), "f64", mask=mask)
    s.set_velocity(*workloads.planewave_velocity(4096, 64, 0.5, 6, amplitude=1.0))
    s.step(1)
    out.append(s.diagnostics()["kinetic_energy"])
    s.close()
    assert all(np.isfinite(out)), out
    return out


@pytest.mark.gpu
def test_every_kernel_family_runs_finite_and_repeats_bit_for_bit():
    first, second = main(), main()
    assert len(first) >= 10 and first == second, (first, second)


if __name__ == "__main__":
    print("all-kernels smoke ok:", " ".join(f"{v:.6e}" for v in main()))
