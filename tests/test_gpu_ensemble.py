"""GPU parity of ttsh_ensemble_step (the paper's sweeps of independent runs).

Every member of an ensemble must compute exactly what ttsh_step computes for it: bit-identical fields, and the same
tolerances against the CPU oracle as the single-system path (fp64 1e-12 after 1 step, 1e-9 after 100)."""
import numpy as np
import pytest

from oracle import BASELINE_PRESET, TTSHOracle
from oracle.ttsh_oracle import process_mask
from paper_2304_03306_b200 import workloads

pytestmark = pytest.mark.gpu

TOL_F64_1, TOL_F64_100, TOL_F32_1 = 1e-12, 1e-9, 1e-5


@pytest.fixture(scope="module")
def ttsh():
    import __graft_entry__ as ge
    ge.build()
    from paper_2304_03306_b200 import ttsh as t
    return t


def rel(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def fields(s):
    return [t.cpu().numpy() for t in s.get_fields()]


def sweep_inputs(Nx, Ny, dx, radii, o1_members=()):
    """An R sweep on one grid: disk masks of growing radius, one seed per member; members listed in o1_members start from
    an O(1) plane-wave field (reading R17) so that the nonlinear terms matter within a few steps."""
    masks, vels = [], []
    for i, R in enumerate(radii):
        m = workloads.disk_mask(Nx, Ny, dx, R)
        masks.append(m)
        if i in o1_members:
            vels.append(workloads.planewave_velocity(Nx, Ny, dx, workloads.SEED0 + 100 + i, amplitude=1.0))
        else:
            vels.append(workloads.gaussian_velocity(Nx, Ny, workloads.SEED0 + 100 + i, 1e-2, m))
    return masks, vels


@pytest.mark.parametrize("Nx,Ny,count,nsteps", [(64, 64, 5, 100), (128, 256, 3, 20), (512, 64, 2, 20)])
def test_ensemble_members_match_oracle_and_single_handles(ttsh, Nx, Ny, count, nsteps):
    dx, dt = 0.5, 0.01
    radii = [0.12 * min(Nx, Ny) * dx * (1 + 0.4 * i) for i in range(count)]
    masks, vels = sweep_inputs(Nx, Ny, dx, radii, o1_members=(1,))
    ens = ttsh.Ensemble(count, Nx, Ny, dx, dt, ttsh.baseline_params(), "f64", masks=masks)
    singles = [ttsh.Solver(Nx, Ny, dx, dt, ttsh.baseline_params(), "f64", mask=masks[i]) for i in range(count)]
    oracles = [TTSHOracle(Nx, Ny, dx, dt, BASELINE_PRESET, mask=masks[i]) for i in range(count)]
    for i in range(count):
        ens.members[i].set_velocity(*vels[i]); singles[i].set_velocity(*vels[i]); oracles[i].set_velocity(*vels[i])
    l0 = ens.launch_count()
    ens.step(1)                       # direct launches
    # Ny = 64: the four hot kernels, one launch each for the whole ensemble; 128 <= Ny <= 1024: k_inv_col (the intermediates are not
    # at hand yet) + k_row_step + k_col_step
    assert ens.launch_count() - l0 == (4 if Ny == 64 else 3)
    for i in range(count):
        singles[i].step(1); oracles[i].step(1)
    for i in range(count):
        g, s1, o = fields(ens.members[i]), fields(singles[i]), oracles[i].get_fields()
        for a, b in zip(g, s1):
            assert np.array_equal(a, b), f"member {i}: ensemble step differs from ttsh_step"
        assert rel(np.stack(g[:2]), np.stack(o[:2])) <= TOL_F64_1 and rel(g[2], o[2]) <= TOL_F64_1 and rel(g[3], o[3]) <= TOL_F64_1
    ens.step(nsteps - 1)              # CUDA-graph replay
    for i in range(count):
        singles[i].step(nsteps - 1); oracles[i].step(nsteps - 1)
    for i in range(count):
        g, s1, o = fields(ens.members[i]), fields(singles[i]), oracles[i].get_fields()
        for a, b in zip(g, s1):
            assert np.array_equal(a, b), f"member {i}: ensemble differs from ttsh_step after {nsteps} steps"
        assert rel(np.stack(g[:2]), np.stack(o[:2])) <= TOL_F64_100 and rel(g[2], o[2]) <= TOL_F64_100
        d, od = ens.members[i].diagnostics(), oracles[i].diagnostics((Nx // 2) * dx, (Ny // 2) * dx)
        assert d["step"] == nsteps and abs(d["t"] - nsteps * dt) < 1e-12
        assert abs(d["kinetic_energy"] - od["kinetic_energy"]) <= 1e-9 * od["kinetic_energy"]
    ens.close()
    for s in singles:
        s.close()


@pytest.mark.parametrize("dtype,Nx,Ny,count", [("f32", 256, 128, 4), ("f64", 1024, 1024, 2), ("f32", 2048, 256, 2), ("f64", 8192, 64, 2),
                                               ("f32", 8192, 64, 2), ("f64", 4096, 64, 3), ("f32", 16384, 64, 2)])
def test_ensemble_bit_identical_to_single_handles_larger_grids(ttsh, dtype, Nx, Ny, count):
    dx, dt = 0.5, 0.01
    radii = [0.1 * min(Nx, Ny) * dx * (1 + 0.5 * i) for i in range(count)]
    masks, vels = sweep_inputs(Nx, Ny, dx, radii, o1_members=(0,))
    ens = ttsh.Ensemble(count, Nx, Ny, dx, dt, ttsh.baseline_params(), dtype, masks=masks)
    singles = [ttsh.Solver(Nx, Ny, dx, dt, ttsh.baseline_params(), dtype, mask=masks[i]) for i in range(count)]
    for i in range(count):
        ens.members[i].set_velocity(*vels[i]); singles[i].set_velocity(*vels[i])
    for n in (3, 5):                  # direct launches, then graph replay
        ens.step(n)
        for s in singles:
            s.step(n)
        for i in range(count):
            for a, b in zip(fields(ens.members[i]), fields(singles[i])):
                assert np.array_equal(a, b), f"member {i} after +{n} steps"
    # one member against the oracle (single step from the evolved state would need the oracle's state: restart instead)
    o = TTSHOracle(Nx, Ny, dx, dt, BASELINE_PRESET, mask=masks[0], transform="fft" if Nx * Ny > 512 * 512 else "matmul")
    v = vels[0]
    if dtype == "f32":
        v = tuple(a.astype(np.float32).astype(np.float64) for a in v)
    ens.members[0].set_velocity(*v); o.set_velocity(*v)
    for i in range(1, count):
        ens.members[i].set_velocity(*vels[i])
    ens.step(1); o.step(1)
    g, of = fields(ens.members[0]), o.get_fields()
    tol = TOL_F64_1 if dtype == "f64" else TOL_F32_1
    assert rel(np.stack(g[:2]), np.stack(of[:2])) <= tol and rel(g[2], of[2]) <= tol
    ens.close()
    for s in singles:
        s.close()


def test_ensemble_hysteresis_ramp_with_live_mask_change(ttsh):
    """The hysteresis protocol: R is ramped on live systems, the state carried over.  Here every member of a
    sweep gets a new mask between ensemble steps; members keep matching the oracle driven the same way."""
    Nx = Ny = 64
    dx, dt = 0.5, 0.01
    radii = [8.0, 10.0, 12.0]
    masks, vels = sweep_inputs(Nx, Ny, dx, radii, o1_members=(0, 1, 2))
    ens = ttsh.Ensemble(3, Nx, Ny, dx, dt, ttsh.baseline_params(), "f64", masks=masks)
    oracles = [TTSHOracle(Nx, Ny, dx, dt, BASELINE_PRESET, mask=masks[i]) for i in range(3)]
    for i in range(3):
        ens.members[i].set_velocity(*vels[i]); oracles[i].set_velocity(*vels[i])
    for ramp in range(3):
        ens.step(10)
        for i in range(3):
            oracles[i].step(10)
            newmask = workloads.disk_mask(Nx, Ny, dx, radii[i] + 0.5 * (ramp + 1))
            ens.members[i].set_mask(newmask)
            oracles[i].K = process_mask(newmask != 0)       # Algorithm 2 on the new mask; state carried over
    ens.step(10)
    for i in range(3):
        oracles[i].step(10)
        g, of = fields(ens.members[i]), oracles[i].get_fields()
        assert rel(np.stack(g[:2]), np.stack(of[:2])) <= TOL_F64_100 and rel(g[2], of[2]) <= TOL_F64_100
        assert ens.members[i].diagnostics()["step"] == 40
    ens.close()


def test_ensemble_argument_validation(ttsh):
    import torch
    p = ttsh.baseline_params()
    a = ttsh.Solver(64, 64, 0.5, 0.01, p, "f64")
    b = ttsh.Solver(64, 64, 0.5, 0.01, p, "f64")          # separate allocation: still a uniform stride for 2 members ...
    c = ttsh.Solver(128, 64, 0.5, 0.01, p, "f64")
    d32 = ttsh.Solver(64, 64, 0.5, 0.01, p, "f32")
    other = ttsh.Solver(64, 64, 0.5, 0.02, p, "f64")
    INV = ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_ensemble_create([])[0] == INV
    assert ttsh.ttsh_ensemble_create([a.h, None])[0] == INV
    assert ttsh.ttsh_ensemble_create([a.h, a.h])[0] == INV                      # the same member twice
    assert ttsh.ttsh_ensemble_create([a.h, c.h])[0] == INV                      # different grid
    assert ttsh.ttsh_ensemble_create([a.h, d32.h])[0] == INV                    # different dtype
    assert ttsh.ttsh_ensemble_create([a.h, other.h])[0] == INV                  # different dt
    ens3 = ttsh.Ensemble(3, 64, 64, 0.5, 0.01, p, "f64")
    hs = [m.h for m in ens3.members]
    assert ttsh.ttsh_ensemble_create([hs[0], hs[2], hs[1]])[0] == INV           # non-uniform workspace stride
    assert ttsh.ttsh_ensemble_create([hs[1], hs[0]])[0] == INV                  # negative stride
    rc, e = ttsh.ttsh_ensemble_create(hs[:2])
    assert rc == ttsh.TTSH_OK
    assert ttsh.ttsh_ensemble_step(e, -1) == INV
    assert ttsh.ttsh_ensemble_step(e, 3) == ttsh.TTSH_ERR_NOT_INITIALIZED       # no member has a state yet
    z = np.zeros((64, 64))
    ens3.members[0].set_velocity(z, z)
    assert ttsh.ttsh_ensemble_step(e, 3) == ttsh.TTSH_ERR_NOT_INITIALIZED       # member 1 still has none
    ens3.members[1].set_velocity(z, z)
    assert ttsh.ttsh_ensemble_step(e, 0) == ttsh.TTSH_OK and ttsh.ttsh_ensemble_step(e, 3) == ttsh.TTSH_OK
    ens3.members[0].set_advection_form(ttsh.TTSH_ADVECTION_LITERAL)
    assert ttsh.ttsh_ensemble_step(e, 1) == INV                                 # the fused step is conservative-form only
    torch.cuda.synchronize()
    assert ttsh.ttsh_ensemble_destroy(e) == ttsh.TTSH_OK and ttsh.ttsh_ensemble_destroy(None) == ttsh.TTSH_OK
    ens3.close()
    for s in (a, b, c, d32, other):
        s.close()


def test_C3_radius_sweep_and_C4_separation_sweep_as_ensembles_10000_steps(ttsh):
    """BASELINE.json configs[2] and [3] as they are stated: the disk-radius sweep R in {40, 80, 160, 240} at 1024^2 and the
    dumbbell separation sweep d in {80, 100, 110, 118} at 1024 x 2048, 10,000 steps each — run as 4-member ensembles.  No
    oracle can follow that far (chaos): finite fields, saturated energies, the confined kinetic energy grows with the
    unmasked area, member 0 stays bit-identical to the same system stepped alone for the first 200 steps, and Psi_2 of every
    dumbbell is a valid order parameter."""
    p = ttsh.baseline_params()
    for name in ("C3", "C4"):
        cfg = workloads.CONFIGS[name]
        sweep = cfg.sweep
        masks = [cfg.mask(R=r) if name == "C3" else cfg.mask(d=r) for r in sweep]
        vels = [workloads.gaussian_velocity(cfg.Nx, cfg.Ny, cfg.seed + 10 * i, 1e-2, masks[i]) for i in range(len(sweep))]
        ens = ttsh.Ensemble(len(sweep), cfg.Nx, cfg.Ny, cfg.dx, cfg.dt, p, "f64", masks=masks)
        alone = ttsh.Solver(cfg.Nx, cfg.Ny, cfg.dx, cfg.dt, p, "f64", mask=masks[0])
        for i, m in enumerate(ens.members):
            m.set_velocity(*vels[i])
        alone.set_velocity(*vels[0])
        ens.step(200); alone.step(200)
        for a, b in zip(fields(ens.members[0]), fields(alone)):
            assert np.array_equal(a, b)
        alone.close()
        for _ in range((cfg.steps - 200) // 1400):
            ens.step(1400)
            for m in ens.members:
                d = m.diagnostics()
                assert d["nonfinite"] == 0 and np.isfinite(d["kinetic_energy"])
        diags = [m.diagnostics() for m in ens.members]
        assert all(d["step"] == cfg.steps for d in diags)
        E = [d["kinetic_energy"] for d in diags]
        assert all(1e-4 < e < 1.0 for e in E) and all(d["max_speed"] < 5.0 for d in diags)
        if name == "C3":
            assert E[0] < E[1] < E[2] < E[3]              # energy per unit box area follows the unmasked area (R^2)
        else:
            for i, m in enumerate(ens.members):
                dsep = sweep[i]
                cl = ((cfg.Nx // 2) * cfg.dx - dsep / 2, (cfg.Ny // 2) * cfg.dx)
                cr = ((cfg.Nx // 2) * cfg.dx + dsep / 2, (cfg.Ny // 2) * cfg.dx)
                o = m.dumbbell_order(cl, cr, dsep / 2)
                assert 0.0 <= o["psi2"] <= 1.0 and o["index_left"] >= 0 and o["index_right"] >= 0
                assert abs(o["omega_left"]) > 0 and abs(o["omega_right"]) > 0
        ens.close()
