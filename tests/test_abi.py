"""The C-ABI library loads and exports every symbol include/ttsh.h declares; host-side argument validation.
No compute calls (no GPU needed)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def ttsh():
    import __graft_entry__ as ge
    ge.build()
    from paper_2304_03306_b200 import ttsh as t
    return t


def test_library_exports_every_declared_symbol(ttsh):
    header = open(os.path.join(ROOT, "include", "ttsh.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(ttsh_[a-z_]+)\s*\(", header))
    assert declared == set(ttsh.SYMBOLS)
    lib = C.CDLL(ttsh.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name


def test_library_was_built_from_the_sources_in_the_tree(ttsh):
    _check_build_info(ttsh)


@pytest.mark.gpu
def test_library_on_the_gpu_box_was_built_from_the_sources_in_the_tree(ttsh):
    """The same check inside the `-m gpu` run: the libttsh.so that the parity tests load on the GPU box (it travels with the
    snapshot; build() is an incremental make) is the one compiled from the sources next to it."""
    _check_build_info(ttsh)


def _check_build_info(ttsh):
    """ttsh_build_info carries the SHA-256 of the CUDA sources the binary was compiled from (csrc/Makefile): a stale libttsh.so
    that travelled with the snapshot instead of being rebuilt would show here."""
    import glob
    import hashlib
    csrc = os.path.join(ROOT, "paper_2304_03306_b200", "csrc")
    files = sorted(glob.glob(os.path.join(csrc, "*.cu")) + glob.glob(os.path.join(csrc, "*.cuh")) + glob.glob(os.path.join(csrc, "*.h"))
                   + [os.path.join(csrc, "..", "..", "include", "ttsh.h"), os.path.join(csrc, "Makefile")],
                   key=lambda p: os.path.relpath(p, csrc))
    h = hashlib.sha256()
    for f in files:
        h.update(open(f, "rb").read())
    info = ttsh.ttsh_build_info()
    assert "sm_100a" in info and ("sources=" + h.hexdigest()[:16]) in info, info


def test_struct_layouts_match_the_header(ttsh):
    assert C.sizeof(ttsh.ttsh_params) == 7 * 8 + 2 * 4
    assert C.sizeof(ttsh.ttsh_diag) == 12 * 8


def test_workspace_bytes_and_size_validation(ttsh):
    assert ttsh.ttsh_workspace_bytes(100, 64, ttsh.TTSH_F64) == 0         # not a power of two
    assert ttsh.ttsh_workspace_bytes(32, 64, ttsh.TTSH_F64) == 0          # below 64
    assert ttsh.ttsh_workspace_bytes(64, 32768, ttsh.TTSH_F64) == 0       # above 16384
    assert ttsh.ttsh_workspace_bytes(16384, 64, ttsh.TTSH_F64) > 0 and ttsh.ttsh_workspace_bytes(64, 16384, ttsh.TTSH_F32) > 0
    assert 12 * 2**31 < ttsh.ttsh_workspace_bytes(16384, 16384, ttsh.TTSH_F64) < 15 * 2**31   # Fig. 6(f) grid: about 27 GB of 180 GB
    assert ttsh.ttsh_workspace_bytes(64, 64, 3) == 0                      # bad dtype
    b64 = ttsh.ttsh_workspace_bytes(4096, 4096, ttsh.TTSH_F64)
    b32 = ttsh.ttsh_workspace_bytes(4096, 4096, ttsh.TTSH_F32)
    U = 4096 * 4096 * 8
    assert 6 * U < b64 < 13 * U and 0.45 * b64 < b32 < 0.55 * b64        # 7 real fields + pruned spectra and intermediates (1.7 GB of 180 GB HBM)


def test_create_rejects_bad_arguments_without_touching_cuda(ttsh):
    p = ttsh.baseline_params()
    fake_ws = 256 * 1000   # never dereferenced: all of these fail validation first
    nbytes = ttsh.ttsh_workspace_bytes(64, 64, ttsh.TTSH_F64)
    cases = [
        (dict(Nx=96), ttsh.TTSH_ERR_UNSUPPORTED_SIZE),
        (dict(dx=0.0), ttsh.TTSH_ERR_INVALID_ARG),
        (dict(dt=-1.0), ttsh.TTSH_ERR_INVALID_ARG),
        (dict(ws=0), ttsh.TTSH_ERR_INVALID_ARG),
        (dict(ws=fake_ws + 8), ttsh.TTSH_ERR_INVALID_ARG),          # misaligned
        (dict(nbytes=nbytes - 1), ttsh.TTSH_ERR_WORKSPACE_TOO_SMALL),
        (dict(dtype=5), ttsh.TTSH_ERR_INVALID_ARG),
        (dict(kind=7), ttsh.TTSH_ERR_INVALID_ARG),
    ]
    for kw, want in cases:
        a = dict(Nx=64, Ny=64, dx=0.5, dt=0.01, dtype=ttsh.TTSH_F64, kind=0, ws=fake_ws, nbytes=nbytes)
        a.update(kw)
        rc, h = ttsh.ttsh_create(a["Nx"], a["Ny"], a["dx"], a["dt"], p, a["dtype"], 0, a["kind"], a["ws"], a["nbytes"], 0)
        assert rc == want, (kw, rc)
        assert not h
    for num, den in ((1, 5), (3, 4), (0, 2), (1, 0)):
        q = ttsh.baseline_params(); q.dealias_num, q.dealias_den = num, den
        rc, h = ttsh.ttsh_create(64, 64, 0.5, 0.01, q, ttsh.TTSH_F64, 0, 0, fake_ws, nbytes, 0)
        assert rc == ttsh.TTSH_ERR_INVALID_ARG
    q = ttsh.baseline_params(); q.Gamma2 = -1.0
    rc, h = ttsh.ttsh_create(64, 64, 0.5, 0.01, q, ttsh.TTSH_F64, 0, 0, fake_ws, nbytes, 0)
    assert rc == ttsh.TTSH_ERR_INVALID_ARG
    for field in ("lambda0", "alpha", "beta", "Gamma0", "Gamma2", "gamma_v", "gamma_w"):      # non-finite parameters
        for bad in (float("nan"), float("inf")):
            q = ttsh.baseline_params(); setattr(q, field, bad)
            rc, h = ttsh.ttsh_create(64, 64, 0.5, 0.01, q, ttsh.TTSH_F64, 0, 0, fake_ws, nbytes, 0)
            assert rc == ttsh.TTSH_ERR_INVALID_ARG and not h, (field, bad)
    assert ttsh.ttsh_step(None, 1) == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_destroy(None) == ttsh.TTSH_OK
    assert "workspace" in ttsh.ttsh_strerror(ttsh.TTSH_ERR_WORKSPACE_TOO_SMALL)


def test_product_path_never_imports_the_oracle():
    imp = re.compile(r"^\s*(from|import)\s+oracle\b|import_module\(.oracle|oracle[/.]ttsh_oracle", re.M)
    pkg = os.path.join(ROOT, "paper_2304_03306_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")) or f == "Makefile":
                assert not imp.search(open(os.path.join(dirpath, f)).read()), f
    imp2 = re.compile(r"^\s*(from|import)\s+paper_2304_03306_b200\b|libttsh", re.M)
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith(".py"):
                assert not imp2.search(open(os.path.join(dirpath, f)).read()), f


def test_ensemble_create_rejects_bad_arguments_without_touching_cuda(ttsh):
    assert ttsh.ttsh_ensemble_create([])[0] == ttsh.TTSH_ERR_INVALID_ARG            # count < 1
    assert ttsh.ttsh_ensemble_create([None])[0] == ttsh.TTSH_ERR_INVALID_ARG        # NULL member
    assert ttsh.ttsh_ensemble_step(None, 1) == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_ensemble_destroy(None) == ttsh.TTSH_OK
    assert ttsh.ttsh_ensemble_launch_count(None) == 0


def test_psd_argument_validation_without_touching_cuda(ttsh):
    assert ttsh.ttsh_psd_workspace_bytes(64, 64, ttsh.TTSH_F64, 0) == 0
    assert ttsh.ttsh_psd_workspace_bytes(64, 64, ttsh.TTSH_F64, 1025) == 0
    assert ttsh.ttsh_psd_workspace_bytes(96, 64, ttsh.TTSH_F64, 4) == 0
    b64 = ttsh.ttsh_psd_workspace_bytes(256, 128, ttsh.TTSH_F64, 10)
    b32 = ttsh.ttsh_psd_workspace_bytes(256, 128, ttsh.TTSH_F32, 10)
    assert 10 * 256 * 128 * 16 <= b64 < 10 * 256 * 128 * 16 + (1 << 16) and 10 * 256 * 128 * 8 <= b32 < b64
    assert ttsh.ttsh_psd_create(None, [0.1], 256, 1 << 20)[0] == ttsh.TTSH_ERR_INVALID_ARG     # NULL handle
    assert ttsh.ttsh_psd_accumulate(None) == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_psd_result(None, 1)[0] == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_psd_reset(None) == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_psd_destroy(None) == ttsh.TTSH_OK
    assert ttsh.ttsh_dumbbell_order(None, 0.0, 0.0, 1.0, 1.0, 1.0)[0] == ttsh.TTSH_ERR_INVALID_ARG


def test_tangent_argument_validation_without_touching_cuda(ttsh):
    assert ttsh.ttsh_tangent_workspace_bytes(64, 64, ttsh.TTSH_F64, 0) == 0
    assert ttsh.ttsh_tangent_workspace_bytes(64, 64, ttsh.TTSH_F64, 65) == 0
    assert ttsh.ttsh_tangent_workspace_bytes(80, 64, ttsh.TTSH_F64, 2) == 0
    b2 = ttsh.ttsh_tangent_workspace_bytes(256, 256, ttsh.TTSH_F64, 2)
    b4 = ttsh.ttsh_tangent_workspace_bytes(256, 256, ttsh.TTSH_F64, 4)
    assert 2 * 3 * 256 * 256 * 8 < b2 < b4 < 4 * 8 * 256 * 256 * 8  # per vector: 3 real fields, 3 intermediates, 5 pruned spectra
    assert ttsh.ttsh_tangent_create(None, 2, 256, 1 << 20)[0] == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_tangent_step(None, 1) == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_tangent_set(None, 0, 1, 1) == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_tangent_orthonormalize(None, 1)[0] == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_tangent_get_fields(None, 0) == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_tangent_destroy(None) == ttsh.TTSH_OK


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_microbench_fma_runs_the_stated_chains(ttsh, dtype):
    """ttsh_microbench_fma (the measured ALU roof of bench.py): with a = 1, b = 0 every chain keeps its start value, so thread i
    writes (8 i + 896) / 1024 exactly; with a = 1, b = 2^-10 each chain grows by 16 x rounds / 1024; the flop count is the stated one."""
    import torch
    code, td = (ttsh.TTSH_F64, torch.float64) if dtype == "f64" else (ttsh.TTSH_F32, torch.float32)
    blocks, rounds = 3, 5
    sink = torch.full((blocks * 256,), -1.0, dtype=td, device="cuda")
    stream = torch.cuda.current_stream()
    rc, flops = ttsh.ttsh_microbench_fma(code, blocks, rounds, 1.0, 0.0, sink.data_ptr(), stream.cuda_stream)
    assert rc == ttsh.TTSH_OK and flops == 2 * 8 * 16 * rounds * 256 * blocks
    i = torch.arange(256, dtype=td, device="cuda").repeat(blocks)
    assert torch.equal(sink, (8 * i + 896) / 1024)
    rc, _ = ttsh.ttsh_microbench_fma(code, blocks, rounds, 1.0, 2.0 ** -10, sink.data_ptr(), stream.cuda_stream)
    assert rc == ttsh.TTSH_OK and torch.equal(sink, (8 * i + 896 + 8 * 16 * rounds) / 1024)
    assert ttsh.ttsh_microbench_fma(code, 0, rounds, 1.0, 0.0, sink.data_ptr(), stream.cuda_stream)[0] == ttsh.TTSH_ERR_INVALID_ARG
    assert ttsh.ttsh_microbench_fma(code, blocks, rounds, 1.0, 0.0, 0, stream.cuda_stream)[0] == ttsh.TTSH_ERR_INVALID_ARG
