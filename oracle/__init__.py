"""CPU oracle for the TTSH pseudospectral step (TEST INFRASTRUCTURE, not product code).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with the CUDA
path under ``paper_2304_03306_b200/`` and never imports it.
"""
from .ttsh_oracle import (  # noqa: F401
    TTSHParams,
    TTSHOracle,
    PAPER_PRESET,
    BASELINE_PRESET,
    dft1,
    dft2,
    idft2,
    dft2_brute,
    signed_index,
    wavenumbers,
    cut_mask,
    process_mask,
    linear_symbol,
    psi2_of_field,
    temporal_psd,
)
