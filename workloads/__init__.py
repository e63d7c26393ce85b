"""Seeded synthetic input generators shared by the CPU oracle tests and the CUDA path.

This package holds NO arithmetic of the AMP-PCG method itself (no PCG step, no
rounding emulation, no precision selector): it only builds the SPD systems
``A x = b`` that BASELINE.json's five configs and the paper's self-contained
examples describe, as plain numpy CSR arrays.  Both ``oracle/`` and
``paper_2505_04155_b200/`` receive these arrays verbatim; neither imports the other.
"""
from .generators import (  # noqa: F401
    CSRSystem,
    CONFIGS,
    make_config,
    poisson2d_5pt,
    poisson3d_7pt,
    vardiff3d_7pt,
    fe27_laplacian,
    random_spd_banded,
    dense_spd_from_spectrum,
    paper_example,
    uniform01,
)
