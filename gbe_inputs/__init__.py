"""Seeded synthetic tight-binding inputs.

These stand in for the paper's solvated polyalanine (Fig. 2/3) and liquid water
(Fig. 4) systems, which are not available.  The module holds NO arithmetic of the
method (no spectral bounds, no graph, no SP2): it only produces a sparse symmetric
Hamiltonian in CSR, a partition vector and an occupation, which are fed identically to the
CPU oracle (`oracle/`) and to the CUDA path (`paper_1603_00937_b200/`).
"""
from .systems import (  # noqa: F401
    CSR,
    TBSystem,
    chain,
    water_box,
    peptide_water,
    random_banded,
    config,
    contiguous_partition,
)
