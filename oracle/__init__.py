"""CPU oracle for the graph-based SP2 density-matrix path of arXiv:1603.00937.

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
`cpu_baseline` / `--impl reference` legs may import this package.  It shares no code with
`paper_1603_00937_b200/` (the CUDA path) and neither imports the other; both consume inputs
from `gbe_inputs/`.

Plain numpy/scipy in float64, following the paper passage by passage (citations `P:Lnn` are
line numbers of the paper text; `A-n` are the readings listed in DESIGN.md section 3):

    gershgorin, normalised_x0      step 0   (readings A-5, A-12)
    build_graph                    step 1   Eq.(2), Eq.(8) P:L86 (reading A-1, A-3, A-4)
    update_graph                   Eq.(8), symbolic form (graph of the next MD step from D(t-dt) and H(t))
    subgraphs, density_pattern     step 2   P:L58, Fig.1, obs. (vi) P:L65 (A-9)
    o_sub                          steps 3-6: Eq.(6) P:L60-63 with SP2   <- parity target
    OneCommunity                   steps 1-6 for one community at a time, branch sequence given (sampled outputs at full size)
    o_diag                         exact zero-temperature projector theta(mu I - H)
    o_fermi, fermi_chebyshev_coeffs  finite-temperature Chebyshev Fermi-operator expansion on the subgraphs, Eq.(7)
    expectation                    <A> = Tr[D A], E_band = Tr[D H]
    error_norms                    max and Frobenius error of the sparse D against a dense reference (Fig.2)
    o_eq5_exact, o_eq5_nested      Eq.(4)-(5) P:L47-56 literally on the full matrix (tiny inputs)

Pins (tests/test_oracle_*.py): closed forms (2x2 projector, periodic-chain projector),
library special cases (one partition / complete graph == eigendecomposition), brute force
(graph + halo by explicit loops), exact rational arithmetic for Eq.(5) == Eq.(6), and
invariants/metamorphic relations.  No function here is "parity unpinned".
"""
from .gbe_oracle import (  # noqa: F401
    gershgorin,
    normalised_x0,
    build_graph,
    update_graph,
    subgraphs,
    density_pattern,
    dense_block,
    sp2_polynomial_coeffs,
    o_sub,
    o_diag,
    o_fermi,
    fermi_chebyshev_coeffs,
    FermiResult,
    expectation,
    error_norms,
    o_eq5_exact,
    o_eq5_nested,
    SubResult,
    OneCommunity,
)
