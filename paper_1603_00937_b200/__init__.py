"""B200-native graph-based SP2 density-matrix path (arXiv:1603.00937) behind the C ABI of include/gbe.h.

    from paper_1603_00937_b200 import DeviceCSR, gbe_build_graph, gbe_density
    H = DeviceCSR.from_host(system.H)
    g = gbe_build_graph(H, tau=1e-5, part=None, n_part=512)
    D_val, log = gbe_density(H, g, n_occ, iters=40)

The CUDA library (libgbe.so, sm_100a) is built in-tree by `python -m paper_1603_00937_b200.build`; the
binding loads it lazily and fails loudly if it is missing - there is no CPU fallback.
"""
from .binding import (  # noqa: F401
    DeviceCSR,
    Graph,
    GbeError,
    Sp2Log,
    EXPORTS,
    LIB_PATH,
    lib,
    gbe_build_graph,
    gbe_build_graph_host,
    gbe_update_graph,
    gbe_density_timed,
    gbe_density_preset,
    gbe_density_fermi,
    gbe_expectation,
    gbe_expectation_static,
    GBE_STATIC_MAX_N,
    gbe_launch_count,
    gbe_graph_set_sp2_path,
    gbe_graph_set_gather_path,
    gbe_graph_set_scatter_path,
    gbe_set_build_scratch_limit,
    gbe_set_packed_max_m,
    gbe_set_dependent_launch,
    gbe_error_norms,
    gbe_graph_export,
    gbe_density,
    gbe_density_host,
    gbe_gather,
    gbe_sp2,
    gbe_scatter,
    gbe_read_log,
)
