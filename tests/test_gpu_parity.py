"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): integer/index work bit-exact; max|D_gpu - D_oracle| <= 1e-10;
|Tr D_gpu - Tr D_oracle| <= 1e-8.  The oracle builds its OWN graph from the same H; the two graphs are
compared first (set equality - an edge whose value sits within rounding of tau may differ, reading A-8;
on these seeded inputs none does) and no oracle input comes from the CUDA path.
"""
import numpy as np
import pytest
import scipy.sparse as sp

import gbe_inputs as gi
import oracle as o

pytestmark = pytest.mark.gpu

TOL_D = 1e-10
TOL_TR = 1e-8


@pytest.fixture(scope="module")
def gbe():
    import torch
    assert torch.cuda.is_available()
    from paper_1603_00937_b200 import build
    build.build()
    import paper_1603_00937_b200 as pkg
    pkg.lib()  # fails loudly if the CUDA library is missing
    return pkg


def run_gpu(gbe, s, iters=None, idem_tol=-1.0, power=2, part="given", H=None, sp2_path=0, gather_path=0, scatter_path=0):
    """sp2_path: 0 = the library's choice, 1 = tiled kernels, 2 = shared-memory-resident kernel, 3 = packed kernel for
    the communities with m <= 160 + tiled kernel for the others (include/gbe.h);
    gather_path: 0 = the library's choice, 1 = staged through shared memory, 2 = direct to global memory;
    scatter_path: 0 = the library's choice (bulk copies where the graph allows), 1 = the register variant."""
    import torch
    Hd = gbe.DeviceCSR.from_host(s.H if H is None else H)
    part_t = None if part is None else torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
    g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part, power=power)
    if sp2_path:
        gbe.gbe_graph_set_sp2_path(g, sp2_path)
        assert g.info["resident_sp2"] == (1 if sp2_path == 2 else 0)
        if sp2_path == 3:  # packed wherever the graph has a community that fits shared memory
            assert g.info["sp2_path_chosen"] == (3 if g.info["n_small"] > 0 else 1)
    if gather_path:
        gbe.gbe_graph_set_gather_path(g, gather_path)
    if scatter_path:
        gbe.gbe_graph_set_scatter_path(g, scatter_path)
    D, log = gbe.gbe_density(Hd, g, s.n_occ, s.iters if iters is None else iters, idem_tol)
    torch.cuda.synchronize()
    ex = {k: v.cpu().numpy() for k, v in g.export().items()}
    return g, ex, D.cpu().numpy(), log


def run_oracle(s, iters=None, idem_tol=-1.0, power=2, H=None):
    H = s.H if H is None else H
    rp, ci = o.build_graph(H, s.tau, power=power)
    return (rp, ci), o.o_sub(H, rp, ci, s.part, s.n_part, s.n_occ, s.iters if iters is None else iters, idem_tol)


def check_structure(ex, graph, r, info):
    rp, ci = graph
    assert np.array_equal(ex["S_row_ptr"], rp) and np.array_equal(ex["S_col"], ci)
    sub_ptr = np.concatenate([[0], np.cumsum([len(i) for i, _ in r.subs])])
    assert np.array_equal(ex["sub_ptr"], sub_ptr)
    assert np.array_equal(ex["sub_idx"], np.concatenate([i for i, _ in r.subs]) if len(r.subs) else [])
    assert np.array_equal(ex["ncore"], [nc for _, nc in r.subs])
    assert np.array_equal(ex["D_row_ptr"], r.D_row_ptr) and np.array_equal(ex["D_col"], r.D_col)
    assert info["nnz_D"] == r.D_val.size and info["sum_m"] == sub_ptr[-1]
    assert info["max_m"] == max(len(i) for i, _ in r.subs)
    assert abs(info["eps_min"] - r.eps_min) <= 1e-13 * abs(r.eps_min)
    assert abs(info["eps_max"] - r.eps_max) <= 1e-13 * abs(r.eps_max)
    assert abs(info["sp2_flops_per_iter"] - sum(2.0 * len(i) ** 3 for i, _ in r.subs)) < 1e-6 * info["sp2_flops_per_iter"]
    # the last SP2 iteration runs the tiles with a core row only (Eq.(6) P:L58-63 keeps the core columns)
    assert abs(info["sp2_flops_last_iter"] - sum(2.0 * len(i) ** 2 * nc for i, nc in r.subs)) <= 1e-6 * info["sp2_flops_per_iter"]
    tl = info["tile"]
    tiles = [(-(-len(i) // tl), min(-(-len(i) // tl), -(-nc // tl))) for i, nc in r.subs]
    assert info["n_tiles"] == sum(T * (T + 1) // 2 for T, _ in tiles)
    assert info["n_tiles_last"] == sum(sum(T - ti for ti in range(Tc)) for T, Tc in tiles)


def check_density(Dg, log, r):
    """Branch bits are compared while the expansion is still moving (|t1 - t2| > 1e-9); once every X_p is
    idempotent to roundoff either branch is a no-op and the bit is decided by rounding order (reading A-8)."""
    assert log.iters_done == r.iters_done
    live = np.abs(r.t1[:-1] - r.t2[:-1]) > 1e-9
    assert np.array_equal(log.branch[live[:log.iters_done]], r.branch[live[:r.iters_done]])
    assert np.abs(log.t1 - r.t1).max() <= TOL_TR and np.abs(log.t2 - r.t2).max() <= TOL_TR
    assert np.abs(Dg - r.D_val).max() <= TOL_D
    assert abs(log.t1[-1] - r.t1[-1]) <= TOL_TR  # |Tr D_gpu - Tr D_oracle| (reading A-11)


# ------------------------------------------------------------------------------- main configurations
@pytest.mark.parametrize("sp2_path", [1, 2, 3])
def test_config1_chain(gbe, sp2_path):
    s = gi.config(1)
    g, ex, Dg, log = run_gpu(gbe, s, sp2_path=sp2_path)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    assert g.info["contiguous_cores"] == 1
    # trace of the assembled D equals the logged core trace
    D = sp.csr_matrix((Dg, ex["D_col"], ex["D_row_ptr"]), shape=(s.n, s.n))
    assert abs(D.diagonal().sum() - log.t1[-1]) < 1e-9


def test_config1_default_partition_is_contiguous_blocks(gbe):
    s = gi.config(1)
    g, ex, Dg, log = run_gpu(gbe, s, part=None)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)


@pytest.mark.parametrize("seed", [0, 1])
def test_shuffled_communities_general_scatter(gbe, seed):
    s = gi.random_banded(200, half_bw=5, n_part=7, seed=seed, tau=1e-4, iters=30, shuffle=True)
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    assert g.info["contiguous_cores"] == 0


def test_config2_water_1024(gbe):
    s = gi.config(2)
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    m = np.diff(ex["sub_ptr"])
    assert m.min() > 128 and m.max() > 512  # several tiles and a ragged tail per community


def test_config3_water_4096_full_size(gbe):
    """BASELINE.json configs[2], the workload bench.py times (24,576 orbitals, 512 communities, 40 iterations):
    every stored entry of D against the oracle's full expansion (the oracle needs about half a minute here)."""
    s = gi.config(3)
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    assert g.info["n"] == 24576 and g.info["n_part"] == 512 and log.iters_done == 40


def test_config4_reduced_peptide_heterogeneous_sizes(gbe):
    """BASELINE.json configs[3] at a size the oracle finishes in about a minute: the same construction
    (random-coil solute + water, reading A-16) with 150 residues in a 30 A cube - 10,626 orbitals, 216 communities
    given by an explicit partition vector, core+halo sizes 200 ... 1,530 (many tiles, ragged tails, two core sizes)."""
    s = gi.peptide_water(150, box=30.0, seed=1)
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    m = np.diff(ex["sub_ptr"])
    assert m.min() < 256 and m.max() > 1400


@pytest.mark.parametrize("tau,n_part", [(1e-3, 256), (1e-3, 32), (1e-6, 128), (1e-7, 64)])
def test_config5_sweep_points(gbe, tau, n_part):
    """BASELINE.json configs[4] (tau x partition sweep), at the 1,024-molecule box the oracle finishes quickly: the
    corners of the grid give core+halo sizes from ~35 (less than one tile) to ~1,600 (25 x 25 tiles)."""
    s = gi.water_box(1024, n_part, seed=0, tau=tau, iters=16)
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    if (tau, n_part) == (1e-3, 256):  # 256 small communities: more than are co-resident -> the packed kernel
        assert g.info["sp2_path_chosen"] == 3 and g.info["n_small"] >= 240


@pytest.mark.parametrize("n_part", [256, 128, 64])
def test_config5_small_m_regime_packed_kernel(gbe, n_part):
    """The small-m regime of BASELINE.json configs[4] (cost law P:L78: more partitions, smaller m), tau = 1e-3 on the
    1,024-molecule box (the same density, hence the same m, as the 24,576-orbital box with 4 x the communities):
    256 communities m ~ 30 - 125 (nearly all packed), 128 communities m ~ 65 - 185 (MIXED: the packed kernel takes m <= 160, the
    tiled kernel the others, in the same iteration), 64 communities m ~ 140 - 285 (mostly tiled).  Both the library's
    choice and the forced packed path against the oracle; the packed path is bitwise reproducible."""
    import torch
    s = gi.water_box(1024, n_part, seed=0, tau=1e-3, iters=20)
    graph, r = run_oracle(s)
    g, ex, Dg, log = run_gpu(gbe, s, sp2_path=3)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    m = np.diff(ex["sub_ptr"])
    assert g.info["n_small"] == int(((m > 0) & (m <= 160)).sum())
    if n_part == 128:
        assert 0 < g.info["n_small"] < n_part  # the mixed case really is mixed
    _, _, Dg2, log2 = run_gpu(gbe, s, sp2_path=3)
    assert np.array_equal(Dg, Dg2) and np.array_equal(log.t1, log2.t1) and np.array_equal(log.t2, log2.t2)
    _, _, Dt, logt = run_gpu(gbe, s, sp2_path=1)
    assert np.abs(Dt - Dg).max() <= 1e-12


@pytest.mark.slow
def test_config5_largest_point_at_full_size(gbe):
    """BASELINE.json configs[4] on the full 24,576-orbital box at the corner with the largest subgraphs (tau = 1e-7, 128
    communities: core+halo 1,493 .. 2,295, up to 36 x 36 tiles per community, 3.4 GB per dense buffer).  Four SP2
    iterations keep the oracle at about a minute; every stored entry of D is compared."""
    s = gi.water_box(4096, 128, seed=0, tau=1e-7, iters=4)
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    assert g.info["max_m"] > 2000


def check_any_size_properties(s, g, ex, Dg, log):
    """Properties of the path that hold at any size (used where the oracle is too slow to run in full)."""
    t1, t2, br = log.t1, log.t2, log.branch
    assert log.iters_done == s.iters and np.isfinite(Dg).all()
    # spectrum of every X_p stays in [0,1]: 0 <= Tr_core X^2 <= Tr_core X (up to roundoff of a sum of ~n terms)
    assert (t2 >= -1e-9).all() and (t2 <= t1 + 1e-9 * s.n).all()
    # the logged branch is the rule of reading A-6 applied to the logged traces
    for k in range(log.iters_done):
        if abs(t1[k] - t2[k]) > 1e-9:
            assert br[k] == (0 if abs(t2[k] - s.n_occ) < abs(2 * t1[k] - t2[k] - s.n_occ) else 1)
    # the update really was X <- X^2 or 2X - X^2 for EVERY community: the next core trace follows exactly
    nxt = np.where(br == 0, t2[:-1], 2 * t1[:-1] - t2[:-1])
    assert np.abs(t1[1:] - nxt).max() <= 1e-9 * max(1.0, s.n_occ)
    D = sp.csr_matrix((Dg, ex["D_col"], ex["D_row_ptr"]), shape=(s.n, s.n))
    assert abs(D.diagonal().sum() - t1[-1]) <= 1e-9 * s.n          # scatter: Tr D = last core trace
    # X_p is symmetric, so D restricted to core x core of one community is symmetric (sampled communities)
    rng = np.random.default_rng(0)
    for p in rng.choice(s.n_part, size=min(8, s.n_part), replace=False):
        idx = ex["sub_idx"][ex["sub_ptr"][p]:ex["sub_ptr"][p] + ex["ncore"][p]]
        blk = D[idx][:, idx].toarray()
        assert np.abs(blk - blk.T).max() <= 1e-11
    # D is zero outside S' by construction: every stored row index of column i lies in the subgraph of i's community
    assert D.nnz <= g.info["nnz_D"]


def check_sampled_communities(s, ex, Dg, log, n_random):
    """Sampled outputs the oracle can compute one by one at any size: for the largest, the smallest and a few random
    communities the oracle derives the subgraph from (H, tau) alone and expands it with the branch sequence the GPU
    logged (the sequence is a global quantity: P:L90); subgraph indices bit for bit, every stored entry of D in the
    community's core columns within the 1e-10 bar."""
    oc = o.OneCommunity(s.H, s.tau, s.part)
    m = np.diff(ex["sub_ptr"])
    rng = np.random.default_rng(1)
    picks = {int(np.argmax(m)), int(np.argmin(np.where(m > 0, m, m.max())))}
    picks |= {int(p) for p in rng.choice(s.n_part, size=min(n_random, s.n_part), replace=False)}
    D = sp.csr_matrix((Dg, ex["D_col"], ex["D_row_ptr"]), shape=(s.n, s.n))
    for p in sorted(picks):
        idx, nc, cols = oc.expand(p, log.branch, log.iters_done)
        a, b = ex["sub_ptr"][p], ex["sub_ptr"][p + 1]
        assert np.array_equal(ex["sub_idx"][a:b], idx) and ex["ncore"][p] == nc
        got = D[idx][:, idx[:nc]].toarray()
        assert np.abs(got - cols).max() <= TOL_D, (p, len(idx))


_FULL_BOX = {}


def _full_box():
    """The 24,576-orbital water box of BASELINE.json configs[2] and configs[4], generated once per test session."""
    if "s" not in _FULL_BOX:
        _FULL_BOX["s"] = gi.water_box(4096, 512, seed=0)
    return _FULL_BOX["s"]


@pytest.mark.slow
@pytest.mark.parametrize("tau", [1e-3, 1e-4, 1e-5, 1e-6, 1e-7])
def test_config5_full_grid_sampled_parity(gbe, tau):
    """BASELINE.json configs[4] at FULL size: every (tau, communities) point of the grid on the 24,576-orbital box, 40 SP2
    iterations, in the launch configuration bench.py --sweep times (the library's own choice of kernels).  Per tau the
    graph S_tau is compared bit for bit with the oracle's own (it does not depend on the partition); per point the
    any-size properties, and element by element (Eq.(6)) the largest, the smallest and two random communities
    against the one-community oracle, which derives the subgraph from (H, tau) alone and replays the logged branch
    sequence (the sequence is a global quantity).  The max |D_gpu - D_oracle| per point goes to
    gpurun_out/config5_full_grid_parity.jsonl for profiles/."""
    import json
    import os
    import torch
    base = _full_box()
    Hd = gbe.DeviceCSR.from_host(base.H)
    rp, ci = o.build_graph(base.H, tau)
    oc = None
    for n_part in (128, 256, 512, 1024):
        part = (np.arange(base.n) // -(-base.n // n_part)).astype(np.int32)  # part = NULL: contiguous blocks
        g = gbe.gbe_build_graph(Hd, tau, None, n_part)
        D, log = gbe.gbe_density(Hd, g, base.n_occ, base.iters)
        torch.cuda.synchronize()
        ex = {k: v.cpu().numpy() for k, v in g.export().items()}
        Dg = D.cpu().numpy()
        assert np.array_equal(ex["S_row_ptr"], rp) and np.array_equal(ex["S_col"], ci)

        class _S:  # what the two checkers read
            pass
        sv = _S()
        sv.H, sv.tau, sv.part, sv.n_part, sv.n, sv.n_occ, sv.iters = base.H, tau, part, n_part, base.n, base.n_occ, base.iters
        check_any_size_properties(sv, g, ex, Dg, log)
        if oc is None:
            oc = o.OneCommunity(base.H, tau, part)
        oc.part = part
        m = np.diff(ex["sub_ptr"])
        rng = np.random.default_rng(int(n_part))
        picks = {int(np.argmax(m)), int(np.argmin(m))} | {int(p) for p in rng.choice(n_part, size=2, replace=False)}
        Dm = sp.csr_matrix((Dg, ex["D_col"], ex["D_row_ptr"]), shape=(base.n, base.n))
        worst = 0.0
        for p in sorted(picks):
            idx, nc, cols = oc.expand(p, log.branch, log.iters_done)
            a, b = ex["sub_ptr"][p], ex["sub_ptr"][p + 1]
            assert np.array_equal(ex["sub_idx"][a:b], idx) and ex["ncore"][p] == nc
            worst = max(worst, float(np.abs(Dm[idx][:, idx[:nc]].toarray() - cols).max()))
        assert worst <= TOL_D, (tau, n_part, worst)
        out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
        if os.path.isdir(out):
            with open(os.path.join(out, "config5_full_grid_parity.jsonl"), "a") as f:
                f.write(json.dumps({"tau": tau, "n_part": n_part, "sp2_path": int(g.info["sp2_path_chosen"]),
                                    "m_min": int(m.min()), "m_max": int(m.max()), "communities_checked": sorted(picks),
                                    "max_abs_dD": worst, "graph_bit_exact": True, "iters": int(log.iters_done)}) + "\n")
        g.free()
        del D, Dg, Dm, ex


@pytest.mark.slow
def test_config4_full_size_properties(gbe):
    """BASELINE.json configs[3] at full size (2,000 residues, ~1.2e5 orbitals, 2 x 27 GB dense batch).  The oracle would
    need ~1e15 flop for the whole batch, so the full-size run is checked (1) through properties that hold at any size and
    (2) element by element on sampled communities the oracle computes one at a time; element-by-element parity of the
    whole batch for the same construction is test_config4_reduced_peptide_heterogeneous_sizes."""
    s = gi.config(4)
    g, ex, Dg, log = run_gpu(gbe, s)
    assert g.info["n"] == s.n and g.info["max_m"] > 1500
    check_any_size_properties(s, g, ex, Dg, log)
    check_sampled_communities(s, ex, Dg, log, n_random=4)


def test_any_size_properties_hold_where_parity_is_known(gbe):
    s = gi.config(2)
    g, ex, Dg, log = run_gpu(gbe, s)
    check_any_size_properties(s, g, ex, Dg, log)
    check_sampled_communities(s, ex, Dg, log, n_random=2)


# ------------------------------------------------------------------------------- pieces
@pytest.mark.parametrize("which", ["chain", "water", "shuffled", "peptide"])
def test_gather_paths_pack_identical_blocks(gbe, which):
    """The staged and the direct gather kernel (include/gbe.h, gbe_graph_set_gather_path): with iters = 0 the result is
    the gathered X0 itself, which must agree bit for bit; the traces of X_0 are summed in another order (rounding);
    the full expansion through the direct kernel meets the same bar against the oracle."""
    s = {"chain": lambda: gi.config(1),
         "water": lambda: gi.water_box(256, 32, seed=3, tau=1e-5, iters=12),
         "shuffled": lambda: gi.random_banded(300, half_bw=6, n_part=9, seed=5, tau=1e-4, iters=20, shuffle=True),
         "peptide": lambda: gi.peptide_water(40, box=20.0, seed=2)}[which]()
    _, _, D1, log1 = run_gpu(gbe, s, iters=0, gather_path=1)
    _, _, D2, log2 = run_gpu(gbe, s, iters=0, gather_path=2)
    assert np.array_equal(D1, D2)
    assert abs(log1.t1[0] - log2.t1[0]) <= 1e-12 * s.n and abs(log1.t2[0] - log2.t2[0]) <= 1e-12 * s.n
    g, ex, Dg, log = run_gpu(gbe, s, gather_path=2)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)


@pytest.mark.parametrize("which", ["chain", "water", "water_ragged", "odd_cores", "shuffled", "wide_cores", "tiny_cores"])
def test_scatter_paths_write_identical_d(gbe, which):
    """The bulk-copy and the register scatter kernel (include/gbe.h, gbe_graph_set_scatter_path) move the same runs: D
    agrees bit for bit after a full expansion and with iters = 0 (D = the core columns of X0: every entry distinct, so a
    run put in the wrong place or cut short cannot hide).  chain / water: even index-range cores - the bulk kernel runs;
    water_ragged: 5 communities - a ragged last group of runs; odd_cores (cores of 33) / shuffled:
    the bulk kernel's conditions fail and the default must fall back; wide_cores: cores of 192 (slots of 1.5 KB);
    tiny_cores: cores of 2 (16-byte runs)."""
    s = {"chain": lambda: gi.config(1),
         "water": lambda: gi.water_box(256, 32, seed=3, tau=1e-5, iters=12),
         "water_ragged": lambda: gi.water_box(40, 5, seed=4, tau=1e-4, iters=8),
         "odd_cores": lambda: gi.random_banded(297, half_bw=6, n_part=9, seed=5, tau=1e-4, iters=10),
         "shuffled": lambda: gi.random_banded(300, half_bw=6, n_part=9, seed=5, tau=1e-4, iters=10, shuffle=True),
         "wide_cores": lambda: gi.water_box(128, 4, seed=6, tau=1e-4, iters=6),
         "tiny_cores": lambda: gi.random_banded(64, half_bw=3, n_part=32, seed=7, tau=1e-4, iters=10)}[which]()
    for iters in (0, None):
        g0, _, D0, _ = run_gpu(gbe, s, iters=iters, scatter_path=0)
        _, _, D1, _ = run_gpu(gbe, s, iters=iters, scatter_path=1)
        assert D0.size == g0.info["nnz_D"] and np.array_equal(D0, D1)
    graph, r = run_oracle(s)
    assert np.abs(D0 - r.D_val).max() <= 1e-10


@pytest.mark.parametrize("which", ["chain", "water_ragged", "odd_cores", "shuffled", "tiny_cores", "peptide", "water_tma"])
@pytest.mark.parametrize("d_offset", [0, 1])
def test_nothing_is_written_outside_workspace_and_d(gbe, which, d_offset):
    """Guard bands around the caller's buffers (the bulk row stores of the gather and the bulk run copies of the scatter
    address whole rows and runs; ragged tails and the last community are where an overrun would show): the workspace and
    D_val are slices of larger buffers filled with a sentinel, which must be intact after gbe_density, and D must equal
    the result in buffers of their own.  d_offset = 1: D_val is only 8-byte aligned - the bulk scatter does not apply and
    the library must fall back by itself.  water_tma: long K loops - the tiled kernel runs its TMA variant."""
    import torch
    s = {"chain": lambda: gi.config(1),
         "water_ragged": lambda: gi.water_box(40, 5, seed=4, tau=1e-4, iters=8),
         "odd_cores": lambda: gi.random_banded(297, half_bw=6, n_part=9, seed=5, tau=1e-4, iters=10),
         "shuffled": lambda: gi.random_banded(300, half_bw=6, n_part=9, seed=5, tau=1e-4, iters=10, shuffle=True),
         "tiny_cores": lambda: gi.random_banded(64, half_bw=3, n_part=32, seed=7, tau=1e-4, iters=10),
         "peptide": lambda: gi.peptide_water(40, box=20.0, seed=2),
         "water_tma": lambda: gi.water_box(384, 3, seed=8, tau=1e-5, iters=6)}[which]()
    Hd = gbe.DeviceCSR.from_host(s.H)
    part_t = torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
    g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
    info = g.info
    if which == "water_tma":  # three communities of m ~ 2,260 (ragged last tile): the X^2 kernel with panels by 2-D TMA
        assert info["x2_tma"] == 1 and info["max_m"] % 64 != 0
    D_ref, _ = gbe.gbe_density(Hd, g, s.n_occ, s.iters, -1.0)
    pad_ws, pad_d, sentinel = 1 << 16, 1024, 1.2345e300
    ws_big = torch.full((info["workspace_bytes"] + 2 * pad_ws,), 0xA5, dtype=torch.uint8, device="cuda")
    d_big = torch.full((info["nnz_D"] + 2 * pad_d + d_offset,), sentinel, dtype=torch.float64, device="cuda")
    ws = ws_big[pad_ws:pad_ws + info["workspace_bytes"]]
    D = d_big[pad_d + d_offset:pad_d + d_offset + info["nnz_D"]]
    def intact():
        return (bool((ws_big[:pad_ws] == 0xA5).all()) and bool((ws_big[pad_ws + info["workspace_bytes"]:] == 0xA5).all())
                and bool((d_big[:pad_d + d_offset] == sentinel).all())
                and bool((d_big[pad_d + d_offset + info["nnz_D"]:] == sentinel).all()))
    for gather_path in (1, 2):
        gbe.gbe_graph_set_gather_path(g, gather_path)
        D.fill_(sentinel)
        gbe.gbe_density(Hd, g, s.n_occ, s.iters, -1.0, workspace=ws, D_val=D, want_log=False)
        torch.cuda.synchronize()
        assert intact() and torch.equal(D, D_ref)
    gbe.gbe_graph_set_gather_path(g, 0)
    # the other SP2 kernels (1 tiled, 2 resident where the graph allows it, 3 packed): same buffers, same bands; their
    # traces are summed in another order, so D agrees to the parity bar, not bit for bit
    for sp2_path in (1, 2, 3):
        try:
            gbe.gbe_graph_set_sp2_path(g, sp2_path)
        except Exception:
            continue  # (the resident kernel does not take this graph)
        D.fill_(sentinel)
        gbe.gbe_density(Hd, g, s.n_occ, s.iters, -1.0, workspace=ws, D_val=D, want_log=False)
        torch.cuda.synchronize()
        assert intact() and float((D - D_ref).abs().max()) <= 1e-10, sp2_path


@pytest.mark.parametrize("sp2_path", [1, 2, 3])
def test_iters_zero_returns_gathered_x0(gbe, sp2_path):
    """gather + scatter alone: D = core columns of X0[s,s]; exact up to the rounding of the two bounds."""
    s = gi.random_banded(150, half_bw=4, n_part=5, seed=3, tau=1e-3)
    g, ex, Dg, log = run_gpu(gbe, s, iters=0, sp2_path=sp2_path)
    graph, r = run_oracle(s, iters=0)
    check_structure(ex, graph, r, g.info)
    assert log.iters_done == 0 and log.t1.size == 1
    assert np.abs(Dg - r.D_val).max() <= 4e-16
    assert abs(log.t1[0] - r.t1[0]) < 1e-12 and abs(log.t2[0] - r.t2[0]) < 1e-12


@pytest.mark.parametrize("power", [1, 3])
def test_graph_power(gbe, power):
    s = gi.random_banded(120, half_bw=3, n_part=4, seed=5, tau=1e-3, iters=25)
    g, ex, Dg, log = run_gpu(gbe, s, power=power)
    graph, r = run_oracle(s, power=power)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)


@pytest.mark.parametrize("which", ["water", "banded_power3", "update"])
def test_graph_build_with_and_without_the_kept_bitmaps(gbe, which):
    """The numeric pass of the thresholded product either reads back the candidate bitmaps of the sizing pass or walks the
    products again (include/gbe.h, gbe_set_build_scratch_limit): same graph bit for bit, and equal to the oracle's."""
    import torch
    if which == "water":
        s, power = gi.water_box(256, 32, seed=3, iters=5), 2
    else:
        s, power = gi.random_banded(300, half_bw=4, n_part=6, seed=8, tau=1e-3, iters=5), 3
    Hd = gbe.DeviceCSR.from_host(s.H)
    exs = []
    for limit in (0, 8 << 30):
        old = gbe.gbe_set_build_scratch_limit(limit)
        try:
            g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part, power=power)
            if which == "update":
                D, _ = gbe.gbe_density(Hd, g, s.n_occ, s.iters)
                g = gbe.gbe_update_graph(g, D, Hd, 1e-4, None, s.n_part)
            torch.cuda.synchronize()
        finally:
            assert gbe.gbe_set_build_scratch_limit(old) == limit
        exs.append({k: v.cpu().numpy() for k, v in g.export().items()})
    for k in exs[0]:
        assert np.array_equal(exs[0][k], exs[1][k]), k
    if which != "update":
        rp, ci = o.build_graph(s.H, s.tau, power=power)
        assert np.array_equal(exs[0]["S_row_ptr"], rp) and np.array_equal(exs[0]["S_col"], ci)


@pytest.mark.parametrize("tau", [1e-1, 1e-3, 1e-7, 0.0, 1.5])
def test_tau_sweep_chain(gbe, tau):
    s = gi.chain(256, 8, tau=tau, iters=30)
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    if tau > 1:
        assert g.info["nnz_S"] == s.n  # self loops only (A-12)


@pytest.mark.parametrize("sp2_path", [1, 2, 3])
def test_idem_tol_stops_on_device(gbe, sp2_path):
    s = gi.config(1)
    g, ex, Dg, log = run_gpu(gbe, s, iters=60, idem_tol=1e-9, sp2_path=sp2_path)
    graph, r = run_oracle(s, iters=60, idem_tol=1e-9)
    assert 15 < log.iters_done < 40
    check_density(Dg, log, r)


# ------------------------------------------------------------------------------- pre-determined SP2 sequence
@pytest.mark.parametrize("sp2_path", [1, 2, 3])
@pytest.mark.parametrize("trace", [True, False])
def test_preset_sequence_from_the_previous_md_step(gbe, trace, sp2_path):
    """'the complete SP2 sequence (the same for each subgraph expansion) ... can be determined beforehand':
    the sequence is the one the oracle chooses for the Hamiltonian of the previous step (another noise draw), applied
    to the current H; the oracle replays the same sequence."""
    import torch
    prev = gi.chain(512, 16, seed=3)
    s = gi.chain(512, 16, seed=0)
    rp, ci = o.build_graph(prev.H, prev.tau)
    seq = o.o_sub(prev.H, rp, ci, prev.part, prev.n_part, prev.n_occ, prev.iters).branch
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, s.iters, replay=(seq, len(seq)))
    Hd = gbe.DeviceCSR.from_host(s.H)
    g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
    gbe.gbe_graph_set_sp2_path(g, sp2_path)
    Dg, log = gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=trace)
    torch.cuda.synchronize()
    assert log.iters_done == len(seq) and np.array_equal(log.branch, seq)
    assert np.abs(Dg.cpu().numpy() - r.D_val).max() <= TOL_D
    assert abs(log.t1[-1] - r.t1[-1]) <= TOL_TR and abs(log.t2[-1] - r.t2[-1]) <= TOL_TR
    if trace:
        assert np.abs(log.t1 - r.t1).max() <= TOL_TR and np.abs(log.t2 - r.t2).max() <= TOL_TR


def test_preset_arbitrary_sequence_on_water(gbe):
    """Any 0/1 sequence is a polynomial (Eq.(1)): a fixed alternating sequence on the 6,144-orbital box, with no
    reduction kernel between the products; compared with the oracle's replay of the same sequence."""
    import torch
    s = gi.config(2)
    seq = np.array([1, 0] * 6, dtype=np.uint8)
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, len(seq), replay=(seq, len(seq)))
    Hd = gbe.DeviceCSR.from_host(s.H)
    g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
    n0 = gbe.gbe_launch_count()
    Dg, log = gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False)
    torch.cuda.synchronize()
    assert g.info["x2_tma"] == 1  # m ~ 500: long K loops, panels by TMA (one launch sets the tensor-map addresses)
    assert gbe.gbe_launch_count() - n0 == 2 + 1 + 1 + 1 + len(seq) + 1 + 1  # bounds(2) gather tensor-maps init x2... final trace scatter
    assert np.abs(Dg.cpu().numpy() - r.D_val).max() <= TOL_D
    assert abs(log.t1[-1] - r.t1[-1]) <= TOL_TR
    with pytest.raises(gbe.GbeError):
        gbe.gbe_density_preset(Hd, g, np.array([0, 2], dtype=np.uint8))


@pytest.mark.parametrize("which", ["water", "shuffled", "chain"])
def test_preset_sequence_in_a_bounded_workspace(gbe, which):
    """with the SP2 sequence fixed beforehand the expansions run "without exchange of information during or between
    the matrix multiplications" - nothing couples the communities, so gbe_density_preset(trace_every_iteration = 0) works
    through them in waves when the workspace holds only part of the batch.  Same kernels on the same tiles: D must be
    BIT FOR BIT the D of the whole-batch run, for any workspace between the minimum (the largest community) and the full
    size; and it must meet the oracle's replay of the same sequence."""
    import torch
    s = {"water": lambda: gi.config(2),
         "shuffled": lambda: gi.random_banded(700, half_bw=6, n_part=23, seed=5, tau=1e-4, iters=20, shuffle=True),
         "chain": lambda: gi.chain(4800, 600, seed=5)}[which]()
    seq = np.array([1, 0, 0, 1, 0, 1, 1, 0, 1, 0, 0, 1][: min(12, s.iters)], dtype=np.uint8)
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, len(seq), replay=(seq, len(seq)))
    Hd = gbe.DeviceCSR.from_host(s.H)
    part_t = torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
    g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
    gbe.gbe_graph_set_sp2_path(g, 1)  # the whole-batch reference on the same (tiled) kernels
    full, small = g.info["workspace_bytes"], g.info["workspace_bytes_preset_min"]
    assert small < full
    D_full, log_full = gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False)
    torch.cuda.synchronize()
    assert np.abs(D_full.cpu().numpy() - r.D_val).max() <= TOL_D
    for nbytes in (small, small + (full - small) // 3, full - 256):
        ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        D_w, log_w = gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False, workspace=ws)
        torch.cuda.synchronize()
        assert torch.equal(D_w, D_full), nbytes
        assert log_w.iters_done == len(seq) and abs(log_w.t1[-1] - r.t1[-1]) <= TOL_TR and abs(log_w.t2[-1] - r.t2[-1]) <= TOL_TR
    # zero iterations: the waves return the gathered X0
    D0f, _ = gbe.gbe_density_preset(Hd, g, seq[:0], trace_every_iteration=False)
    D0w, l0 = gbe.gbe_density_preset(Hd, g, seq[:0], trace_every_iteration=False,
                                     workspace=torch.empty(small, dtype=torch.uint8, device="cuda"))
    torch.cuda.synchronize()
    assert torch.equal(D0f, D0w) and abs(l0.t1[0] - r.t1[0]) <= TOL_TR
    # below the minimum, or with per-iteration traces (which couple the communities), the small workspace is refused
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False,
                               workspace=torch.empty(small - 256, dtype=torch.uint8, device="cuda"))
    assert e.value.status == -5
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=True,
                               workspace=torch.empty(small, dtype=torch.uint8, device="cuda"))
    assert e.value.status == -5


@pytest.mark.parametrize("which", ["water_ragged", "shuffled", "peptide"])
def test_guard_bands_waves_and_fermi(gbe, which):
    """The same guard bands (test_nothing_is_written_outside_workspace_and_d) around the SMALLEST workspace the pre-set
    sequence accepts (waves of communities: dense offsets are shifted per wave) and around the Fermi expansion's
    workspace (four dense batches)."""
    import torch
    s = {"water_ragged": lambda: gi.water_box(40, 5, seed=4, tau=1e-4, iters=8),
         "shuffled": lambda: gi.random_banded(300, half_bw=6, n_part=9, seed=5, tau=1e-4, iters=10, shuffle=True),
         "peptide": lambda: gi.peptide_water(40, box=20.0, seed=2)}[which]()
    Hd = gbe.DeviceCSR.from_host(s.H)
    part_t = torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
    g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
    gbe.gbe_graph_set_sp2_path(g, 1)
    info = g.info
    pad_ws, pad_d, sentinel = 1 << 16, 1024, 1.2345e300
    d_big = torch.full((info["nnz_D"] + 2 * pad_d,), sentinel, dtype=torch.float64, device="cuda")
    D = d_big[pad_d:pad_d + info["nnz_D"]]
    seq = np.array([1, 0, 0, 1, 0, 1, 1, 0], dtype=np.uint8)
    D_ref, _ = gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False)
    F_ref, _ = gbe.gbe_density_fermi(Hd, g, 0.0, 1.5, 21)
    for nbytes, run, ref in (
            (info["workspace_bytes_preset_min"],
             lambda ws: gbe.gbe_density_preset(Hd, g, seq, trace_every_iteration=False, workspace=ws, D_val=D, want_log=False), D_ref),
            (info["workspace_bytes_fermi"],
             lambda ws: gbe.gbe_density_fermi(Hd, g, 0.0, 1.5, 21, workspace=ws, D_val=D, want_n_elec=False), F_ref)):
        ws_big = torch.full((nbytes + 2 * pad_ws,), 0xA5, dtype=torch.uint8, device="cuda")
        D.fill_(sentinel)
        run(ws_big[pad_ws:pad_ws + nbytes])
        torch.cuda.synchronize()
        assert bool((ws_big[:pad_ws] == 0xA5).all()) and bool((ws_big[pad_ws + nbytes:] == 0xA5).all())
        assert bool((d_big[:pad_d] == sentinel).all()) and bool((d_big[pad_d + info["nnz_D"]:] == sentinel).all())
        assert torch.equal(D, ref)


# ------------------------------------------------------------------------------- Eq.(8): graph of the next MD step
@pytest.mark.parametrize("which", ["chain", "water"])
def test_update_graph_eq8_md_step(gbe, which):
    """One MD step: D(t - dt) on S(t - dt), then S(t) from Eq.(8) with the moved Hamiltonian H(t), then D(t) on
    S(t).  Graph, halos and the new D against the oracle, which does the same from its own D(t - dt)."""
    import torch
    if which == "chain":
        s0, s1, tau_d = gi.chain(512, 16, seed=0), gi.chain(512, 16, seed=1), 1e-4
    else:
        s0, s1, tau_d = gi.water_box(256, 32, seed=0, iters=20), gi.water_box(256, 32, seed=0, iters=20), 1e-4
        # H(t): the same box with every element moved by up to 0.1 %, kept symmetric
        Hs = s1.H.to_scipy()
        Hs.data = Hs.data * (1.0 + 1e-3 * np.cos(np.arange(Hs.nnz) * 0.37))
        s1.H = gi.CSR.from_scipy((Hs + Hs.T) * 0.5)
    g0, ex0, D0, log0 = run_gpu(gbe, s0)
    H1 = gbe.DeviceCSR.from_host(s1.H)
    g1 = gbe.gbe_update_graph(g0, torch.from_numpy(D0).cuda(), H1, tau_d, None, s1.n_part)
    D1, log1 = gbe.gbe_density(H1, g1, s1.n_occ, s1.iters)
    torch.cuda.synchronize()
    ex1 = {k: v.cpu().numpy() for k, v in g1.export().items()}
    # oracle: its own previous step, its own Eq.(8)
    (rp0, ci0), r0 = run_oracle(s0)
    rp1, ci1 = o.update_graph(r0.D_row_ptr, r0.D_col, r0.D_val, s1.H, tau_d)
    r1 = o.o_sub(s1.H, rp1, ci1, s1.part, s1.n_part, s1.n_occ, s1.iters)
    check_structure(ex1, (rp1, ci1), r1, g1.info)
    check_density(D1.cpu().numpy(), log1, r1)
    assert g1.info["nnz_S"] >= ex0["S_col"].size or which == "water"


# ------------------------------------------------------------------------------- Eq.(7): finite-temperature expansion
def run_fermi(gbe, s, mu, beta, order):
    import torch
    Hd = gbe.DeviceCSR.from_host(s.H)
    part_t = torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
    g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
    D, ne = gbe.gbe_density_fermi(Hd, g, mu, beta, order)
    torch.cuda.synchronize()
    ex = {k: v.cpu().numpy() for k, v in g.export().items()}
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_fermi(s.H, rp, ci, s.part, s.n_part, mu, beta, order)
    assert np.array_equal(ex["D_row_ptr"], r.D_row_ptr) and np.array_equal(ex["D_col"], r.D_col)
    return g, D.cpu().numpy(), ne, r


@pytest.mark.parametrize("order", [1, 2, 7, 64])
def test_fermi_chebyshev_chain(gbe, order):
    """Eq.(7) P:L67-72 on config 1's chain (16 communities of 40-48 orbitals, less than one tile each), odd and even
    orders (the recurrence ping-pongs two buffers) and the shortest series."""
    s = gi.config(1)
    g, Dg, ne, r = run_fermi(gbe, s, 0.3, 2.0, order)
    assert np.abs(Dg - r.D_val).max() <= TOL_D
    assert abs(ne - r.n_elec) <= TOL_TR


def test_fermi_chebyshev_water_and_shuffled(gbe):
    """Several tiles with ragged tails (6,144-orbital water box, order 60) and non-contiguous communities."""
    s = gi.config(2)
    w_mid = -11.0  # inside the O-p / H-s manifold of the synthetic water model
    g, Dg, ne, r = run_fermi(gbe, s, w_mid, 0.8, 60)
    assert np.abs(Dg - r.D_val).max() <= TOL_D
    assert abs(ne - r.n_elec) <= 1e-7
    s2 = gi.random_banded(200, half_bw=5, n_part=7, seed=1, tau=1e-4, shuffle=True)
    g, Dg, ne, r = run_fermi(gbe, s2, 0.0, 1.5, 33)
    assert np.abs(Dg - r.D_val).max() <= TOL_D and abs(ne - r.n_elec) <= TOL_TR
    with pytest.raises(gbe.GbeError):
        gbe.gbe_density_fermi(gbe.DeviceCSR.from_host(s2.H), g, 0.0, -1.0, 10)


# ------------------------------------------------------------------------------- observables
def test_band_energy_and_expectation_values(gbe):
    """The whole chain on both sides: the GPU takes the expectation of ITS density matrix, the oracle of its own (no
    oracle input comes from the CUDA path); |D_gpu - D_oracle| <= 1e-10 bounds the difference by 1e-10 * sum|A|."""
    import torch
    s = gi.config(2)
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    Hd = gbe.DeviceCSR.from_host(s.H)
    Dt = torch.from_numpy(Dg).cuda()
    e_gpu = gbe.gbe_expectation(g, Dt, Hd)
    e_ref = o.expectation(r.D_row_ptr, r.D_col, r.D_val, s.H)
    assert abs(e_gpu - e_ref) <= 1e-10 * np.abs(s.H.val).sum()
    assert abs(e_gpu - e_ref) <= 1e-9 * abs(e_ref)
    assert gbe.gbe_expectation(g, Dt, Hd) == e_gpu  # fixed reduction order: reproducible
    # Tr[D I] is the trace the SP2 log reports; a non-symmetric operand exercises the transposed lookup
    eye = gi.CSR.from_scipy(sp.identity(s.n, format="csr"))
    assert abs(gbe.gbe_expectation(g, Dt, gbe.DeviceCSR.from_host(eye)) - log.t1[-1]) <= 1e-8
    rng = np.random.default_rng(1)
    A = sp.random(s.n, s.n, density=2e-3, random_state=rng, format="csr") + sp.triu(s.H.to_scipy(), k=1)
    Ac = gi.CSR.from_scipy(A)
    a_ref = o.expectation(r.D_row_ptr, r.D_col, r.D_val, Ac)
    assert abs(gbe.gbe_expectation(g, Dt, gbe.DeviceCSR.from_host(Ac)) - a_ref) <= 1e-10 * np.abs(Ac.val).sum()
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_expectation(g, Dt, gbe.DeviceCSR.from_host(gi.chain(32, 4).H))
    assert e.value.status == -4


def test_error_norms_against_the_exact_projector(gbe):
    """Fig.2: max and Frobenius error of D against the exact projector, on the device; the oracle measures its own
    D against the same reference.  A random non-symmetric reference with a padded leading dimension catches a
    transposed or mis-strided lookup."""
    import torch
    s = gi.config(1)
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    Dx = o.o_diag(s.H, int(s.n_occ))
    Dt = torch.from_numpy(Dg).cuda()
    got = gbe.gbe_error_norms(g, Dt, torch.from_numpy(Dx).cuda())
    want = o.error_norms(r.D_row_ptr, r.D_col, r.D_val, Dx)
    tol = 4e-10 * np.sqrt(r.D_val.size * want[1]) + 1e-15
    assert abs(got[0] - want[0]) <= TOL_D and abs(got[1] - want[1]) <= tol and abs(got[2] - want[2]) <= tol
    assert abs(want[0] - 3.04e-4) < 2e-5  # the survey's probe value for config 1
    assert gbe.gbe_error_norms(g, Dt, torch.from_numpy(Dx).cuda()) == got  # reproducible
    rng = np.random.default_rng(3)
    R = rng.normal(size=(s.n, s.n))
    Rpad = torch.zeros(s.n, s.n + 24, dtype=torch.float64, device="cuda")
    Rpad[:, :s.n] = torch.from_numpy(R).cuda()
    got = gbe.gbe_error_norms(g, Dt, Rpad[:, :s.n])
    want = o.error_norms(r.D_row_ptr, r.D_col, r.D_val, R)
    assert abs(got[0] - want[0]) <= 1e-9 and abs(got[1] - want[1]) <= 1e-9 * want[1] and abs(got[2] - want[2]) <= 1e-9 * want[2]
    # shuffled communities: rows of D with many short runs of stored columns
    s2 = gi.random_banded(300, half_bw=5, n_part=11, seed=4, tau=1e-3, shuffle=True)
    g2, ex2, Dg2, _ = run_gpu(gbe, s2)
    _, r2 = run_oracle(s2)
    R2 = rng.normal(size=(s2.n, s2.n))
    got = gbe.gbe_error_norms(g2, torch.from_numpy(Dg2).cuda(), torch.from_numpy(R2).cuda())
    want = o.error_norms(r2.D_row_ptr, r2.D_col, r2.D_val, R2)
    assert abs(got[0] - want[0]) <= 1e-9 and abs(got[1] - want[1]) <= 1e-9 * want[1] and abs(got[2] - want[2]) <= 1e-9 * want[2]
    import ctypes as C
    out = (C.c_double * 3)()
    assert gbe.lib().gbe_error_norms(g.handle, Dt.data_ptr(), Rpad.data_ptr(), s.n - 1, None, out) == -1  # ld_ref < n


# ------------------------------------------------------------------------------- seeded random shapes
@pytest.mark.parametrize("case", range(24))
def test_random_shapes_and_partitions(gbe, case):
    """Seeded random banded Hamiltonians with random sizes (5 .. 330 orbitals: below one 8 x 8 sub-tile up to several
    64 x 64 tiles with ragged tails), bandwidths, thresholds, graph powers, and arbitrary partition vectors (unequal,
    non-contiguous, some communities empty).  Graph, halos, D pattern bit-exact; D within 1e-10."""
    rng = np.random.default_rng(1000 + case)
    n = int(rng.integers(5, 330))
    n_part = int(rng.integers(1, max(2, n // 3)))
    s = gi.random_banded(n, half_bw=int(rng.integers(1, 9)), n_part=n_part, seed=case, gap=float(rng.uniform(0.5, 3.0)),
                         tau=float(rng.choice([0.0, 1e-6, 1e-4, 1e-2, 0.3])), iters=int(rng.integers(3, 26)),
                         shuffle=bool(rng.integers(0, 2)))
    if case % 3 == 0:  # an arbitrary partition vector: unequal communities, possibly empty ones
        s.part = rng.integers(0, n_part, size=n).astype(np.int32)
    s.n_occ = float(rng.integers(0, n + 1)) if case % 5 == 0 else s.n_occ
    power = int(rng.integers(1, 4))
    graph, r = run_oracle(s, power=power)
    fits = None
    for sp2_path in (1, 2, 3):  # tiled kernels; the resident kernel where every community fits it; the packed kernel
        if sp2_path == 2 and not fits:
            continue
        g, ex, Dg, log = run_gpu(gbe, s, power=power, sp2_path=sp2_path)
        fits = g.info["resident_fits"]
        assert fits == (1 if 0 < g.info["max_m"] <= 160 else 0)
        check_structure(ex, graph, r, g.info)
        check_density(Dg, log, r)


# ------------------------------------------------------------------------------- degenerate shapes
def test_one_partition_equals_exact_projector(gbe):
    s = gi.config(1)
    s.part = np.zeros(s.n, np.int32)
    s.n_part = 1
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    D = sp.csr_matrix((Dg, ex["D_col"], ex["D_row_ptr"]), shape=(s.n, s.n)).toarray()
    assert abs(D - o.o_diag(s.H, 256)).max() < 1e-10
    assert abs(log.t1[-1] - s.n_occ) <= 1e-8  # north_star trace bar, attainable here (A-11)


def test_single_vertex_cores_and_empty_partitions(gbe):
    s = gi.chain(96, 96, tau=1e-3, iters=25)  # one vertex per core
    g, ex, Dg, log = run_gpu(gbe, s)
    graph, r = run_oracle(s)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    s2 = gi.random_banded(90, n_part=9, seed=11, tau=1e-3, iters=25)
    s2.part = (s2.part // 2 * 2).astype(np.int32)  # odd communities are empty
    g, ex, Dg, log = run_gpu(gbe, s2)
    graph, r = run_oracle(s2)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)
    assert (ex["ncore"][1::2] == 0).all()


@pytest.mark.parametrize("gather_path", [1, 2])
def test_missing_diagonal_entries(gbe, gather_path):
    s = gi.random_banded(64, half_bw=3, n_part=4, seed=8, tau=1e-3, iters=25)
    a = s.H.to_dense()
    a[np.arange(0, 64, 3), np.arange(0, 64, 3)] = 0.0  # not stored -> H_kk = 0 (A-12)
    H = gi.CSR.from_dense(a)
    assert H.nnz < s.H.nnz
    g, ex, Dg, log = run_gpu(gbe, s, H=H, gather_path=gather_path)
    graph, r = run_oracle(s, H=H)
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)


def test_h_may_change_between_build_and_density(gbe):
    """MD use: the graph fixes S, the communities and D's pattern; H values are read at gather time."""
    import torch
    s = gi.chain(256, 8, seed=0, tau=1e-4, iters=30)
    s_new = gi.chain(256, 8, seed=7, tau=1e-4, iters=30)
    Hd0, Hd1 = gbe.DeviceCSR.from_host(s.H), gbe.DeviceCSR.from_host(s_new.H)
    g = gbe.gbe_build_graph(Hd0, s.tau, None, s.n_part)
    Dg, log = gbe.gbe_density(Hd1, g, s.n_occ, s.iters)
    torch.cuda.synchronize()
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s_new.H, rp, ci, s.part, s.n_part, s.n_occ, s.iters)
    check_density(Dg.cpu().numpy(), log, r)


def test_density_host_and_phase_calls(gbe):
    import torch
    s = gi.chain(256, 8, tau=1e-4, iters=30)
    Hd = gbe.DeviceCSR.from_host(s.H)
    g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
    ws = g.new_workspace()
    D1, log1 = gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws)
    Dh, logh = gbe.gbe_density_host(s.H, g, s.n_occ, s.iters, workspace=ws, want_log=True)
    with pytest.raises(gbe.GbeError):
        gbe.gbe_density_host(None, g, s.n_occ, s.iters, workspace=ws)  # no H was left with a device-built graph
    gh = gbe.gbe_build_graph_host(s.H, s.tau, None, s.n_part)
    Dh2, _ = gbe.gbe_density_host(None, gh, s.n_occ, s.iters)           # one upload for build + density
    assert np.array_equal(Dh, Dh2)
    D3 = torch.empty_like(D1)
    gbe.gbe_gather(Hd, g, ws)
    gbe.gbe_sp2(g, s.n_occ, s.iters, -1.0, ws)
    gbe.gbe_scatter(g, ws, D3)
    log3 = gbe.gbe_read_log(g, ws)
    torch.cuda.synchronize()
    assert np.array_equal(D1.cpu().numpy(), Dh) and np.array_equal(D1.cpu().numpy(), D3.cpu().numpy())  # reproducible
    assert np.array_equal(log1.branch, logh.branch) and np.array_equal(log1.t1, log3.t1)


def test_side_stream_and_two_graphs_in_flight(gbe):
    """Everything is enqueued on the caller's stream: two systems on two non-default streams at once, results equal to
    the ones computed alone on the default stream."""
    import torch
    sa, sb = gi.chain(256, 8, seed=1, tau=1e-4, iters=30), gi.random_banded(180, n_part=6, seed=2, tau=1e-3, iters=25)
    ref = []
    for s in (sa, sb):
        g, ex, Dg, log = run_gpu(gbe, s, part=None)
        ref.append(Dg)
    st = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs, keep = [], []
    for s, stream in zip((sa, sb), st):
        with torch.cuda.stream(stream):
            Hd = gbe.DeviceCSR.from_host(s.H)
            g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part, stream=stream)
            ws = g.new_workspace()
            D = torch.empty(g.info["nnz_D"], dtype=torch.float64, device="cuda")
            keep.append((Hd, g, ws))
            outs.append(D)
    for _ in range(3):  # interleave enqueues on the two streams, no synchronisation in between
        for (Hd, g, ws), D, s, stream in zip(keep, outs, (sa, sb), st):
            gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws, D_val=D, want_log=False, stream=stream)
    torch.cuda.synchronize()
    for D, r in zip(outs, ref):
        assert np.array_equal(D.cpu().numpy(), r)  # same kernels, same reduction order: bit-identical


def test_tma_path_in_a_cuda_graph_and_with_two_workspaces(gbe):
    """The tiled kernel with panels by 2-D TMA (long K loops): its tensor maps are encoded once per graph and pointed at
    the dense buffers of each call ON THE DEVICE, so the call stays capturable, and the same graph handle can serve two
    workspaces in turn (each call re-points the maps) - results bit-identical to the eager run, and to the oracle."""
    import torch
    s = gi.water_box(256, 32, seed=3, tau=1e-5, iters=12)
    Hd = gbe.DeviceCSR.from_host(s.H)
    g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
    assert g.info["x2_tma"] == 1 and g.info["sp2_path_chosen"] == 1
    graph, r = run_oracle(s)
    ws_a, ws_b = g.new_workspace(), g.new_workspace()
    D_a = torch.empty(g.info["nnz_D"], dtype=torch.float64, device="cuda")
    D_b, D_c = torch.zeros_like(D_a), torch.zeros_like(D_a)
    gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws_a, D_val=D_a, want_log=False)
    gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws_b, D_val=D_b, want_log=False)   # same graph, other workspace
    gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws_a, D_val=D_c, want_log=False)   # and back, no sync in between
    torch.cuda.synchronize()
    assert torch.equal(D_a, D_b) and torch.equal(D_a, D_c)
    assert np.abs(D_a.cpu().numpy() - r.D_val).max() <= TOL_D
    side = torch.cuda.Stream()
    cg = torch.cuda.CUDAGraph()
    D_g = torch.zeros_like(D_a)
    with torch.cuda.stream(side):
        with torch.cuda.graph(cg, stream=side):
            gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws_b, D_val=D_g, want_log=False, stream=side)
    gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws_a, D_val=D_c, want_log=False)   # maps now point at ws_a ...
    torch.cuda.synchronize()
    for _ in range(2):
        D_g.zero_()
        cg.replay()                                                                         # ... the replay re-points them
        torch.cuda.synchronize()
        assert torch.equal(D_g, D_a)


@pytest.mark.parametrize("sp2_path", [0, 3])
def test_density_is_capturable_in_a_cuda_graph(gbe, sp2_path):
    """gbe_density without a log only enqueues kernels on the caller's stream (no allocation, no synchronisation, the
    branch decision stays on the device), so the whole SP2 loop can be captured once and replayed - the way to run
    launch-bound small systems (config 1: 82 launches of a few microseconds each)."""
    import torch
    s = gi.config(1)
    Hd = gbe.DeviceCSR.from_host(s.H)
    g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
    gbe.gbe_graph_set_sp2_path(g, sp2_path)
    ws = g.new_workspace()
    D_eager = torch.empty(g.info["nnz_D"], dtype=torch.float64, device="cuda")
    gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws, D_val=D_eager, want_log=False)
    torch.cuda.synchronize()
    D_graph = torch.zeros_like(D_eager)
    side = torch.cuda.Stream()
    cg = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(cg, stream=side):
            gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws, D_val=D_graph, want_log=False, stream=side)
    for _ in range(3):
        D_graph.zero_()
        cg.replay()
        torch.cuda.synchronize()
        assert torch.equal(D_graph, D_eager)
    # H may change between replays (values are read at gather time): replay after perturbing H in place
    Hd.val.mul_(1.0 + 1e-3)
    gbe.gbe_density(Hd, g, s.n_occ, s.iters, workspace=ws, D_val=D_eager, want_log=False)
    cg.replay()
    torch.cuda.synchronize()
    assert torch.equal(D_graph, D_eager)


def test_packed_kernel_launches_and_reproducibility(gbe):
    """The packed kernel (gbe_small.cu): ONE launch per SP2 iteration - every bin of launch n + 1 starts by summing the
    trace pairs launch n left (the same fixed order in every bin, so bitwise the same decision everywhere; one trace
    kernel after the last launch) - so 600 small communities (more than can be co-resident, no grid barrier possible)
    take 40 + 1 launches for the loop instead of 80."""
    import torch
    s = gi.chain(4800, 600, seed=5)
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, s.iters)
    Hd = gbe.DeviceCSR.from_host(s.H)
    g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
    assert g.info["sp2_path_chosen"] == 3 and g.info["n_small"] == 600 and 0 < g.info["n_bins"] <= 600
    n0 = gbe.gbe_launch_count()
    D0, log0 = gbe.gbe_density(Hd, g, s.n_occ, s.iters)
    torch.cuda.synchronize()
    assert gbe.gbe_launch_count() - n0 == 2 + 1 + 2 + s.iters + 1 + 1  # bounds(2), gather, init + trace of X_0, loop, final trace, scatter
    check_density(D0.cpu().numpy(), log0, r)
    for _ in range(10):
        D1, log1 = gbe.gbe_density(Hd, g, s.n_occ, s.iters)
        assert torch.equal(D0, D1) and np.array_equal(log0.t1, log1.t1) and np.array_equal(log0.t2, log1.t2)
    # a pre-determined sequence without trace logging on the packed path: no reduction at all between the products
    gbe.gbe_graph_set_sp2_path(g, 3)
    n0 = gbe.gbe_launch_count()
    Dp, logp = gbe.gbe_density_preset(Hd, g, r.branch, trace_every_iteration=False)
    torch.cuda.synchronize()
    assert gbe.gbe_launch_count() - n0 == 2 + 1 + 1 + s.iters + 1 + 1  # ..., init, loop, final trace, scatter
    assert np.abs(Dp.cpu().numpy() - r.D_val).max() <= TOL_D
    assert abs(logp.t1[-1] - r.t1[-1]) <= TOL_TR and abs(logp.t2[-1] - r.t2[-1]) <= TOL_TR


def test_resident_kernel_launches_and_choice(gbe):
    """The shared-memory-resident SP2 kernel (one launch for the whole loop) is what the library picks for config 1;
    both paths give the same D to rounding and each is bitwise reproducible."""
    import torch
    s = gi.config(1)
    Hd = gbe.DeviceCSR.from_host(s.H)
    g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
    assert g.info["resident_fits"] == 1 and g.info["resident_sp2"] == 1
    assert g.info["resident_cluster"] == 1  # 16 communities: one thread-block cluster, exchange through DSMEM
    n0 = gbe.gbe_launch_count()
    D_res, log_res = gbe.gbe_density(Hd, g, s.n_occ, s.iters)
    torch.cuda.synchronize()
    assert gbe.gbe_launch_count() - n0 == 2 + 1 + 1 + 1 + 1  # bounds(2), gather, state init, SP2 loop, scatter
    for _ in range(10):  # a race between the CTAs of the cluster or the warps of a CTA would show up as run-to-run noise
        D_res2, log2 = gbe.gbe_density(Hd, g, s.n_occ, s.iters)
        assert torch.equal(D_res, D_res2) and np.array_equal(log2.t1, log_res.t1) and np.array_equal(log2.t2, log_res.t2)
    gbe.gbe_graph_set_sp2_path(g, 1)
    n0 = gbe.gbe_launch_count()
    D_til, log_til = gbe.gbe_density(Hd, g, s.n_occ, s.iters)
    torch.cuda.synchronize()
    assert g.info["x2_tma"] == 0  # m = 48: short K loops, panels by cp.async
    assert gbe.gbe_launch_count() - n0 == 2 + 1 + 2 + 2 * s.iters + 1
    assert float((D_res - D_til).abs().max()) <= 1e-12
    live = np.abs(log_til.t1[:-1] - log_til.t2[:-1]) > 1e-9
    assert np.array_equal(log_res.branch[live], log_til.branch[live])
    # a water-box graph does not fit: the request is refused, the choice stays with the tiled kernels
    w = gi.water_box(64, 8)
    gw = gbe.gbe_build_graph(gbe.DeviceCSR.from_host(w.H), w.tau, None, w.n_part)
    assert gw.info["max_m"] > 160 and gw.info["resident_fits"] == 0 and gw.info["resident_sp2"] == 0
    with pytest.raises(gbe.GbeError):
        gbe.gbe_graph_set_sp2_path(gw, 2)


def test_resident_kernel_more_communities_than_sms(gbe):
    """600 communities of 8 sites: more CTAs than can be co-resident, so the trace-driven loop stays on the tiled kernels
    (the grid barrier needs every community on the device at once) while a pre-determined sequence without trace
    logging (no exchange between the subgraph expansions) runs the resident kernel as a plain launch."""
    import torch
    s = gi.chain(4800, 600, seed=5)
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, s.iters)
    Hd = gbe.DeviceCSR.from_host(s.H)
    g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
    assert g.info["resident_fits"] == 1 and g.info["resident_sp2"] == 0 and g.info["resident_cluster"] == 0
    Dg, log = gbe.gbe_density(Hd, g, s.n_occ, s.iters)
    torch.cuda.synchronize()
    check_density(Dg.cpu().numpy(), log, r)
    # 148 of these communities are co-resident: the cooperative launch with the exchange through L2, run to run identical
    s148 = gi.chain(1184, 148, seed=6)
    H148 = gbe.DeviceCSR.from_host(s148.H)
    g148 = gbe.gbe_build_graph(H148, s148.tau, None, s148.n_part)
    assert g148.info["resident_sp2"] == 1 and g148.info["resident_cluster"] == 0
    rp8, ci8 = o.build_graph(s148.H, s148.tau)
    r148 = o.o_sub(s148.H, rp8, ci8, s148.part, s148.n_part, s148.n_occ, s148.iters)
    D0, log0 = gbe.gbe_density(H148, g148, s148.n_occ, s148.iters)
    check_density(D0.cpu().numpy(), log0, r148)
    for _ in range(10):
        D1, log1 = gbe.gbe_density(H148, g148, s148.n_occ, s148.iters)
        assert torch.equal(D0, D1) and np.array_equal(log0.t1, log1.t1)
    gbe.gbe_graph_set_sp2_path(g, 2)
    n0 = gbe.gbe_launch_count()
    Dp, logp = gbe.gbe_density_preset(Hd, g, r.branch, trace_every_iteration=False)
    torch.cuda.synchronize()
    assert gbe.gbe_launch_count() - n0 == 2 + 1 + 1 + 1 + 1 + 1  # bounds(2), gather, init, SP2 loop, final trace, scatter
    assert np.abs(Dp.cpu().numpy() - r.D_val).max() <= TOL_D
    assert abs(logp.t1[-1] - r.t1[-1]) <= TOL_TR and abs(logp.t2[-1] - r.t2[-1]) <= TOL_TR


def test_resident_kernel_largest_community(gbe):
    """Communities at the capacity of the resident kernel (m up to 160: 64 work units, 210 KB of shared memory)."""
    s = gi.random_banded(1450, half_bw=6, n_part=10, seed=11, tau=1e-4, iters=25)
    graph, r = run_oracle(s)
    g, ex, Dg, log = run_gpu(gbe, s, sp2_path=2)
    assert g.info["max_m"] == 160
    check_structure(ex, graph, r, g.info)
    check_density(Dg, log, r)


@pytest.mark.parametrize("n", [2, 3, 9])
def test_tiny_matrices(gbe, n):
    s = gi.random_banded(n, half_bw=1, n_part=min(2, n), seed=n, tau=1e-3, iters=12)
    if n == 2:
        # Gershgorin bounds of a 2 x 2 matrix are symmetric about the mean eigenvalue, so at half filling the two
        # candidate traces tie EXACTLY in every iteration and rounding picks the branch (reading A-8): use another filling
        s.n_occ = 0.75
    graph, r = run_oracle(s)
    for sp2_path in (1, 2):
        g, ex, Dg, log = run_gpu(gbe, s, sp2_path=sp2_path)
        check_structure(ex, graph, r, g.info)
        check_density(Dg, log, r)


def test_errors(gbe):
    import torch
    s = gi.chain(64, 4)
    Hd = gbe.DeviceCSR.from_host(s.H)
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_build_graph(Hd, -1.0, None, 4)
    assert e.value.status == -1
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_build_graph(Hd, 1e-5, torch.full((64,), 9, dtype=torch.int32).cuda(), 4)
    assert e.value.status == -1  # partition id out of range
    a = s.H.to_dense()
    a[0, 1] += 0.5
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_build_graph(gbe.DeviceCSR.from_host(gi.CSR.from_dense(a)), 1e-5, None, 4, check_symmetry=True)
    assert e.value.status == -2
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_build_graph(gbe.DeviceCSR.from_host(gi.CSR.from_dense(np.zeros((4, 4)), keep_zeros=True)), 1e-5, None, 2)
    assert e.value.status == -3  # eps_max == eps_min
    # an H that is symmetric only to rounding (one entry off by one ulp) is refused by check_symmetry: with the default
    # power 2 only the upper triangle of floor(A A)_tau is formed, which is the whole product only for a bitwise symmetric A
    a = s.H.to_dense()
    a[3, 2] = np.nextafter(a[3, 2], 0.0)
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_build_graph(gbe.DeviceCSR.from_host(gi.CSR.from_dense(a)), 1e-5, None, 4, check_symmetry=True)
    assert e.value.status == -2
    g = gbe.gbe_build_graph(Hd, 1e-5, None, 4, check_symmetry=True)
    # a degenerate H (a multiple of I) given to gbe_density: reported through the log, D stays finite without one
    Hdeg = gbe.DeviceCSR.from_host(gi.CSR.from_dense(np.eye(64) * 0.25))
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_density(Hdeg, g, 32.0, 5)
    assert e.value.status == -3
    Ddeg, _ = gbe.gbe_density(Hdeg, g, 32.0, 5, want_log=False)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(Ddeg).all())
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_density(Hd, g, 32.0, 10, workspace=torch.empty(256, dtype=torch.uint8, device="cuda"))
    assert e.value.status == -5
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_density(Hd, g, 65.0, 10)
    assert e.value.status == -1
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_density(gbe.DeviceCSR.from_host(gi.chain(32, 4).H), g, 16.0, 10)
    assert e.value.status == -4


# ------------------------------------------------------------------------------- programmatic dependent launch
def test_dependent_launch_changes_when_kernels_start_not_what_they_compute(gbe):
    """include/gbe.h gbe_set_dependent_launch: the SP2 kernels of an iteration are launched as programmatic dependents of
    one another (the trace kernel waits for the X^2 launch and releases the next one after its decision; the bins of the
    packed kernel wait for the previous launch).  Switching that off must not change a single bit - tiled path (both X^2
    kernels: cp.async and TMA panels), packed path, with an idempotency stop in the middle of the loop, eagerly and
    replayed from a CUDA graph."""
    import torch
    cases = [(gi.config(2), dict(iters=40, idem_tol=-1.0)),              # 6,144 orbitals, TMA panels (mean m >= 360)
             (gi.config(1), dict(iters=60, idem_tol=1e-9)),              # chain, cp.async panels, stops on the device
             (gi.chain(4800, 600, seed=5), dict(iters=40, idem_tol=-1.0)),  # 600 small communities: packed kernel
             # mixed graph (m ~ 65 - 185): the tiled launch for the larger communities runs NEXT TO the packed launch of
             # the same iteration and synchronises with it through the published decision; stops on the device
             (gi.water_box(1024, 128, seed=0, tau=1e-3, iters=30), dict(iters=30, idem_tol=1e-7, paths=(1, 3)))]
    prev = gbe.gbe_set_dependent_launch(True)
    try:
        for s, kw in cases:
            Hd = gbe.DeviceCSR.from_host(s.H)
            part_t = torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
            g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
            for path in kw.get("paths", (1, 3) if g.info["n_small"] == s.n_part else (1,)):
                gbe.gbe_graph_set_sp2_path(g, path)
                out = {}
                for on in (True, False, True):
                    assert gbe.gbe_set_dependent_launch(on) in (True, False)
                    D, log = gbe.gbe_density(Hd, g, s.n_occ, kw["iters"], kw["idem_tol"])
                    torch.cuda.synchronize()
                    key = (D.clone(), log.t1.copy(), log.t2.copy(), log.branch.copy(), log.iters_done)
                    if on in out:
                        ref = out[on]
                    else:
                        out[on] = key
                        ref = out[True]
                    assert torch.equal(ref[0], key[0]) and np.array_equal(ref[1], key[1]) and np.array_equal(ref[2], key[2])
                    assert np.array_equal(ref[3], key[3]) and ref[4] == key[4]
                # replay from a CUDA graph captured with dependent launches on
                gbe.gbe_set_dependent_launch(True)
                ws = g.new_workspace()
                Dg = torch.empty(g.info["nnz_D"], dtype=torch.float64, device="cuda")
                st = torch.cuda.Stream()
                with torch.cuda.stream(st):
                    gbe.gbe_density(Hd, g, s.n_occ, kw["iters"], kw["idem_tol"], workspace=ws, D_val=Dg, want_log=False, stream=st)
                    st.synchronize()
                    cg = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(cg, stream=st):
                        gbe.gbe_density(Hd, g, s.n_occ, kw["iters"], kw["idem_tol"], workspace=ws, D_val=Dg, want_log=False,
                                        stream=st)
                    Dg.zero_()
                    cg.replay()
                    st.synchronize()
                assert torch.equal(Dg, out[True][0])
            g.free()
    finally:
        gbe.gbe_set_dependent_launch(prev)
