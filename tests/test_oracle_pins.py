"""Pins for the CPU oracle (CPU only).  Each test fixes a part of `oracle/` to something other than
itself: a closed form, a library special case, brute force by explicit loops, exact rational
arithmetic, or an invariant stated by the paper.  Citations: P:Lnn = paper line; A-n = DESIGN.md reading.
"""
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.sparse as sp

import gbe_inputs as gi
import oracle as o
from oracle.gbe_oracle import _branch

HERE = os.path.dirname(__file__)


def dense_D(r, n):
    return sp.csr_matrix((r.D_val, r.D_col, r.D_row_ptr), shape=(n, n)).toarray()


def pattern_mask(r, n):
    return sp.csr_matrix((np.ones_like(r.D_val), r.D_col, r.D_row_ptr), shape=(n, n)).toarray() > 0


# ----------------------------------------------------------------------------- step 0
def test_gershgorin_hand_example():
    # rows: 1 -+ (2+0.5) -> [-1.5, 3.5]; -3 -+ (2+1) -> [-6, 0]; (missing diagonal = 0, A-12) -+ 1.5 -> [-1.5, 1.5]
    a = np.array([[1.0, -2.0, 0.5], [-2.0, -3.0, 1.0], [0.5, 1.0, 0.0]])
    H = gi.CSR.from_dense(a)  # the zero diagonal is not stored
    assert H.nnz == 8
    lo, hi = o.gershgorin(H)
    assert lo == -6.0 and hi == 3.5


def test_x0_maps_spectrum_into_unit_interval_and_flips_order():
    s = gi.random_banded(64, seed=3)
    lo, hi = o.gershgorin(s.H)
    w = np.linalg.eigvalsh(s.H.to_dense())
    assert lo <= w.min() and w.max() <= hi
    X0 = o.normalised_x0(s.H, lo, hi).toarray()
    wx = np.linalg.eigvalsh(X0)
    assert wx.min() >= 0 and wx.max() <= 1
    # lowest H eigenvalue <-> largest X0 eigenvalue (occupied states go to 1)
    np.testing.assert_allclose(np.sort((hi - w) / (hi - lo)), wx, atol=1e-13)


# ----------------------------------------------------------------------------- step 1
def brute_graph(Hd, tau, power):
    """A-1 by explicit loops over dense arrays (no sparse library, no matmul)."""
    n = Hd.shape[0]
    lo = min(Hd[i, i] - sum(abs(Hd[i, j]) for j in range(n) if j != i) for i in range(n))
    hi = max(Hd[i, i] + sum(abs(Hd[i, j]) for j in range(n) if j != i) for i in range(n))
    X0 = [[((hi if i == j else 0.0) - Hd[i, j]) / (hi - lo) for j in range(n)] for i in range(n)]
    stored = [[(Hd[i, j] != 0.0) or i == j for j in range(n)] for i in range(n)]
    A = [[X0[i][j] if stored[i][j] and abs(X0[i][j]) >= tau else 0.0 for j in range(n)] for i in range(n)]
    keepA = [[stored[i][j] and abs(X0[i][j]) >= tau for j in range(n)] for i in range(n)]
    edges = {(i, i) for i in range(n)} | {(i, j) for i in range(n) for j in range(n) if keepA[i][j]}
    T = A
    for _ in range(2, power + 1):
        Tn = [[0.0] * n for _ in range(n)]
        for i in range(n):
            for j in range(n):
                s, touched = 0.0, False
                for k in range(n):
                    if keepA[i][k] and T[k][j] != 0.0:
                        s += A[i][k] * T[k][j]
                        touched = True
                if touched and abs(s) >= tau:
                    Tn[i][j] = s
                    edges.add((i, j))
        T = Tn
    return edges | {(j, i) for (i, j) in edges}


@pytest.mark.parametrize("power", [1, 2, 3])
@pytest.mark.parametrize("tau", [0.3, 1e-2, 1e-4])
def test_graph_brute_force(tau, power):
    s = gi.random_banded(14, half_bw=2, seed=power + 7)
    rp, ci = o.build_graph(s.H, tau, power=power)
    got = {(i, int(j)) for i in range(s.n) for j in ci[rp[i]:rp[i + 1]]}
    assert got == brute_graph(s.H.to_dense(), tau, power)


def brute_graph_diag_dropped(Hd, tau, power):
    """brute_graph with the MISTAKE the missing-diagonal branch of normalised_x0 guards against: an unstored H_kk
    treated as 'no entry of X0' (X0_kk = 0) instead of X0_kk = eps_max / (eps_max - eps_min) (A-12)."""
    n = Hd.shape[0]
    lo = min(Hd[i, i] - sum(abs(Hd[i, j]) for j in range(n) if j != i) for i in range(n))
    hi = max(Hd[i, i] + sum(abs(Hd[i, j]) for j in range(n) if j != i) for i in range(n))
    A = [[(((hi if i == j else 0.0) - Hd[i, j]) / (hi - lo)) if Hd[i, j] != 0.0 else 0.0 for j in range(n)] for i in range(n)]
    A = [[v if abs(v) >= tau else 0.0 for v in row] for row in A]
    edges = {(i, i) for i in range(n)} | {(i, j) for i in range(n) for j in range(n) if A[i][j] != 0.0}
    T = A
    for _ in range(2, power + 1):
        Tn = [[0.0] * n for _ in range(n)]
        for i in range(n):
            for j in range(n):
                s = sum(A[i][k] * T[k][j] for k in range(n) if A[i][k] != 0.0 and T[k][j] != 0.0)
                if abs(s) >= tau:
                    Tn[i][j] = s
                    edges.add((i, j))
        T = Tn
    return edges | {(j, i) for (i, j) in edges}


def test_unstored_diagonal_is_a_zero_of_H_not_of_X0():
    """A-12: a row of H without a stored diagonal has H_kk = 0, hence X0_kk = eps_max / (eps_max - eps_min) != 0.
    Pins the missing-diagonal branch of normalised_x0 (and through it build_graph) against explicit loops over the
    dense matrix.  The diagonal of A enters the VALUES of T^(2) = floor(A A)_tau on the pattern of A, so it decides edges
    from power 3 on (at power 2 a term A_ii A_ij needs A_ij != 0, an edge already): the test demands that dropping the
    diagonal WOULD change the graph, so that the branch is really exercised."""
    sensitive = 0
    for seed in range(6):
        s = gi.random_banded(14, half_bw=2, seed=40 + seed)
        Hd = s.H.to_dense()
        Hd[np.arange(0, 14, 2), np.arange(0, 14, 2)] = 0.0  # every other diagonal entry unstored
        H = gi.CSR.from_dense(Hd)
        assert H.nnz == s.H.nnz - 7
        lo, hi = o.gershgorin(H)
        X0 = o.normalised_x0(H, lo, hi).toarray()
        for i in range(14):
            for j in range(14):  # (eps_max delta_ij - H_ij) / (eps_max - eps_min), written out
                assert X0[i, j] == ((hi if i == j else 0.0) - Hd[i, j]) / (hi - lo)
        for power in (2, 3, 4):
            for tau in (0.05, 5e-3, 2e-3, 1e-3):
                rp, ci = o.build_graph(H, tau, power=power)
                got = {(i, int(j)) for i in range(14) for j in ci[rp[i]:rp[i + 1]]}
                assert got == brute_graph(Hd, tau, power)
                sensitive += got != brute_graph_diag_dropped(Hd, tau, power)
    assert sensitive >= 3


def test_graph_properties():
    s = gi.chain(64, 4)
    for tau in (1e-1, 1e-3, 1e-5):
        rp, ci = o.build_graph(s.H, tau)
        P = sp.csr_matrix((np.ones(ci.size), ci, rp), shape=(64, 64)).toarray() > 0
        assert P.diagonal().all()  # self loops (A-4, T^(0) = I P:L56)
        assert (P == P.T).all()
        for i in range(64):
            assert np.all(np.diff(ci[rp[i]:rp[i + 1]]) > 0)
    # tau > 1: nothing survives but the self loops (A-12)
    rp, ci = o.build_graph(s.H, 1.5)
    assert np.array_equal(ci, np.arange(64))
    # edges only grow as tau falls (obs. (ii) P:L65)
    sets = []
    for tau in (1e-1, 1e-2, 1e-3, 1e-4):
        rp, ci = o.build_graph(s.H, tau)
        sets.append({(i, int(j)) for i in range(64) for j in ci[rp[i]:rp[i + 1]]})
    assert all(a <= b for a, b in zip(sets, sets[1:]))
    # chain config 1: |i-j| <= 8 band at tau = 1e-5 (two hops of reach 4)
    s1 = gi.config(1)
    rp, ci = o.build_graph(s1.H, s1.tau)
    bw = max(abs(i - int(j)) for i in range(s1.n) for j in ci[rp[i]:rp[i + 1]])
    assert bw == 8


# ----------------------------------------------------------------------------- step 2
def test_subgraphs_and_pattern_brute_force():
    rng = np.random.default_rng(5)
    n, n_part = 40, 7  # partition 6 is left empty
    adj = rng.random((n, n)) < 0.08
    adj = adj | adj.T | np.eye(n, dtype=bool)
    S = sp.csr_matrix(adj)
    S.sort_indices()
    part = rng.integers(0, 6, n).astype(np.int32)
    subs = o.subgraphs(S.indptr, S.indices, part, n_part)
    assert len(subs) == n_part and subs[6][1] == 0 and subs[6][0].size == 0
    owner_seen = np.zeros(n, int)
    pat = np.zeros((n, n), bool)
    for p, (idx, nc) in enumerate(subs):
        core = [i for i in range(n) if part[i] == p]
        halo = sorted({k for i in core for k in range(n) if adj[k, i]} - set(core))
        assert list(idx[:nc]) == core and list(idx[nc:]) == halo  # core first, both ascending
        owner_seen[core] += 1
        for k in core + halo:
            for i in core:
                pat[k, i] = True
    assert (owner_seen == 1).all()  # every vertex in exactly one core
    rp, ci = o.density_pattern(subs, n)
    got = sp.csr_matrix((np.ones(ci.size), ci, rp), shape=(n, n)).toarray() > 0
    assert (got == pat).all()
    assert (got | ~adj).all()  # S is a subset of S' (extra edges are harmless, obs. (iii) P:L65)


# ----------------------------------------------------------------------------- exact projector
def test_o_diag_closed_form_uniform_ring():
    # uniform periodic nearest-neighbour ring, odd filling: D_ij = sin(pi n_occ d/N) / (N sin(pi d/N))
    N, n_occ = 30, 11
    s = gi.chain(N, 1, reach=1, noise=0.0, periodic=True, alternate=False)
    D = o.o_diag(s.H, n_occ)
    d = (np.arange(N)[:, None] - np.arange(N)[None, :]) % N
    with np.errstate(invalid="ignore", divide="ignore"):
        ref = np.sin(np.pi * n_occ * d / N) / (N * np.sin(np.pi * d / N))
    ref[d == 0] = n_occ / N
    np.testing.assert_allclose(D, ref, atol=1e-13)


def test_o_diag_invariants():
    s = gi.random_banded(80, seed=2)
    D = o.o_diag(s.H, 40)
    Hd = s.H.to_dense()
    assert abs(D - D.T).max() < 1e-14
    assert abs(D @ D - D).max() < 1e-13
    assert abs(np.trace(D) - 40) < 1e-12
    assert abs(Hd @ D - D @ Hd).max() < 1e-12


# ----------------------------------------------------------------------------- SP2 special cases
def test_two_level_closed_form():
    # H = [[a, b], [b, -a]], n_occ = 1: D = (I - H / sqrt(a^2 + b^2)) / 2
    a, b = 0.7, -0.4
    H = gi.CSR.from_dense(np.array([[a, b], [b, -a]]))
    rp, ci = o.build_graph(H, 0.0)
    r = o.o_sub(H, rp, ci, np.zeros(2, np.int32), 1, 1.0, 40)
    ref = 0.5 * (np.eye(2) - np.array([[a, b], [b, -a]]) / np.hypot(a, b))
    np.testing.assert_allclose(dense_D(r, 2), ref, atol=1e-14)


def test_branch_tie_takes_2x_minus_x2_hand_worked():
    """A-6: a tie of the two next-trace errors goes to 2X - X^2.  Hand-worked, every number exact in binary:
    H = diag(-1, 0, 1), no off-diagonals: eps_min = -1, eps_max = 1, X0 = diag(1, 1/2, 0); t1 = 3/2, t2 = 5/4.
    n_occ = 3/2: |t2 - n_occ| = 1/4 = |2 t1 - t2 - n_occ| -> tie -> branch 1: X1 = diag(1, 3/4, 0), t1 = 7/4, t2 = 25/16.
    (The other direction would give X1 = diag(1, 1/4, 0), t1 = 5/4.)  Then |25/16 - 3/2| = 1/16 < |7/2 - 25/16 - 3/2| = 7/16
    -> branch 0: X2 = diag(1, 9/16, 0)."""
    assert _branch(1.0, 0.5, 1.0) == 1  # |0.5 - 1| == |2 - 0.5 - 1|
    assert _branch(1.5, 1.25, 1.5) == 1
    H = gi.CSR.from_dense(np.diag([-1.0, 1e-300, 1.0]))  # the middle diagonal entry stored (value ~ 0)
    rp, ci = o.build_graph(H, 1e-5)
    for n_part, part in ((1, np.zeros(3, np.int32)), (3, np.arange(3, dtype=np.int32))):
        r = o.o_sub(H, rp, ci, part, n_part, 1.5, 2)
        assert (r.eps_min, r.eps_max) == (-1.0, 1.0)
        assert list(r.branch) == [1, 0]
        assert list(r.t1) == [1.5, 1.75, 1.5625] and list(r.t2[:2]) == [1.25, 1.5625]
        np.testing.assert_array_equal(np.diag(dense_D(r, 3)), [1.0, 0.5625, 0.0])


@pytest.mark.parametrize("system", ["chain", "banded"])
def test_one_partition_equals_eigendecomposition(system):
    s = gi.config(1) if system == "chain" else gi.random_banded(96, seed=1)
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, np.zeros(s.n, np.int32), 1, s.n_occ, 40)
    D = o.o_diag(s.H, int(s.n_occ))
    assert abs(dense_D(r, s.n) - D).max() < 1e-12
    assert abs(r.t1[-1] - s.n_occ) < 1e-8  # north_star trace bar holds here (A-11)


def test_complete_graph_any_partition_equals_eigendecomposition():
    s = gi.random_banded(48, seed=4, n_part=5, shuffle=True)
    n = s.n
    rp = np.arange(n + 1, dtype=np.int64) * n
    ci = np.tile(np.arange(n, dtype=np.int32), n)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, 40)
    assert abs(dense_D(r, n) - o.o_diag(s.H, n // 2)).max() < 1e-12
    # tau = 0 on a dense H gives the complete graph from build_graph itself
    Hd = s.H.to_dense() + 1e-3
    Hfull = gi.CSR.from_dense(Hd)
    rp2, ci2 = o.build_graph(Hfull, 0.0)
    assert np.array_equal(rp2, rp) and np.array_equal(ci2, ci)


# ----------------------------------------------------------------------------- Eq.(5) == Eq.(6)
def _toy(n=12, half_bw=2, seed=0):
    rng = np.random.default_rng(seed)
    a = np.zeros((n, n))
    for d in range(1, half_bw + 2):  # H reaches one further than the graph: x[s] != masked X (A-2)
        v = np.round(rng.normal(scale=0.4, size=n - d), 3)
        a[np.arange(n - d), np.arange(d, n)] = v
    a = a + a.T + np.diag(np.round(rng.normal(size=n), 3))
    return a


@pytest.mark.parametrize("communities", [1, 3])
def test_eq5_exact_rational_equals_subgraph_expansion(communities):
    """Brute force in exact rationals: the globally thresholded recurrence Eq.(5) (unmasked X on the left,
    pattern S') equals the partitioned subgraph expansion Eq.(6), entry for entry."""
    n = 12
    a = _toy(n)
    H = gi.CSR.from_dense(a)
    lo, hi = o.gershgorin(H)
    # band graph |i-j| <= 2 (any S is allowed: obs. (viii) P:L65)
    adj = np.abs(np.arange(n)[:, None] - np.arange(n)[None, :]) <= 2
    S = sp.csr_matrix(adj)
    S.sort_indices()
    part = (np.arange(n) // communities).astype(np.int32)
    n_part = n // communities
    branches = [1, 0, 1, 1]
    r = o.o_sub(H, S.indptr, S.indices, part, n_part, n / 2, 4, replay=(branches, 4), keep_blocks=True)
    X0 = o.normalised_x0(H, lo, hi).toarray()
    P = o.o_eq5_exact(X0, r.subs, branches)
    Pf = np.array([[float(P[i, j]) for j in range(n)] for i in range(n)])
    got = dense_D(r, n)
    assert abs(got - Pf).max() < 5e-15
    mask = pattern_mask(r, n)
    assert all(P[i, j] == 0 for i in range(n) for j in range(n) if not mask[i, j])  # obs. (iv) P:L65
    assert abs(Pf - Pf.T).max() > 1e-4  # P_tau is not symmetric (obs. (i) P:L65)
    # the truly exact statement: redo the subgraph polynomial in rationals and compare with ==
    c = o.sp2_polynomial_coeffs(branches)
    for idx, nc in r.subs:
        m = len(idx)
        x = [[Fraction(X0[idx[i], idx[j]]) for j in range(m)] for i in range(m)]
        pw = [[Fraction(int(i == j)) for j in range(m)] for i in range(m)]
        acc = [[c[0] * pw[i][j] for j in range(m)] for i in range(m)]
        for deg in range(1, len(c)):
            pw = [[sum(x[i][k] * pw[k][j] for k in range(m)) for j in range(m)] for i in range(m)]
            for i in range(m):
                for j in range(m):
                    acc[i][j] += c[deg] * pw[i][j]
        for cc in range(nc):
            for rr in range(m):
                assert acc[rr][cc] == P[idx[rr], idx[cc]]


def test_eq5_nested_float_more_iterations():
    s = gi.chain(96, 6, tau=1e-3)
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, 10)
    lo, hi = o.gershgorin(s.H)
    X0 = o.normalised_x0(s.H, lo, hi).toarray()
    P = o.o_eq5_nested(X0, r.subs, list(r.branch))
    assert abs(dense_D(r, s.n) - P).max() < 1e-13


def test_masked_global_sp2_is_not_the_target():
    """Finding 1 / obs. (ix) P:L65: X <- floor(X X)_S differs from P_tau at the size of the truncation error."""
    n = 12
    a = _toy(n)
    H = gi.CSR.from_dense(a)
    lo, hi = o.gershgorin(H)
    adj = np.abs(np.arange(n)[:, None] - np.arange(n)[None, :]) <= 2
    S = sp.csr_matrix(adj)
    S.sort_indices()
    branches = [1, 0, 1, 1]
    r = o.o_sub(H, S.indptr, S.indices, np.arange(n, dtype=np.int32), n, n / 2, 4, replay=(branches, 4))
    X = o.normalised_x0(H, lo, hi).toarray()
    for b in branches:
        Y = np.where(adj, X @ X, 0.0)
        X = Y if b == 0 else 2 * X - Y
    assert abs(np.where(adj, X, 0) - dense_D(r, n)).max() > 1e-4


def test_sp2_polynomial_and_order():
    br = [1, 0, 0, 1, 1, 0]
    c = o.sp2_polynomial_coeffs(br)
    assert len(c) - 1 == 2 ** len(br)
    for x in (Fraction(0), Fraction(1), Fraction(1, 3), Fraction(7, 9)):
        y = x
        for b in br:
            y = y * y if b == 0 else 2 * y - y * y
        assert sum(ck * x ** k for k, ck in enumerate(c)) == y
    iters, order, bar = map(int, open(os.path.join(HERE, "golden", "sp2_order.txt")).read().split())
    assert 2 ** iters == order and order > bar  # 'over a billion in only 30 iterations'


# ----------------------------------------------------------------------------- invariants / metamorphic
def test_per_iteration_invariants():
    s = gi.config(1)
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, 30, keep_blocks=True)
    assert r.iters_done == 30 and r.t1.size == 31 and r.branch.size == 30
    for n in range(30):
        assert -1e-12 <= r.t2[n] <= r.t1[n] + 1e-12  # spectrum of every x_p in [0,1] (A-5)
        nxt = r.t1[n + 1]
        if r.branch[n] == 0:
            assert abs(nxt - r.t2[n]) < 1e-9 and nxt <= r.t1[n] + 1e-12  # X^2 never raises the trace
        else:
            assert abs(nxt - (2 * r.t1[n] - r.t2[n])) < 1e-9 and nxt >= r.t1[n] - 1e-12
    for x in r.blocks:
        assert abs(x - x.T).max() < 1e-13  # each dense polynomial stays symmetric
    D, mask = dense_D(r, s.n), pattern_mask(r, s.n)
    assert abs(D - D.T).max() > 1e-5  # assembled P_tau is not symmetric (obs. (i))
    assert abs(D[~mask]).max() == 0


def test_direct_sum_uses_one_joint_sequence():
    a, b = gi.chain(64, 4, seed=1), gi.random_banded(48, n_part=3, seed=2, tau=1e-4)
    Hd = np.zeros((112, 112))
    Hd[:64, :64] = a.H.to_dense()
    Hd[64:, 64:] = 3.0 + b.H.to_dense()
    H = gi.CSR.from_dense(Hd)
    part = np.concatenate([a.part, 4 + b.part]).astype(np.int32)
    bounds = o.gershgorin(H)
    rp, ci = o.build_graph(H, 1e-4)
    n_occ = 50.0
    r = o.o_sub(H, rp, ci, part, 7, n_occ, 35)
    D = dense_D(r, 112)
    assert abs(D[:64, 64:]).max() == 0 and abs(D[64:, :64]).max() == 0
    # each block separately, forced to the JOINT bounds and branch sequence (Eq.(4): one polynomial)
    Ha, Hb = gi.CSR.from_dense(Hd[:64, :64]), gi.CSR.from_dense(Hd[64:, 64:])
    Sa = sp.csr_matrix(sp.csr_matrix((np.ones(ci.size), ci, rp), shape=(112, 112))[:64, :64])
    Sb = sp.csr_matrix(sp.csr_matrix((np.ones(ci.size), ci, rp), shape=(112, 112))[64:, 64:])
    for S_ in (Sa, Sb):
        S_.sort_indices()
    ra = o.o_sub(Ha, Sa.indptr, Sa.indices, a.part, 4, 0, 35, replay=(r.branch, 35), bounds=bounds)
    rb = o.o_sub(Hb, Sb.indptr, Sb.indices, b.part, 3, 0, 35, replay=(r.branch, 35), bounds=bounds)
    assert abs(D[:64, :64] - dense_D(ra, 64)).max() < 1e-13
    assert abs(D[64:, 64:] - dense_D(rb, 48)).max() < 1e-13
    assert abs(r.t1[-1] - (ra.t1[-1] + rb.t1[-1])) < 1e-10


def test_relabelling_permutes_D():
    s = gi.random_banded(72, n_part=6, seed=9, tau=1e-3)
    rng = np.random.default_rng(0)
    perm = rng.permutation(s.n)  # new label of old vertex v is inv[v]; row i of the new H is old row perm[i]
    Hp = gi.CSR.from_dense(s.H.to_dense()[np.ix_(perm, perm)])
    rp, ci = o.build_graph(s.H, s.tau)
    rpp, cip = o.build_graph(Hp, s.tau)
    # stop at convergence: iterating past it doubles roundoff per step (A-7)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, 40, idem_tol=1e-10)
    rq = o.o_sub(Hp, rpp, cip, s.part[perm], s.n_part, s.n_occ, 40, idem_tol=1e-10)
    assert np.array_equal(r.branch, rq.branch) and r.iters_done < 40
    assert abs(dense_D(r, s.n)[np.ix_(perm, perm)] - dense_D(rq, s.n)).max() < 1e-12


def test_local_order_is_roundoff_only():
    s = gi.config(1)
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, s.iters)
    q = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, s.iters, local_perm_seed=1)
    assert np.array_equal(r.branch, q.branch)
    assert abs(r.D_val - q.D_val).max() < 1e-12  # the noise floor the GPU parity bar (1e-10) sits above


def test_idem_tol_stops_early_and_matches_fixed_count():
    s = gi.config(1)
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, 60, idem_tol=1e-9)
    assert 15 < r.iters_done < 40 and r.t1.size == r.iters_done + 1
    assert abs(r.t1[-1] - r.t2[-1]) <= 1e-9
    q = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, r.iters_done)
    assert np.array_equal(r.D_val, q.D_val)


def test_error_falls_with_tau_and_is_insensitive_to_partition_count():
    s = gi.config(1)
    D = o.o_diag(s.H, 256)
    errs = []
    for tau in (1e-2, 1e-3, 1e-4, 1e-5, 1e-6):
        rp, ci = o.build_graph(s.H, tau)
        r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, 40)
        errs.append(abs(dense_D(r, s.n) - D)[pattern_mask(r, s.n)].max())
    assert all(a > b for a, b in zip(errs[:4], errs[1:4])) and errs[4] <= errs[3]  # obs. (ii) P:L65; the power-2 graph saturates at |i-j| <= 8
    rp, ci = o.build_graph(s.H, 1e-5)
    e = []
    for n_part in (8, 16, 64):
        r = o.o_sub(s.H, rp, ci, gi.contiguous_partition(s.n, n_part), n_part, s.n_occ, 40)
        e.append(abs(dense_D(r, s.n) - D)[pattern_mask(r, s.n)].max())
    assert max(e) / min(e) < 5  # 'fairly insensitive to the number of graph partitions'
    assert abs(errs[3] - 3.04e-4) < 2e-5  # survey probe value for config 1


# ------------------------------------------------------------------------------- observables
def test_expectation_band_energy_is_the_sum_of_occupied_eigenvalues():
    """Closed form: for the exact projector Tr[D H] = sum of the n_occ lowest eigenvalues; Tr[D I] = n_occ."""
    s = gi.random_banded(60, half_bw=4, n_part=4, seed=2)
    Hd = s.H.to_dense()
    D = o.o_diag(s.H, 30)
    Dc = gi.CSR.from_dense(D, keep_zeros=True)
    e = o.expectation(Dc.row_ptr, Dc.col_idx, Dc.val, s.H)
    assert abs(e - np.linalg.eigvalsh(Hd)[:30].sum()) < 1e-10
    assert abs(o.expectation(Dc.row_ptr, Dc.col_idx, Dc.val, np.eye(60)) - 30.0) < 1e-10


def test_expectation_uses_the_transpose_of_a_nonsymmetric_operand():
    """Tr[D A] = sum_ki D_ki A_ik, by explicit loops on a non-symmetric D (the assembled P_tau, obs. (i)) and a
    non-symmetric A - a transposed operand or a dropped off-pattern term would change the value."""
    rng = np.random.default_rng(5)
    n = 9
    D = rng.normal(size=(n, n)) * (rng.uniform(size=(n, n)) < 0.5)
    A = rng.normal(size=(n, n)) * (rng.uniform(size=(n, n)) < 0.6)
    want = sum(D[k, i] * A[i, k] for k in range(n) for i in range(n))
    Dc, Ac = gi.CSR.from_dense(D), gi.CSR.from_dense(A)
    assert abs(o.expectation(Dc.row_ptr, Dc.col_idx, Dc.val, Ac) - want) < 1e-13
    assert abs(want - np.trace(D @ A)) < 1e-13
    assert abs(o.expectation(Dc.row_ptr, Dc.col_idx, Dc.val, Ac) - np.trace(D @ A.T)) > 1e-3


def test_error_norms_on_a_hand_worked_example():
    """Fig.2: Frobenius norm of the density-matrix error.  3 x 3 example worked by hand: D stores (0,0)=1, (0,2)=2,
    (1,1)=-1, (2,0)=0 (a stored zero counts as stored); the reference is [[1.5,0.25,2],[0,-1,0.5],[3,0,0.125]]."""
    rp, col, val = np.array([0, 2, 3, 4]), np.array([0, 2, 1, 0]), np.array([1.0, 2.0, -1.0, 0.0])
    ref = np.array([[1.5, 0.25, 2.0], [0.0, -1.0, 0.5], [3.0, 0.0, 0.125]])
    mx, f_in, f_all = o.error_norms(rp, col, val, ref)
    assert mx == 3.0                                   # entry (2,0): |0 - 3|
    assert f_in == 0.25 + 0.0 + 0.0 + 9.0               # stored entries: (0,0), (0,2), (1,1), (2,0)
    assert f_all == 9.25 + 0.0625 + 0.25 + 0.015625     # + what the reference holds where D stores nothing
    # a transposed pattern or a transposed reference changes all three
    assert o.error_norms(rp, col, val, ref.T) != (mx, f_in, f_all)


def test_error_norms_full_norm_is_the_dense_frobenius_norm_and_falls_with_tau():
    """Against numpy's norm of the dense difference, on the chain: obs. (ii) P:L65, the error falls as tau falls."""
    s = gi.chain(128, 8)
    Dx = o.o_diag(s.H, 64)
    prev = None
    for tau in (1e-2, 1e-4, 1e-6):
        rp, ci = o.build_graph(s.H, tau)
        r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, 40)
        mx, f_in, f_all = o.error_norms(r.D_row_ptr, r.D_col, r.D_val, Dx)
        Dd = sp.csr_matrix((r.D_val, r.D_col, r.D_row_ptr), shape=(s.n, s.n)).toarray()
        assert abs(f_all - np.linalg.norm(Dd - Dx, "fro") ** 2) <= 1e-12 * max(1.0, f_all)
        assert f_in <= f_all and mx ** 2 <= f_in * (1 + 1e-12)
        assert prev is None or f_all < prev
        prev = f_all


# ------------------------------------------------------------------------------- Eq.(8): graph of the next MD step
def test_update_graph_is_paths_of_length_two_by_brute_force():
    """S = every (i, j) joined by a path of length <= 2 in M = I u pat(|D| >= tau) u pat(H), symmetrised - explicit loops."""
    rng = np.random.default_rng(3)
    n = 14
    Hd = np.zeros((n, n))
    for i in range(n - 1):
        Hd[i, i + 1] = Hd[i + 1, i] = -1.0
    Hd[np.arange(n), np.arange(n)] = rng.normal(size=n)
    D = rng.normal(size=(n, n)) * (rng.uniform(size=(n, n)) < 0.15)      # not symmetric, some entries below tau
    D[np.abs(D) < 0.05] *= 1e-3
    tau = 1e-2
    H, Dc = gi.CSR.from_dense(Hd), gi.CSR.from_dense(D)
    rp, ci = o.update_graph(Dc.row_ptr, Dc.col_idx, Dc.val, H, tau)
    M = (np.abs(D) >= tau) | (Hd != 0) | np.eye(n, dtype=bool)
    want = np.zeros((n, n), dtype=bool)
    for i in range(n):
        for k in range(n):
            if M[i, k]:
                for j in range(n):
                    if M[k, j]:
                        want[i, j] = True
    want |= want.T
    got = np.zeros((n, n), dtype=bool)
    for i in range(n):
        got[i, ci[rp[i]:rp[i + 1]]] = True
    assert np.array_equal(got, want)
    assert (got & M).sum() == M.sum()          # S contains M (self loops make every edge a path of length two)
    assert np.all(np.diff(ci[rp[3]:rp[4]]) > 0)


def test_update_graph_follows_the_previous_density_matrix():
    """S(t) 'cannot increase by more than paths of length two between two MD steps' - with H unchanged and the
    previous D on the previous graph, every new edge is a path of length two of old edges and H edges; and a density
    matrix computed on the updated graph is at least as accurate as on the old one (extra edges are harmless, obs. (iii))."""
    s = gi.chain(128, 8, tau=1e-3, iters=30)
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, s.iters)
    rp2, ci2 = o.update_graph(r.D_row_ptr, r.D_col, r.D_val, s.H, 1e-4)
    n = s.n
    old = sp.csr_matrix((np.ones(ci.size), ci, rp), shape=(n, n)).toarray() > 0
    Dpat = sp.csr_matrix((np.ones(r.D_col.size), r.D_col, r.D_row_ptr), shape=(n, n)).toarray() > 0
    new = sp.csr_matrix((np.ones(ci2.size), ci2, rp2), shape=(n, n)).toarray() > 0
    reach = (Dpat | (s.H.to_dense() != 0) | np.eye(n, dtype=bool)).astype(int)
    two = (reach @ reach) > 0
    assert not (new & ~(two | two.T)).any()
    r2 = o.o_sub(s.H, rp2, ci2, s.part, s.n_part, s.n_occ, s.iters)
    exact = o.o_diag(s.H, int(s.n_occ))
    def err(res):
        D = sp.csr_matrix((res.D_val, res.D_col, res.D_row_ptr), shape=(n, n)).toarray()
        mask = sp.csr_matrix((np.ones(res.D_col.size), res.D_col, res.D_row_ptr), shape=(n, n)).toarray() > 0
        return np.abs((D - exact)[mask]).max()
    assert err(r2) <= err(r) * 1.01


# ------------------------------------------------------------------------------- Eq.(7): finite-temperature expansion
def test_fermi_coefficients_reproduce_the_fermi_function():
    """Closed form: sum_n c_n T_n(x) -> f(x) pointwise; the coefficients of a smooth f decay geometrically, so with
    order 400 at beta*a = 20 the series equals the Fermi function to 1e-12 on a grid of x (numpy's chebval)."""
    lo, hi, mu, beta = -3.0, 5.0, 0.4, 5.0
    c = o.fermi_chebyshev_coeffs(mu, beta, 400, lo, hi)
    x = np.linspace(-1, 1, 201)
    a, b = 0.5 * (hi - lo), 0.5 * (hi + lo)
    f = 1.0 / (1.0 + np.exp(beta * (a * x + b - mu)))
    assert np.abs(np.polynomial.chebyshev.chebval(x, c) - f).max() < 1e-12
    assert abs(c[0] - np.mean(1.0 / (1.0 + np.exp(beta * (a * np.cos(np.pi * (np.arange(4096) + 0.5) / 4096) + b - mu))))) < 1e-13


def test_o_fermi_one_partition_equals_the_fermi_function_of_the_eigenvalues():
    """Library special case: one partition => D = V f(eps) V^T from the dense eigendecomposition, to within the
    truncation bound sum_{n > order} |c_n| of the Chebyshev series (plus roundoff)."""
    s = gi.random_banded(72, half_bw=5, n_part=1, seed=4)
    mu, beta, order = 0.1, 3.0, 120
    rp, ci = o.build_graph(s.H, 0.0)
    r = o.o_fermi(s.H, rp, ci, s.part, 1, mu, beta, order)
    w, v = np.linalg.eigh(s.H.to_dense())
    exact = (v * (1.0 / (1.0 + np.exp(beta * (w - mu))))) @ v.T
    D = sp.csr_matrix((r.D_val, r.D_col, r.D_row_ptr), shape=(s.n, s.n)).toarray()
    tail = np.abs(o.fermi_chebyshev_coeffs(mu, beta, 600, r.eps_min, r.eps_max)[order + 1:]).sum()
    assert tail < 1e-6
    assert np.linalg.norm(D - exact, 2) <= tail + 1e-12
    assert abs(r.n_elec - (1.0 / (1.0 + np.exp(beta * (w - mu)))).sum()) <= s.n * (tail + 1e-12)
    assert np.abs(D - D.T).max() < 1e-13


def test_o_fermi_reaches_the_zero_temperature_projector_and_respects_the_graph():
    """beta -> large with mu in the gap: the Fermi operator tends to theta(mu - H), so the partitioned
    finite-temperature result approaches the partitioned SP2 result; and P_tau is zero outside S' (obs. (iv))."""
    s = gi.chain(96, 6, tau=1e-3, iters=30)
    rp, ci = o.build_graph(s.H, s.tau)
    rs = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, s.iters)
    w = np.linalg.eigvalsh(s.H.to_dense())
    mu = 0.5 * (w[47] + w[48])
    rf = o.o_fermi(s.H, rp, ci, s.part, s.n_part, mu, 40.0, 600)
    assert np.array_equal(rf.D_row_ptr, rs.D_row_ptr) and np.array_equal(rf.D_col, rs.D_col)
    assert np.abs(rf.D_val - rs.D_val).max() < 1e-6
    assert abs(rf.n_elec - rs.t1[-1]) < 1e-5


# ----------------------------------------------------------------------------- one community at a time
@pytest.mark.parametrize("tau", [0.2, 1e-2, 1e-4])
def test_one_community_brute_force(tau):
    """OneCommunity against explicit loops: the subgraph from the brute-force edge set of A-1 (no sparse library, no
    matmul) and the expansion of the dense principal submatrix with the given branches by triple loops."""
    s = gi.random_banded(14, half_bw=2, n_part=4, seed=11, shuffle=True)
    Hd = s.H.to_dense()
    n = s.n
    edges = brute_graph(Hd, tau, 2)
    lo = min(Hd[i, i] - sum(abs(Hd[i, j]) for j in range(n) if j != i) for i in range(n))
    hi = max(Hd[i, i] + sum(abs(Hd[i, j]) for j in range(n) if j != i) for i in range(n))
    branch = [1, 0, 0, 1, 1]
    oc = o.OneCommunity(s.H, tau, s.part)
    for p in range(s.n_part):
        core = [i for i in range(n) if s.part[i] == p]
        halo = sorted({k for i in core for k in range(n) if (k, i) in edges} - set(core))
        idx, nc, cols = oc.expand(p, branch, len(branch))
        assert list(idx) == core + halo and nc == len(core)
        sidx = core + halo
        m = len(sidx)
        X = [[((hi if a == b else 0.0) - Hd[sidx[a], sidx[b]]) / (hi - lo) for b in range(m)] for a in range(m)]
        for b_n in branch:
            Y = [[sum(X[a][k] * X[k][b] for k in range(m)) for b in range(m)] for a in range(m)]
            X = Y if b_n == 0 else [[2.0 * X[a][b] - Y[a][b] for b in range(m)] for a in range(m)]
        want = np.array(X).reshape(m, m)[:, :nc]
        assert np.abs(cols - want).max() <= 1e-13


@pytest.mark.parametrize("system", ["chain", "water", "shuffled"])
def test_one_community_equals_the_whole_batch(system):
    """Every community of a small system, one at a time with the sequence the whole batch chose, reproduces o_sub's block:
    same subgraph (bit for bit) and the same core columns."""
    s = {"chain": lambda: gi.config(1),
         "water": lambda: gi.water_box(48, 6, seed=2, tau=1e-4, iters=12),
         "shuffled": lambda: gi.random_banded(120, half_bw=4, n_part=5, seed=4, tau=1e-3, iters=10, shuffle=True)}[system]()
    rp, ci = o.build_graph(s.H, s.tau)
    r = o.o_sub(s.H, rp, ci, s.part, s.n_part, s.n_occ, s.iters, keep_blocks=True)
    oc = o.OneCommunity(s.H, s.tau, s.part)
    assert (oc.lo, oc.hi) == (r.eps_min, r.eps_max)
    for p in range(s.n_part):
        idx, nc, cols = oc.expand(p, r.branch, r.iters_done)
        assert np.array_equal(idx, r.subs[p][0]) and nc == r.subs[p][1]
        assert np.abs(cols - r.blocks[p][:, :nc]).max() <= 1e-14
