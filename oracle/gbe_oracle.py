"""Plain, slow, obviously-correct CPU implementation (float64) of the hot path.

TEST INFRASTRUCTURE ONLY - see oracle/__init__.py for who may import this and for the pins.
Shares no code with the CUDA path.  `H` arguments are duck-typed CSR objects with the fields
`n, row_ptr (int64), col_idx (int32, ascending in a row), val (float64)`.

Citations: `P:Lnn` = line nn of the paper text; `A-n` = reading n in DESIGN.md section 3.
"""
from __future__ import annotations

from dataclasses import dataclass
from fractions import Fraction

import numpy as np
import scipy.sparse as sp


# ----------------------------------------------------------------------------------------
# step 0 - spectral bounds and the normalised matrix X0 the polynomial is applied to
# ----------------------------------------------------------------------------------------
def gershgorin(H) -> tuple[float, float]:
    """Gershgorin bounds over all stored entries of the GLOBAL H (reading A-5):
        eps_min = min_i (H_ii - sum_{j != i} |H_ij|),  eps_max = max_i (H_ii + sum_{j != i} |H_ij|).
    A row without a stored diagonal has H_ii = 0 (A-12).  The recursive expansion of
    theta(mu I - H) needs the spectrum mapped into [0, 1]; the paper does not say how."""
    lo, hi = np.inf, -np.inf
    for i in range(H.n):
        a, b = int(H.row_ptr[i]), int(H.row_ptr[i + 1])
        cols, vals = H.col_idx[a:b], H.val[a:b]
        d = float(vals[cols == i].sum()) if np.any(cols == i) else 0.0
        r = float(np.abs(vals[cols != i]).sum())
        lo, hi = min(lo, d - r), max(hi, d + r)
    return lo, hi


def normalised_x0(H, eps_min: float, eps_max: float) -> sp.csr_matrix:
    """X0 = (eps_max I - H) / (eps_max - eps_min): spectrum in [0,1], occupied states near 1.
    This is the X of Eq.(1)-(2) for the SP2 expansion (ref. 35)."""
    delta = eps_max - eps_min
    if not delta > 0:
        raise ValueError("degenerate spectrum bounds (A-12)")
    n = H.n
    Hs = sp.csr_matrix((H.val, H.col_idx, H.row_ptr), shape=(n, n))
    # explicit element-wise form so that every entry is (eps_max*delta_ij - H_ij)/delta, one division each
    coo = Hs.tocoo()
    diag_present = np.zeros(n, dtype=bool)
    diag_present[coo.row[coo.row == coo.col]] = True
    data = np.where(coo.row == coo.col, (eps_max - coo.data) / delta, (0.0 - coo.data) / delta)
    rows, cols = coo.row, coo.col
    miss = np.nonzero(~diag_present)[0]
    if miss.size:
        rows = np.concatenate([rows, miss])
        cols = np.concatenate([cols, miss])
        data = np.concatenate([data, np.full(miss.size, (eps_max - 0.0) / delta)])
    X0 = sp.csr_matrix((data, (rows, cols)), shape=(n, n))
    X0.sort_indices()
    return X0


# ----------------------------------------------------------------------------------------
# step 1 - the data-dependency graph S_tau
# ----------------------------------------------------------------------------------------
def _threshold(M: sp.csr_matrix, tau: float) -> sp.csr_matrix:
    """Keep entries with |value| >= tau (A-3: magnitude, kept on equality; P:L38 'magnitude below ... tau ... ignored')."""
    M = M.tocoo()
    keep = np.abs(M.data) >= tau
    out = sp.csr_matrix((M.data[keep], (M.row[keep], M.col[keep])), shape=M.shape)
    out.sort_indices()
    return out


def build_graph(H, tau: float, power: int = 2, bounds: tuple[float, float] | None = None):
    """S_tau from (H, tau) alone (reading A-1 of Eq.(2), in the spirit of Eq.(8)):
        A = floor(X0)_tau ;  T^(1) = A ;  T^(n) = floor(A T^(n-1))_tau, n = 2..power
        S = I  u  pat(T^(1)) u ... u pat(T^(power)),  then S u S^T.
    Every vertex carries a self loop (T^(0) = I; A-4).  Returns (row_ptr int64, col int32)
    with ascending columns."""
    if not (tau >= 0):
        raise ValueError("tau must be >= 0")
    lo, hi = bounds if bounds is not None else gershgorin(H)
    X0 = normalised_x0(H, lo, hi)
    n = H.n
    A = _threshold(X0, tau)
    pat = sp.identity(n, dtype=np.int8, format="csr")
    T = A
    for k in range(1, power + 1):
        if k > 1:
            T = _threshold(sp.csr_matrix(A @ T), tau)  # (A T)_ij = sum_k A_ik T_kj, then thresholded
        Tp = T.copy()
        Tp.data = np.ones_like(Tp.data, dtype=np.int8)
        pat = pat + Tp.astype(np.int8)
    pat = pat + pat.T
    pat = sp.csr_matrix(pat)
    pat.sort_indices()
    return pat.indptr.astype(np.int64), pat.indices.astype(np.int32)


def update_graph(D_row_ptr, D_col, D_val, H, tau: float):
    """Eq.(8) P:L84-88 in the symbolic form the paper uses (eps = 0):
        S_tau(t) <- floor( ( floor(D(t - dt))_tau + H(t) )^2 )_eps
    'the non-zero pattern of the thresholded density matrix ... combined with the non-zero pattern of H(t), and instead
    of the matrix square we use paths of length two'.  M = I u pat(|D_ij| >= tau) u pat(H); S = pat(M M); then S u S^T
    (D is not symmetric, obs. (i) P:L65; self loops as in build_graph, A-4).  Returns (row_ptr int64, col int32)."""
    n = H.n
    D = sp.csr_matrix((D_val, D_col, D_row_ptr), shape=(n, n)).tocoo()
    keep = np.abs(D.data) >= tau
    M = sp.csr_matrix((np.ones(int(keep.sum()), dtype=np.int64), (D.row[keep], D.col[keep])), shape=(n, n))
    Hp = sp.csr_matrix((np.ones(len(H.col_idx), dtype=np.int64), H.col_idx, H.row_ptr), shape=(n, n))
    M = M + Hp + sp.identity(n, dtype=np.int64, format="csr")
    M.data[:] = 1
    S = sp.csr_matrix(M @ M)          # entry (i, j) > 0 iff a path i - k - j of length two exists in M
    S.data[:] = 1
    S = sp.csr_matrix(S + S.T)
    S.sort_indices()
    return S.indptr.astype(np.int64), S.indices.astype(np.int32)


# ----------------------------------------------------------------------------------------
# step 2 - subgraphs (core + halo) and the pattern of the assembled result
# ----------------------------------------------------------------------------------------
def subgraphs(S_row_ptr, S_col, part, n_part: int):
    """For community p with core C_p = {i : part[i] = p}: s_p = C_p u {k : (k,i) in S, i in C_p}
    (P:L58 'core ... vertex i and all halo ... vertices that are directly connected to i'; communities
    obs. (vi) P:L65).  Local order: core ascending, then halo ascending.  Returns a list of
    (idx int32 array, ncore)."""
    part = np.asarray(part)
    out = []
    for p in range(n_part):
        core = np.nonzero(part == p)[0]
        nb = [S_col[S_row_ptr[i]:S_row_ptr[i + 1]] for i in core]
        allv = np.unique(np.concatenate(nb)) if nb else np.zeros(0, dtype=np.int64)
        halo = np.setdiff1d(allv, core, assume_unique=False)
        out.append((np.concatenate([core, halo]).astype(np.int32), int(core.size)))
    return out


def density_pattern(subs, n: int):
    """Pattern S' of the assembled P_tau (A-9): entry (k, i) is stored iff k is in the subgraph of the
    community that owns column i (P:L60-63 'assembled, column by column').  CSR, ascending columns."""
    rows = [np.repeat(idx, nc) for idx, nc in subs]
    cols = [np.tile(idx[:nc], idx.size) for idx, nc in subs]
    rows = np.concatenate(rows) if rows else np.zeros(0, dtype=np.int64)
    cols = np.concatenate(cols) if cols else np.zeros(0, dtype=np.int64)
    m = sp.csr_matrix((np.ones(rows.size, dtype=np.int8), (rows, cols)), shape=(n, n))
    m.sort_indices()
    return m.indptr.astype(np.int64), m.indices.astype(np.int32)


# ----------------------------------------------------------------------------------------
# step 3 - dense principal submatrix
# ----------------------------------------------------------------------------------------
def dense_block(H, idx, eps_min: float, eps_max: float) -> np.ndarray:
    """x[s] = X0[s, s]: the FULL principal submatrix - every stored H entry with both indices in s
    (A-2; P:L63 'small dense principal submatrix')."""
    Hs = H if sp.issparse(H) else sp.csr_matrix((H.val, H.col_idx, H.row_ptr), shape=(H.n, H.n))
    Hss = Hs[idx][:, idx].toarray()
    m = len(idx)
    delta = eps_max - eps_min
    return (eps_max * np.eye(m) - Hss) / delta


# ----------------------------------------------------------------------------------------
# steps 4-6 - the subgraph SP2 expansion, Eq.(6)
# ----------------------------------------------------------------------------------------
@dataclass
class SubResult:
    D_row_ptr: np.ndarray
    D_col: np.ndarray
    D_val: np.ndarray  # P_tau(H) on pattern S', CSR order; NOT symmetric (obs. (i) P:L65)
    t1: np.ndarray  # iters_done + 1 global core traces of X_n
    t2: np.ndarray  # iters_done + 1 global core traces of X_n^2
    branch: np.ndarray  # uint8, 0: X <- X^2, 1: X <- 2X - X^2
    iters_done: int
    eps_min: float
    eps_max: float
    subs: list
    blocks: list | None = None  # final dense X_p (kept on request)


def _branch(t1: float, t2: float, n_occ: float) -> int:
    """A-6: pick the polynomial whose next trace is closer to n_occ; Tr(X^2) = t2, Tr(2X-X^2) = 2 t1 - t2.
    Tie -> 2X - X^2.  ('the complete SP2 sequence (the same for each subgraph expansion) for the
    correct total occupation'; second-order f_n.)"""
    return 0 if abs(t2 - n_occ) < abs(2.0 * t1 - t2 - n_occ) else 1


def o_sub(H, S_row_ptr, S_col, part, n_part: int, n_occ: float, iters: int, idem_tol: float = -1.0,
          replay=None, bounds: tuple[float, float] | None = None, keep_blocks: bool = False,
          local_perm_seed: int | None = None) -> SubResult:
    """The partitioned subgraph expansion (Eq.(6)) of the SP2 polynomial:

      1. eps_min, eps_max by Gershgorin on the global H (A-5); X0 = (eps_max I - H)/(eps_max - eps_min)
      2. s_p from S (step 2);  x_p = X0[s_p, s_p] dense (A-2)
      3. for n = 0..iters-1:  t1 = sum_p sum_{i<ncore_p} (X_p)_ii ;  Y_p = X_p X_p ;
             t2 = sum_p sum_{i<ncore_p} (Y_p)_ii ;
             [idem_tol >= 0 and n >= 1 and |t1 - t2| <= idem_tol: stop]  (A-7)
             b_n = _branch(t1, t2, n_occ), the SAME for every p (Eq.(4): one polynomial)
             X_p <- Y_p  or  2 X_p - Y_p
      4. D[s_p[r], s_p[c]] = (X_p)[r, c], r < m_p, c < ncore_p (A-9, A-10)

    replay = (branch array, iters_done) forces a given sequence (isolates arithmetic from decisions).
    local_perm_seed permutes the local order inside every subgraph before the expansion and undoes it
    afterwards - mathematically a no-op (obs. (ix) P:L65), used to measure the roundoff floor."""
    lo, hi = bounds if bounds is not None else gershgorin(H)
    subs = subgraphs(S_row_ptr, S_col, part, n_part)
    Hs = sp.csr_matrix((H.val, H.col_idx, H.row_ptr), shape=(H.n, H.n))
    X = [dense_block(Hs, idx, lo, hi) for idx, _ in subs]
    perms = None
    if local_perm_seed is not None:
        rng = np.random.default_rng(local_perm_seed)
        perms = [rng.permutation(len(idx)) for idx, _ in subs]
        X = [x[np.ix_(q, q)] for x, q in zip(X, perms)]

    def core_trace(mats):
        tot = 0.0
        for p, (idx, nc) in enumerate(subs):
            d = np.diagonal(mats[p])
            if perms is not None:
                inv = np.argsort(perms[p])
                d = d[inv]
            tot += float(d[:nc].sum())
        return tot

    t1s, t2s, brs = [], [], []
    iters_done = 0
    max_iters = iters if replay is None else int(replay[1])
    for n in range(max_iters):
        t1 = core_trace(X)
        Y = [x @ x for x in X]
        t2 = core_trace(Y)
        t1s.append(t1)
        t2s.append(t2)
        if replay is None and idem_tol >= 0 and n >= 1 and abs(t1 - t2) <= idem_tol:
            break
        b = _branch(t1, t2, n_occ) if replay is None else int(replay[0][n])
        brs.append(b)
        X = Y if b == 0 else [2.0 * x - y for x, y in zip(X, Y)]
        iters_done = n + 1
    if len(t1s) == iters_done:  # log entry for the final X as well
        t1s.append(core_trace(X))
        t2s.append(core_trace([x @ x for x in X]))

    if perms is not None:
        X = [x[np.ix_(np.argsort(q), np.argsort(q))] for x, q in zip(X, perms)]
    rp, ci = density_pattern(subs, H.n)
    rows = np.concatenate([np.repeat(idx, nc) for idx, nc in subs]) if subs else np.zeros(0, int)
    cols = np.concatenate([np.tile(idx[:nc], idx.size) for idx, nc in subs]) if subs else np.zeros(0, int)
    vals = np.concatenate([x[:, :nc].reshape(-1) for x, (idx, nc) in zip(X, subs)]) if subs else np.zeros(0)
    # place the values at their CSR positions (every (k,i) occurs exactly once: each i has one owner)
    D = sp.csr_matrix((np.arange(1, rows.size + 1, dtype=np.float64), (rows, cols)), shape=(H.n, H.n))
    D.sort_indices()
    assert np.array_equal(D.indptr, rp) and np.array_equal(D.indices, ci)
    order = D.data.astype(np.int64) - 1
    return SubResult(rp, ci, vals[order], np.array(t1s), np.array(t2s), np.array(brs, dtype=np.uint8),
                     iters_done, lo, hi, subs, X if keep_blocks else None)


# ----------------------------------------------------------------------------------------
# one community at a time (full-size inputs, where the whole batch is too much work for a CPU)
# ----------------------------------------------------------------------------------------
class OneCommunity:
    """The same definitions as build_graph / subgraphs / o_sub, evaluated for ONE community p at a time, so that
    sampled outputs of a full-size system can be computed one by one:

      graph rows  S_tau is I u pat(A) u pat(floor(A A)_tau), then S u S^T (reading A-1 of Eq.(2), power 2).
                  The rows of S u S^T that belong to the core vertices C_p are the rows C_p of S together with the
                  columns C_p of S, i.e. floor(A[C_p, :] A)_tau and floor(A A[:, C_p])_tau - two thin products.
      subgraph    s_p = C_p u {k : (k, i) in S, i in C_p}, core ascending then halo ascending (obs. (vi) P:L65)
      expansion   x_p = X0[s_p, s_p] (A-2), then the GIVEN branch sequence b_0 .. b_{iters-1} ('the same for
                  each subgraph expansion' - the sequence is a global quantity, so it is an input here), and the
                  core columns of the result (Eq.(6)).
    The global quantities a single community cannot produce (eps_min/eps_max, A) are computed once from the whole H."""

    def __init__(self, H, tau: float, part, bounds: tuple[float, float] | None = None):
        if not (tau >= 0):
            raise ValueError("tau must be >= 0")
        self.H, self.tau, self.part = H, float(tau), np.asarray(part)
        self.lo, self.hi = bounds if bounds is not None else gershgorin(H)
        self.A = _threshold(normalised_x0(H, self.lo, self.hi), tau)
        self.A_csc = self.A.tocsc()
        self.Hs = sp.csr_matrix((H.val, H.col_idx, H.row_ptr), shape=(H.n, H.n))

    def subgraph(self, p: int):
        """(idx int32, ncore) of community p, from the rows and columns C_p of S."""
        core = np.nonzero(self.part == p)[0]
        if core.size == 0:
            return np.zeros(0, dtype=np.int32), 0
        A_rows = self.A[core, :]                                        # A[C_p, :]
        A_cols = self.A_csc[:, core]                                    # A[:, C_p]
        AA_rows = _threshold(sp.csr_matrix(A_rows @ self.A), self.tau)  # floor(A A)_tau, rows C_p
        AA_cols = _threshold(sp.csr_matrix(self.A @ A_cols), self.tau)  # floor(A A)_tau, columns C_p
        reached = [core, A_rows.tocoo().col, AA_rows.tocoo().col, A_cols.tocoo().row, AA_cols.tocoo().row]
        allv = np.unique(np.concatenate(reached))
        halo = np.setdiff1d(allv, core)
        return np.concatenate([core, halo]).astype(np.int32), int(core.size)

    def expand(self, p: int, branch, iters: int):
        """(idx, ncore, X[:, :ncore]) after `iters` SP2 steps with the given branches (0: X^2, 1: 2X - X^2)."""
        idx, nc = self.subgraph(p)
        X = dense_block(self.Hs, idx, self.lo, self.hi)
        for n in range(iters):
            Y = X @ X
            X = Y if int(branch[n]) == 0 else 2.0 * X - Y
        return idx, nc, X[:, :nc]


# ----------------------------------------------------------------------------------------
# finite-temperature expansion, Eq.(7)
# ----------------------------------------------------------------------------------------
def fermi_chebyshev_coeffs(mu: float, beta: float, order: int, eps_min: float, eps_max: float, nq: int = 2048) -> np.ndarray:
    """c_0..c_order of f(x) = 1/(1 + exp(beta (a x + b - mu))) on x in [-1, 1], a = (eps_max - eps_min)/2,
    b = (eps_max + eps_min)/2, by Chebyshev-Gauss quadrature with nq nodes:
        c_n = (2 - delta_n0)/nq * sum_k f(cos th_k) cos(n th_k),  th_k = pi (k + 1/2)/nq.
    (Eq.(7): 'the Fermi-operator expansion ... Chebyshev'.)"""
    a, b = 0.5 * (eps_max - eps_min), 0.5 * (eps_max + eps_min)
    th = np.pi * (np.arange(nq) + 0.5) / nq
    arg = beta * (a * np.cos(th) + b - mu)
    f = np.where(arg > 0, np.exp(-np.abs(arg)) / (1.0 + np.exp(-np.abs(arg))), 1.0 / (1.0 + np.exp(-np.abs(arg))))
    n = np.arange(order + 1)
    c = (np.cos(np.outer(n, th)) @ f) * (2.0 / nq)
    c[0] *= 0.5
    return c


@dataclass
class FermiResult:
    D_row_ptr: np.ndarray
    D_col: np.ndarray
    D_val: np.ndarray
    n_elec: float      # sum over all core diagonals
    coeffs: np.ndarray
    eps_min: float
    eps_max: float
    subs: list


def o_fermi(H, S_row_ptr, S_col, part, n_part: int, mu: float, beta: float, order: int,
            bounds: tuple[float, float] | None = None) -> FermiResult:
    """The partitioned subgraph expansion (Eq.(6)) of the finite-temperature Fermi operator (Eq.(7)):
      1. Gershgorin bounds of the global H (A-5); Ht = (H - b)/a with spectrum in [-1, 1]
      2. per community: xt = Ht[s_p, s_p] (full principal submatrix, A-2); T_0 = I, T_1 = xt,
         T_{n+1} = 2 xt T_n - T_{n-1} (Eq.(5) P:L51-56 with the Chebyshev alpha_n);  D_p = sum_{n<=order} c_n T_n
      3. core columns of D_p assembled as in o_sub."""
    lo, hi = bounds if bounds is not None else gershgorin(H)
    a, b = 0.5 * (hi - lo), 0.5 * (hi + lo)
    c = fermi_chebyshev_coeffs(mu, beta, order, lo, hi)
    subs = subgraphs(S_row_ptr, S_col, part, n_part)
    Hs = sp.csr_matrix((H.val, H.col_idx, H.row_ptr), shape=(H.n, H.n))
    blocks, n_elec = [], 0.0
    for idx, nc in subs:
        m = len(idx)
        xt = (Hs[idx][:, idx].toarray() - b * np.eye(m)) / a
        Tm, Tn = np.eye(m), xt.copy()
        D = c[0] * Tm + c[1] * Tn
        for n in range(1, order):
            Tm, Tn = Tn, 2.0 * (xt @ Tn) - Tm
            D = D + c[n + 1] * Tn
        blocks.append(D)
        n_elec += float(np.diagonal(D)[:nc].sum())
    rp, ci = density_pattern(subs, H.n)
    rows = np.concatenate([np.repeat(idx, nc) for idx, nc in subs]) if subs else np.zeros(0, int)
    cols = np.concatenate([np.tile(idx[:nc], idx.size) for idx, nc in subs]) if subs else np.zeros(0, int)
    vals = np.concatenate([x[:, :nc].reshape(-1) for x, (idx, nc) in zip(blocks, subs)]) if subs else np.zeros(0)
    Dm = sp.csr_matrix((np.arange(1, rows.size + 1, dtype=np.float64), (rows, cols)), shape=(H.n, H.n))
    Dm.sort_indices()
    order_ = Dm.data.astype(np.int64) - 1
    return FermiResult(rp, ci, vals[order_], n_elec, c, lo, hi, subs)


# ----------------------------------------------------------------------------------------
# observables
# ----------------------------------------------------------------------------------------
def expectation(D_row_ptr, D_col, D_val, A, n: int | None = None) -> float:
    """<A> = Tr[D A] = sum_{k,i} D_ki A_ik (P:L72 'expectation values ... Tr[DA]'; E_band = Tr[DH]).
    D given as CSR arrays (the assembled, non-symmetric P_tau), A a duck-typed CSR object or a dense array."""
    if hasattr(A, "row_ptr"):
        n = A.n
        Ad = sp.csr_matrix((A.val, A.col_idx, A.row_ptr), shape=(n, n))
    else:
        Ad = sp.csr_matrix(np.asarray(A))
        n = Ad.shape[0]
    D = sp.csr_matrix((D_val, D_col, D_row_ptr), shape=(n, n))
    return float(D.multiply(Ad.T).sum())


def error_norms(D_row_ptr, D_col, D_val, D_ref) -> tuple[float, float, float]:
    """Error of the assembled sparse D against a dense reference (Fig.2: "the error in the calculated density
    matrix ... as measured by the Frobenius norm (normalized per atom)"; obs. (ii) P:L65: the error is set by tau).
    Returns (max |D - D_ref| over the stored entries of D,
             sum (D - D_ref)^2 over the stored entries,
             ||D - D_ref||_F^2 over the full matrix: where D stores nothing it is zero, obs. (iv) P:L65)."""
    D_ref = np.asarray(D_ref, dtype=np.float64)
    n = D_ref.shape[0]
    D = np.zeros((n, n))
    stored = np.zeros((n, n), dtype=bool)
    for k in range(n):
        cols = np.asarray(D_col[D_row_ptr[k]:D_row_ptr[k + 1]])
        D[k, cols] = D_val[D_row_ptr[k]:D_row_ptr[k + 1]]
        stored[k, cols] = True
    diff = D - D_ref
    inside = diff[stored]
    return (float(np.abs(inside).max()) if inside.size else 0.0, float((inside * inside).sum()),
            float((diff * diff).sum()))


# ----------------------------------------------------------------------------------------
# exact projector
# ----------------------------------------------------------------------------------------
def o_diag(H, n_occ: int) -> np.ndarray:
    """D = theta(mu I - H) from a dense symmetric eigendecomposition: the projector onto the
    n_occ lowest eigenvectors."""
    n = H.n
    Hd = sp.csr_matrix((H.val, H.col_idx, H.row_ptr), shape=(n, n)).toarray()
    w, v = np.linalg.eigh(Hd)
    k = int(round(n_occ))
    vo = v[:, :k]
    return vo @ vo.T


# ----------------------------------------------------------------------------------------
# Eq.(4)-(5) literally, on the full matrix (tiny inputs) - proves o_sub == P_tau of the paper
# ----------------------------------------------------------------------------------------
def sp2_polynomial_coeffs(branches) -> list[int]:
    """Monomial coefficients c_n (exact integers) of the composed SP2 polynomial p(x) in x = X0:
    p_0 = x; p_{k+1} = p_k^2 (b=0) or 2 p_k - p_k^2 (b=1).  Degree 2^len(branches) - 'an expansion
    order of over a billion in only 30 iterations'.  This is P(X) = sum c_n T^(n)(X) of
    Eq.(1) P:L36 with T^(n)(X) = X^n."""
    p = [0, 1]
    for b in branches:
        sq = [0] * (2 * len(p) - 1)
        for i, a in enumerate(p):
            if a:
                for j, c in enumerate(p):
                    sq[i + j] += a * c
        if b == 0:
            p = sq
        else:
            p = [(2 * p[i] if i < len(p) else 0) - sq[i] for i in range(len(sq))]
    return p


def _column_masks(subs, n: int) -> np.ndarray:
    """mask[k, i] = True iff (k, i) is an edge of S' (A-9): k in the subgraph of i's community."""
    mask = np.zeros((n, n), dtype=bool)
    for idx, nc in subs:
        mask[np.ix_(idx, idx[:nc])] = True
    return mask


def o_eq5_exact(X0_dense, subs, branches):
    """Eq.(4)-(5) in exact rational arithmetic with the monomial basis:
        T^(0) = I ;  T^(n) = floor( X0 T^(n-1) )_{S'}   (alpha_n = 1, no lower-order terms; X0 UNMASKED on the left)
        P_tau = sum_n c_n T^(n),  c_n = sp2_polynomial_coeffs(branches).
    X0_dense: n x n array of floats (converted exactly) or Fractions.  Returns an object array of Fractions."""
    n = len(X0_dense)
    X = [[Fraction(X0_dense[i][j]) for j in range(n)] for i in range(n)]
    mask = _column_masks(subs, n)
    c = sp2_polynomial_coeffs(branches)
    T = [[Fraction(int(i == j)) for j in range(n)] for i in range(n)]
    P = [[c[0] * T[i][j] for j in range(n)] for i in range(n)]
    nzX = [[k for k in range(n) if X[i][k] != 0] for i in range(n)]
    for deg in range(1, len(c)):
        Tn = [[Fraction(0)] * n for _ in range(n)]
        for i in range(n):
            for j in range(n):
                if mask[i, j]:
                    s = Fraction(0)
                    for k in nzX[i]:
                        t = T[k][j]
                        if t != 0:
                            s += X[i][k] * t
                    Tn[i][j] = s
        T = Tn
        if c[deg]:
            for i in range(n):
                for j in range(n):
                    if T[i][j] != 0:
                        P[i][j] += c[deg] * T[i][j]
    out = np.empty((n, n), dtype=object)
    for i in range(n):
        for j in range(n):
            out[i, j] = P[i][j]
    return out


def o_eq5_nested(X0_dense: np.ndarray, subs, branches) -> np.ndarray:
    """Same P_tau in floating point for more iterations.  Column i of T^(n) is (M_i X0)^n e_i with M_i the
    mask of column i, so column i of P_tau is p(M_i X0) e_i and the composed polynomial can be applied
    in its nested form: apply_0(v) = M_i (X0 v); apply_{k+1}(v) = apply_k(apply_k(v)) or
    2 apply_k(v) - apply_k(apply_k(v)) - 2^k masked mat-vecs with the FULL X0 per column."""
    n = X0_dense.shape[0]
    mask = _column_masks(subs, n)
    out = np.zeros((n, n))
    for i in range(n):
        e = np.zeros(n)
        e[i] = 1.0
        out[:, i] = _nested(X0_dense, mask[:, i], branches, len(branches), e)
    return out


def _nested(X0, m, branches, k, v):
    """p_k(M X0) v with p_0(x) = x, p_{j+1} = f_j(p_j): p_k(A) v = f_{k-1}(p_{k-1}(A)) v."""
    if k == 0:
        return np.where(m, X0 @ v, 0.0)
    w = _nested(X0, m, branches, k - 1, v)
    ww = _nested(X0, m, branches, k - 1, w)
    return ww if branches[k - 1] == 0 else 2.0 * w - ww
