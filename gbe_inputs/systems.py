"""Seeded synthetic tight-binding Hamiltonians (stand-ins for the paper's test systems).

Recipes follow BASELINE.json `configs` and SURVEY.md section 8(d) / readings A-13, A-14, A-16
(listed again in DESIGN.md).  Everything here is *input construction*: geometry, a sigma-only
Slater-Koster hopping model, CSR assembly, orbital ordering and the partition vector.  None of
the method's arithmetic (spectral bounds, graph S_tau, subgraph extraction, SP2) lives here.

All generators are deterministic functions of their arguments (numpy PCG64 with the given seed).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import scipy.sparse as sp
from scipy.spatial import cKDTree


# ----------------------------------------------------------------------------------------
# containers
# ----------------------------------------------------------------------------------------
@dataclass
class CSR:
    """Plain CSR triple with the dtypes the C ABI uses (include/gbe.h: gbe_csr_view)."""

    n: int
    row_ptr: np.ndarray  # int64, n+1
    col_idx: np.ndarray  # int32, nnz, ascending within a row
    val: np.ndarray  # float64, nnz

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])

    def to_scipy(self) -> sp.csr_matrix:
        return sp.csr_matrix((self.val, self.col_idx, self.row_ptr), shape=(self.n, self.n))

    def to_dense(self) -> np.ndarray:
        return self.to_scipy().toarray()

    @staticmethod
    def from_scipy(m) -> "CSR":
        m = sp.csr_matrix(m)
        m.sum_duplicates()
        m.sort_indices()
        return CSR(
            n=m.shape[0],
            row_ptr=np.ascontiguousarray(m.indptr, dtype=np.int64),
            col_idx=np.ascontiguousarray(m.indices, dtype=np.int32),
            val=np.ascontiguousarray(m.data, dtype=np.float64),
        )

    @staticmethod
    def from_dense(a: np.ndarray, keep_zeros: bool = False) -> "CSR":
        a = np.asarray(a, dtype=np.float64)
        if keep_zeros:
            n = a.shape[0]
            rp = np.arange(n + 1, dtype=np.int64) * n
            ci = np.tile(np.arange(n, dtype=np.int32), n)
            return CSR(n, rp, ci, a.reshape(-1).copy())
        return CSR.from_scipy(sp.csr_matrix(a))


@dataclass
class TBSystem:
    """One benchmark/parity workload: H, the caller-chosen communities and the run parameters."""

    name: str
    H: CSR
    part: np.ndarray  # int32, vertex -> partition id
    n_part: int
    n_occ: float
    tau: float = 1e-5
    iters: int = 40
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return self.H.n


def contiguous_partition(n: int, n_part: int) -> np.ndarray:
    """part[i] = i // ceil(n / n_part): the library's default when the caller passes no partition."""
    blk = -(-n // n_part)
    return (np.arange(n, dtype=np.int64) // blk).astype(np.int32)


# ----------------------------------------------------------------------------------------
# config 1: open 1-D chain (BASELINE.json configs[0]; reading A-13)
# ----------------------------------------------------------------------------------------
def chain(n: int = 512, n_part: int = 16, seed: int = 0, reach: int = 4, noise: float = 0.05,
          tau: float = 1e-5, iters: int = 40, periodic: bool = False,
          alternate: bool = True) -> TBSystem:
    """Open chain, one orbital per site: H_ii = (+1 even, -1 odd) + U(-noise, noise);
    H_{i,i+-d} = -exp(-(d-1)) for d = 1..reach; half filling."""
    rng = np.random.Generator(np.random.PCG64(seed))
    diag = np.where(np.arange(n) % 2 == 0, 1.0, -1.0) if alternate else np.zeros(n)
    diag = diag + rng.uniform(-noise, noise, size=n) if noise > 0 else diag.astype(np.float64)
    rows, cols, vals = [np.arange(n)], [np.arange(n)], [diag]
    for d in range(1, reach + 1):
        t = -np.exp(-(d - 1.0))
        if periodic:
            i = np.arange(n)
            j = (i + d) % n
        else:
            i = np.arange(n - d)
            j = i + d
        rows += [i, j]
        cols += [j, i]
        vals += [np.full(i.size, t), np.full(i.size, t)]
    m = sp.coo_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(n, n))
    return TBSystem(
        name=f"chain{n}", H=CSR.from_scipy(m), part=contiguous_partition(n, n_part), n_part=n_part,
        n_occ=float(n // 2), tau=tau, iters=iters,
        meta=dict(kind="chain", n=n, seed=seed, reach=reach, periodic=periodic),
    )


# ----------------------------------------------------------------------------------------
# shared sigma-only Slater-Koster assembly (reading A-14)
# ----------------------------------------------------------------------------------------
def _sk_hamiltonian(pos: np.ndarray, box: float, has_p: np.ndarray, eps_s: np.ndarray,
                    eps_p: np.ndarray, cutoff: float = 6.0) -> tuple[CSR, np.ndarray]:
    """H over atoms at `pos` (periodic cube of edge `box`, minimum image).

    Atom a carries an s orbital (on-site eps_s[a]) and, if has_p[a], three p orbitals
    (eps_p[a]); orbital order per atom: s, px, py, pz.  Radial function f(r) = -2 exp(-1.5 r),
    r < cutoff; blocks between atoms a != b with l = (R_b - R_a)/r:
        s_a - s_b   : f          s_a - p_b(alpha): +f l_alpha
        p_a(alpha) - s_b : -f l_alpha      p_a(alpha) - p_b(beta): f l_alpha l_beta
    No same-atom off-diagonal elements.  Returns (H, orbital offset per atom)."""
    na = pos.shape[0]
    norb = np.where(has_p, 4, 1).astype(np.int64)
    off = np.concatenate([[0], np.cumsum(norb)])
    n = int(off[-1])
    wrapped = np.mod(pos, box)
    wrapped[wrapped >= box] = 0.0
    tree = cKDTree(wrapped, boxsize=box)
    pairs = tree.query_pairs(r=cutoff, output_type="ndarray")
    a, b = pairs[:, 0], pairs[:, 1]
    d = wrapped[b] - wrapped[a]
    d -= box * np.round(d / box)
    r = np.sqrt((d * d).sum(1))
    keep = (r < cutoff) & (r > 0)
    a, b, d, r = a[keep], b[keep], d[keep], r[keep]
    l = d / r[:, None]
    f = -2.0 * np.exp(-1.5 * r)

    rows, cols, vals = [], [], []

    def add(ri, ci, v):
        rows.extend([ri, ci])
        cols.extend([ci, ri])
        vals.extend([v, v])

    # s-s
    add(off[a], off[b], f)
    pa, pb = has_p[a], has_p[b]
    for al in range(3):
        # s_a - p_b(alpha)
        m = pb
        add(off[a][m], off[b][m] + 1 + al, (f * l[:, al])[m])
        # p_a(alpha) - s_b
        m = pa
        add(off[a][m] + 1 + al, off[b][m], (-f * l[:, al])[m])
        for be in range(3):
            m = pa & pb
            add(off[a][m] + 1 + al, off[b][m] + 1 + be, (f * l[:, al] * l[:, be])[m])
    # on-site
    diag = np.empty(n)
    diag[off[:-1]] = eps_s
    for al in range(3):
        diag[off[:-1][has_p] + 1 + al] = eps_p[has_p]
    rows.append(np.arange(n))
    cols.append(np.arange(n))
    vals.append(diag)
    m = sp.coo_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(n, n))
    return CSR.from_scipy(m), off


def _random_rotations(rng: np.random.Generator, k: int) -> np.ndarray:
    """k uniform random rotation matrices from normalised 4-D Gaussian quaternions."""
    q = rng.normal(size=(k, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q.T
    R = np.empty((k, 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z)
    R[:, 0, 1] = 2 * (x * y - z * w)
    R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w)
    R[:, 1, 1] = 1 - 2 * (x * x + z * z)
    R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w)
    R[:, 2, 1] = 2 * (y * z + x * w)
    R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def _excluded_points(rng: np.random.Generator, k: int, box: float, dmin: float) -> np.ndarray:
    """k points uniform in the periodic cube subject to a minimum mutual distance dmin (random sequential addition)."""
    nc = max(1, int(box // dmin))
    cell = box / nc
    grid: dict[tuple[int, int, int], list[int]] = {}
    pts = np.zeros((k, 3))
    i = 0
    while i < k:
        cand = rng.uniform(0.0, box, size=(64, 3))
        for p in cand:
            c = tuple((np.floor(p / cell).astype(int) % nc).tolist())
            ok = True
            for dx in (-1, 0, 1):
                for dy in (-1, 0, 1):
                    for dz in (-1, 0, 1):
                        for j in grid.get(((c[0] + dx) % nc, (c[1] + dy) % nc, (c[2] + dz) % nc), ()):
                            d = p - pts[j]
                            d -= box * np.round(d / box)
                            if d @ d < dmin * dmin:
                                ok = False
                                break
                        if not ok:
                            break
                    if not ok:
                        break
                if not ok:
                    break
            if ok:
                pts[i] = p
                grid.setdefault(c, []).append(i)
                i += 1
                if i == k:
                    break
    return pts


def _water_geometry(rng: np.random.Generator, n_mol: int, box: float, min_oo: float = 0.0) -> np.ndarray:
    """(n_mol, 3, 3): O, H1, H2 positions; O uniform in the cube (optionally at least min_oo apart), O-H 0.96 A,
    HOH 104.5 deg."""
    o = rng.uniform(0.0, box, size=(n_mol, 3)) if min_oo <= 0 else _excluded_points(rng, n_mol, box, min_oo)
    R = _random_rotations(rng, n_mol)
    half = np.deg2rad(104.5 / 2.0)
    h_local = 0.96 * np.array([[np.sin(half), 0.0, np.cos(half)], [-np.sin(half), 0.0, np.cos(half)]])
    h = o[:, None, :] + np.einsum("kij,hj->khi", R, h_local)
    return np.concatenate([o[:, None, :], h], axis=1)


def _rcb_order(points: np.ndarray, leaf: int = 4) -> np.ndarray:
    """Recursive coordinate bisection: permutation that lists points leaf by leaf
    (split the longest extent at the median until a leaf holds <= `leaf` points)."""
    out = []

    def rec(idx):
        if idx.size <= leaf:
            out.append(idx)
            return
        p = points[idx]
        ax = int(np.argmax(p.max(0) - p.min(0)))
        order = np.argsort(p[:, ax], kind="stable")
        half = idx.size // 2
        rec(idx[order[:half]])
        rec(idx[order[half:]])

    rec(np.arange(points.shape[0]))
    return np.concatenate(out)


WATER_DENSITY_A3 = 29.915  # A^3 per molecule at 1 g/cm^3, 18.015 g/mol


def water_box(n_mol: int = 1024, n_part: int = 128, seed: int = 0, tau: float = 1e-5,
              iters: int = 40, cutoff: float = 6.0, min_oo: float = 0.0, occ_per_mol: float = 4.0) -> TBSystem:
    """Periodic water box (BASELINE.json configs[1], [2]): 6 orbitals per molecule
    (O s, px, py, pz, H1 s, H2 s); on-site -20 / -10 / -12 eV; n_occ = 4 per molecule.
    Molecules are ordered by recursive coordinate bisection; partitions are contiguous runs.
    The literal model (min_oo = 0, 4 electrons per molecule) has no HOMO-LUMO gap (reading A-15).  The optional
    "gapped" variant - oxygens at least min_oo = 2.4 A apart and occ_per_mol = 3 - has a gap of about 1 eV, so SP2
    converges and the error against the exact projector is meaningful; it is used for reporting only."""
    rng = np.random.Generator(np.random.PCG64(seed))
    box = (WATER_DENSITY_A3 * n_mol) ** (1.0 / 3.0)
    geo = _water_geometry(rng, n_mol, box, min_oo)  # drawn before ordering: independent of n_part
    order = _rcb_order(geo[:, 0, :], leaf=4)
    geo = geo[order]
    pos = geo.reshape(-1, 3)
    has_p = np.tile(np.array([True, False, False]), n_mol)
    eps_s = np.tile(np.array([-20.0, -12.0, -12.0]), n_mol)
    eps_p = np.tile(np.array([-10.0, 0.0, 0.0]), n_mol)
    H, _ = _sk_hamiltonian(pos, box, has_p, eps_s, eps_p, cutoff)
    n = 6 * n_mol
    mol_per_part = -(-n_mol // n_part)
    part = (np.arange(n) // 6 // mol_per_part).astype(np.int32)
    return TBSystem(
        name=f"water{n_mol}", H=H, part=part, n_part=n_part, n_occ=float(occ_per_mol) * n_mol, tau=tau, iters=iters,
        meta=dict(kind="water", n_mol=n_mol, box=box, seed=seed, cutoff=cutoff, min_oo=min_oo, occ_per_mol=occ_per_mol),
    )


# ----------------------------------------------------------------------------------------
# config 4: polypeptide-like random coil in water (reading A-16)
# ----------------------------------------------------------------------------------------
def _self_avoiding_walk(rng: np.random.Generator, n_beads: int, box: float, bond: float = 1.5,
                        dmin: float = 1.5) -> np.ndarray:
    """Off-lattice self-avoiding walk in a periodic cube: consecutive beads `bond` apart,
    non-bonded beads at least `dmin` apart (minimum image).  Growth with retry + backtracking."""
    cell = dmin
    nc = int(box // cell)
    cell = box / nc
    grid: dict[tuple[int, int, int], list[int]] = {}
    pos = np.zeros((n_beads, 3))

    def key(p):
        return tuple((np.floor(np.mod(p, box) / cell).astype(int) % nc).tolist())

    def ok(p, skip):
        k = key(p)
        for dx in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dz in (-1, 0, 1):
                    for j in grid.get(((k[0] + dx) % nc, (k[1] + dy) % nc, (k[2] + dz) % nc), ()):
                        if j == skip:
                            continue
                        d = p - pos[j]
                        d -= box * np.round(d / box)
                        if d @ d < dmin * dmin:
                            return False
        return True

    pos[0] = rng.uniform(0, box, 3)
    grid.setdefault(key(pos[0]), []).append(0)
    i = 1
    while i < n_beads:
        placed = False
        for _ in range(64):
            v = rng.normal(size=3)
            v *= bond / np.linalg.norm(v)
            p = pos[i - 1] + v
            if ok(p, i - 1):
                pos[i] = p
                grid.setdefault(key(p), []).append(i)
                placed = True
                break
        if placed:
            i += 1
        else:  # backtrack a few beads
            back = min(i - 1, 5)
            for j in range(i - back, i):
                grid[key(pos[j])].remove(j)
            i -= back
    return pos


def peptide_water(n_res: int = 2000, box: float = 60.0, seed: int = 0, tau: float = 1e-5,
                  iters: int = 40, waters_per_part: int = 8, cutoff: float = 6.0) -> TBSystem:
    """Random-coil polypeptide-like chain solvated in the water construction above
    (BASELINE.json configs[3]).  Per residue: 3 backbone heavy atoms on the walk + 7 heavy atoms
    and 10 H uniform in a 2 A ball around a random backbone bead of that residue; heavy atoms carry
    s,p (on-site -20/-10), H carries s (-12).  Water molecules whose O is < 2 A from any solute
    atom are removed.  Cores: one residue (50 orbitals) each, then `waters_per_part` waters each.
    n_occ = 25 per residue + 4 per water."""
    rng = np.random.Generator(np.random.PCG64(seed))
    back = _self_avoiding_walk(rng, 3 * n_res, box)

    def ball(k):
        v = rng.normal(size=(k, 3))
        v /= np.linalg.norm(v, axis=1, keepdims=True)
        return v * (2.0 * rng.uniform(size=(k, 1)) ** (1.0 / 3.0))

    res_pos = np.empty((n_res, 20, 3))
    bb = back.reshape(n_res, 3, 3)
    res_pos[:, :3] = bb
    anchor = rng.integers(0, 3, size=(n_res, 17))
    side = bb[np.arange(n_res)[:, None], anchor] + ball(n_res * 17).reshape(n_res, 17, 3)
    res_pos[:, 3:10] = side[:, :7]  # heavy
    res_pos[:, 10:] = side[:, 7:]  # H
    solute = res_pos.reshape(-1, 3)

    n_cand = int(round(box ** 3 / WATER_DENSITY_A3))
    geo = _water_geometry(rng, n_cand, box)
    tree = cKDTree(np.mod(solute, box) % box, boxsize=box)
    dist, _ = tree.query(np.mod(geo[:, 0, :], box) % box, k=1)
    geo = geo[dist >= 2.0]
    geo = geo[_rcb_order(geo[:, 0, :], leaf=4)]
    n_wat = geo.shape[0]

    pos = np.concatenate([solute, geo.reshape(-1, 3)])
    res_p = np.tile(np.array([True] * 10 + [False] * 10), n_res)
    wat_p = np.tile(np.array([True, False, False]), n_wat)
    has_p = np.concatenate([res_p, wat_p])
    eps_s = np.where(has_p, -20.0, -12.0)
    eps_p = np.where(has_p, -10.0, 0.0)
    H, off = _sk_hamiltonian(pos, box, has_p, eps_s, eps_p, cutoff)
    n = H.n
    n_sol = 50 * n_res
    part = np.empty(n, dtype=np.int32)
    part[:n_sol] = np.arange(n_sol) // 50
    part[n_sol:] = n_res + (np.arange(n - n_sol) // 6 // waters_per_part)
    n_part = int(part.max()) + 1
    return TBSystem(
        name=f"peptide{n_res}", H=H, part=part, n_part=n_part, n_occ=25.0 * n_res + 4.0 * n_wat,
        tau=tau, iters=iters,
        meta=dict(kind="peptide_water", n_res=n_res, n_wat=n_wat, box=box, seed=seed, cutoff=cutoff),
    )


# ----------------------------------------------------------------------------------------
# small generic inputs for tests
# ----------------------------------------------------------------------------------------
def random_banded(n: int = 96, half_bw: int = 6, n_part: int = 6, seed: int = 0, gap: float = 2.0,
                  tau: float = 1e-3, iters: int = 20, shuffle: bool = False) -> TBSystem:
    """Random symmetric banded matrix with an alternating on-site term of size `gap`/2 (keeps a
    spectral gap at half filling).  With shuffle=True the vertex labels and the partition vector are
    randomly permuted (non-contiguous communities, as METIS would return)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    a = np.zeros((n, n))
    for d in range(1, half_bw + 1):
        v = rng.normal(scale=0.5 * np.exp(-0.7 * (d - 1)), size=n - d)
        a[np.arange(n - d), np.arange(d, n)] = v
    a = a + a.T
    a[np.arange(n), np.arange(n)] = np.where(np.arange(n) % 2 == 0, gap, -gap) + rng.uniform(-0.1, 0.1, n)
    part = contiguous_partition(n, n_part)
    if shuffle:
        perm = rng.permutation(n)
        a = a[np.ix_(perm, perm)]
        part = part[perm]
    return TBSystem(
        name=f"banded{n}", H=CSR.from_dense(a), part=part.astype(np.int32), n_part=n_part,
        n_occ=float(n // 2), tau=tau, iters=iters, meta=dict(kind="banded", seed=seed, shuffle=shuffle),
    )


def config(i: int, **kw) -> TBSystem:
    """BASELINE.json `configs[i-1]` (1-based, as SURVEY.md numbers them). Config 5 is a sweep over
    tau x n_part on config 3's geometry: pass tau= and n_part=."""
    if i == 1:
        return chain(512, 16, seed=0, **kw)
    if i == 2:
        return water_box(1024, kw.pop("n_part", 128), seed=0, **kw)
    if i == 3 or i == 5:
        return water_box(4096, kw.pop("n_part", 512), seed=0, **kw)
    if i == 4:
        return peptide_water(2000, seed=0, **kw)
    raise ValueError(f"no config {i}")
