"""CPU-only: the seeded input generators (gbe_inputs/) produce what DESIGN.md section 4 says - deterministic, exactly
symmetric Hamiltonians of the stated shapes.  They hold none of the method's arithmetic and serve both the oracle and
the CUDA path."""
import numpy as np

import gbe_inputs as gi


def _sym(H):
    A = H.to_scipy()
    return abs(A - A.T).max() == 0.0


def test_chain_is_the_stated_model():
    s = gi.config(1)
    a = s.H.to_dense()
    assert s.n == 512 and s.n_occ == 256 and s.n_part == 16 and s.tau == 1e-5 and s.iters == 40
    assert _sym(s.H) and np.array_equal(s.part, np.arange(512) // 32)
    assert np.allclose(np.diag(a, 1), -1.0) and np.allclose(np.diag(a, 4), -np.exp(-3.0)) and np.all(np.diag(a, 5) == 0)
    d = np.diag(a)
    assert np.all(np.abs(d[0::2] - 1.0) <= 0.05) and np.all(np.abs(d[1::2] + 1.0) <= 0.05)   # +1 / -1 plus U(-0.05, 0.05)
    assert np.array_equal(gi.config(1).H.val, s.H.val)                                      # deterministic
    assert not np.array_equal(gi.chain(512, 16, seed=1).H.val, s.H.val)


def test_water_box_shape_and_symmetry():
    s = gi.water_box(128, 16, seed=0)
    assert s.n == 768 and s.n_occ == 512.0 and _sym(s.H)
    a = s.H.to_dense()
    d = np.diag(a).reshape(-1, 6)
    assert np.all(d[:, 0] == -20.0) and np.all(d[:, 1:4] == -10.0) and np.all(d[:, 4:] == -12.0)
    # no same-atom off-diagonal elements: the O block of every molecule is diagonal
    for k in range(0, 768, 6):
        blk = a[k:k + 4, k:k + 4]
        assert np.count_nonzero(blk - np.diag(np.diag(blk))) == 0
    # hopping f(r) = -2 exp(-1.5 r) times direction cosines: bounded by 2; s-s elements (H1-H2 columns 4, 5 of a molecule
    # against those of another) are never below the value at the 6 A cutoff
    offd = a - np.diag(np.diag(a))
    assert np.abs(offd).max() <= 2.0
    ss = np.abs(offd[4::6, :][:, 4::6])
    assert ss[ss > 0].min() >= 2.0 * np.exp(-1.5 * 6.0) * (1 - 1e-12)
    # partitions are contiguous runs of whole molecules
    assert np.all(np.diff(s.part) >= 0) and np.all(s.part.reshape(-1, 6) == s.part.reshape(-1, 6)[:, :1])
    box = s.meta["box"]
    assert abs(box ** 3 / 128 - gi.systems.WATER_DENSITY_A3) < 1e-9                          # 1 g/cm^3


def test_water_geometry_does_not_depend_on_the_partition_count():
    a, b = gi.water_box(64, 8, seed=3), gi.water_box(64, 16, seed=3)
    assert np.array_equal(a.H.val, b.H.val) and np.array_equal(a.H.col_idx, b.H.col_idx)
    assert a.n_part == 8 and b.n_part == 16


def test_gapped_variant_keeps_the_oxygens_apart_and_has_a_gap():
    s = gi.water_box(64, 8, seed=0, min_oo=2.4, occ_per_mol=3.0)
    assert s.n_occ == 192.0 and _sym(s.H)
    w = np.linalg.eigvalsh(s.H.to_dense())
    assert w[192] - w[191] > 0.5
    lit = gi.water_box(64, 8, seed=0)
    wl = np.linalg.eigvalsh(lit.H.to_dense())
    assert wl[256] - wl[255] < 0.2                                                           # reading A-15: no gap as written


def test_peptide_construction_small():
    s = gi.peptide_water(12, box=14.0, seed=0)
    assert _sym(s.H) and s.n == 12 * 50 + 6 * s.meta["n_wat"]
    assert np.array_equal(np.bincount(s.part)[:12], np.full(12, 50))                          # one residue per core
    assert s.n_occ == 25.0 * 12 + 4.0 * s.meta["n_wat"]


def test_random_banded_shuffle_is_a_relabelling():
    a = gi.random_banded(40, half_bw=3, n_part=4, seed=2, shuffle=False)
    b = gi.random_banded(40, half_bw=3, n_part=4, seed=2, shuffle=True)
    assert np.allclose(np.sort(np.linalg.eigvalsh(a.H.to_dense())), np.sort(np.linalg.eigvalsh(b.H.to_dense())))
    assert sorted(np.bincount(a.part)) == sorted(np.bincount(b.part)) and not np.array_equal(a.part, b.part)


def test_bench_helpers_blob_hash_traffic_record_and_oracle_sample(tmp_path, monkeypatch):
    """bench.py host logic: the git blob hash that ties profiles/x2_traffic.json to the kernel source it was captured on,
    the refusal of a stale or foreign record, and the sizing of the oracle sample of the reference arm."""
    import hashlib
    import json
    import os
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    import bench
    f = tmp_path / "k.cu"
    f.write_bytes(b"hello\n")
    assert bench.git_blob_sha1(str(f)) == hashlib.sha1(b"blob 6\0hello\n").hexdigest() == "ce013625030ba8dba906f756967f9e9ca394464a"
    rec = tmp_path / "x2_traffic.json"
    monkeypatch.setattr(bench, "X2_TRAFFIC_JSON", str(rec))
    monkeypatch.setattr(bench, "X2_SOURCE", str(f))
    assert bench.x2_traffic("water4096")[0] is None                      # no record
    rec.write_text(json.dumps({"workload": "water4096", "dram_bytes_per_launch": 2.0e9,
                               "gbe_x2_cu_blob": bench.git_blob_sha1(str(f))}))
    assert bench.x2_traffic("water4096")[0] == 2.0e9
    assert bench.x2_traffic("water1024")[0] is None                      # another workload
    f.write_bytes(b"changed\n")
    assert bench.x2_traffic("water4096")[0] is None                      # the kernel source changed since the capture
    monkeypatch.setattr(bench, "cpu_cores", lambda: 16)
    assert bench.oracle_sample_molecules("water4096", 3, 300.0) == 4096   # three passes of the real workload fit
    assert bench.oracle_sample_molecules("water4096", 25, 300.0) < 4096   # the driver's 20 + 5 do not: a smaller box
    assert bench.oracle_sample_molecules("water4096", 10 ** 6, 300.0) == 256
