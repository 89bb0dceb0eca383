"""gbe_expectation_static: the entry point that allocates nothing (include/gbe.h) against gbe_expectation, the existing
path with pool allocations.  Collected last on purpose (the suite runs with `pytest -x`).

Both run the same two kernels in the same order on the same inputs; only where the n per-row partial sums live differs
(a static 1 MiB device array inside the library against a pool allocation), so the results agree bit for bit - asserted
within the tolerance the observable tests use (1e-10 * sum|A|, tests/test_gpu_parity.py) and, stricter, exactly.
"""
import numpy as np
import pytest
import scipy.sparse as sp

import gbe_inputs as gi

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gbe():
    import torch
    assert torch.cuda.is_available()
    from paper_1603_00937_b200 import build
    build.build()
    import paper_1603_00937_b200 as pkg
    pkg.lib()  # fails loudly if the CUDA library is missing
    return pkg


def density(gbe, s):
    import torch
    Hd = gbe.DeviceCSR.from_host(s.H)
    part_t = torch.from_numpy(np.asarray(s.part, dtype=np.int32)).cuda()
    g = gbe.gbe_build_graph(Hd, s.tau, part_t, s.n_part)
    D, _ = gbe.gbe_density(Hd, g, s.n_occ, s.iters, -1.0)
    torch.cuda.synchronize()
    return g, Hd, D


def test_static_scratch_expectation_matches_the_allocating_path_on_calls_in_a_row(gbe):
    import torch
    big, small = gi.config(2), gi.config(1)  # 6,144 and 512 orbitals: the second call reads 512 of 6,144 stale words
    gb, Hb, Db = density(gbe, big)
    gs, Hs, Ds = density(gbe, small)
    eye = gbe.DeviceCSR.from_host(gi.CSR.from_scipy(sp.identity(big.n, format="csr")))
    rng = np.random.default_rng(3)
    Ar = gi.CSR.from_scipy(sp.random(big.n, big.n, density=2e-3, random_state=rng, format="csr") + sp.triu(big.H.to_scipy(), k=1))
    Ard = gbe.DeviceCSR.from_host(Ar)  # non-symmetric operand: the transposed lookup
    ref = {"big_H": gbe.gbe_expectation(gb, Db, Hb), "small_H": gbe.gbe_expectation(gs, Ds, Hs),
           "big_I": gbe.gbe_expectation(gb, Db, eye), "big_A": gbe.gbe_expectation(gb, Db, Ard)}
    scale = {"big_H": np.abs(big.H.val).sum(), "small_H": np.abs(small.H.val).sum(), "big_I": float(big.n),
             "big_A": np.abs(Ar.val).sum()}
    out = torch.full((8,), float("nan"), dtype=torch.float64, device="cuda")

    # two calls in a row, each read back before the next: large problem first, so the second finds stale partials
    n0 = gbe.gbe_launch_count()
    gbe.gbe_expectation_static(gb, Db, Hb, out[0:1])
    torch.cuda.synchronize()
    assert gbe.gbe_launch_count() - n0 == 2  # the library's own kernels ran, two of them
    first = float(out[0])
    gbe.gbe_expectation_static(gs, Ds, Hs, out[1:2])
    torch.cuda.synchronize()
    second = float(out[1])
    assert abs(first - ref["big_H"]) <= 1e-10 * scale["big_H"] and first == ref["big_H"]
    assert abs(second - ref["small_H"]) <= 1e-10 * scale["small_H"] and second == ref["small_H"]

    # four calls enqueued back to back on one stream (stream order keeps them apart), nothing read in between; device
    # memory in use does not move (set-up - module load, the address look-up - happened in the calls above)
    free0, _ = torch.cuda.mem_get_info()
    gbe.gbe_expectation_static(gb, Db, eye, out[2:3])
    gbe.gbe_expectation_static(gs, Ds, Hs, out[3:4])
    gbe.gbe_expectation_static(gb, Db, Ard, out[4:5])
    gbe.gbe_expectation_static(gb, Db, Hb, out[5:6])
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    got = out.cpu().numpy()
    for slot, key in ((2, "big_I"), (3, "small_H"), (4, "big_A"), (5, "big_H")):
        assert abs(got[slot] - ref[key]) <= 1e-10 * scale[key], (key, got[slot], ref[key])
        assert got[slot] == ref[key], (key, got[slot], ref[key])
    assert np.isnan(got[6:]).all()  # one double written per call

    # a side stream, ordered after the work above by the synchronize
    side = torch.cuda.Stream()
    gbe.gbe_expectation_static(gb, Db, Hb, out[6:7], stream=side)
    side.synchronize()
    assert float(out[6]) == ref["big_H"]

    # argument errors: nothing launched
    n1 = gbe.gbe_launch_count()
    with pytest.raises(gbe.GbeError) as e:
        gbe.gbe_expectation_static(gb, Db, Hs, out[7:8])  # operand of another dimension
    assert e.value.status == -4
    assert gbe.lib().gbe_expectation_static(gb.handle, Db.data_ptr(), None, None, out.data_ptr()) == -1
    v = Hb.view()
    import ctypes as C
    assert gbe.lib().gbe_expectation_static(gb.handle, Db.data_ptr(), C.byref(v), None, None) == -1
    assert gbe.gbe_launch_count() == n1
    for g in (gb, gs):
        g.free()


def test_static_scratch_limit(gbe):
    """n == GBE_STATIC_MAX_N fills the array to its last word and works; one community more is rejected with GBE_ELIMIT
    (-7) before anything is launched, while the allocating path still takes it."""
    import torch
    nmax = gbe.GBE_STATIC_MAX_N
    assert nmax == 131072
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    for n, ok in ((nmax, True), (nmax + 8, False)):
        s = gi.chain(n, 2048, seed=1)
        Hd = gbe.DeviceCSR.from_host(s.H)
        g = gbe.gbe_build_graph(Hd, s.tau, None, s.n_part)
        gen = torch.Generator(device="cuda").manual_seed(n)
        D = torch.rand(g.info["nnz_D"], dtype=torch.float64, device="cuda", generator=gen) - 0.5
        ref = gbe.gbe_expectation(g, D, Hd)
        assert ref != 0.0
        n0 = gbe.gbe_launch_count()
        if ok:
            gbe.gbe_expectation_static(g, D, Hd, out[0:1])
            torch.cuda.synchronize()
            assert float(out[0]) == ref
        else:
            with pytest.raises(gbe.GbeError) as e:
                gbe.gbe_expectation_static(g, D, Hd, out[1:2])
            assert e.value.status == -7 and "limit" in str(e.value)
            assert gbe.gbe_launch_count() == n0 and float(out[1]) == 0.0
        g.free()
