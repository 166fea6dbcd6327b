"""lqx_norm2_noalloc (include/lqx.h): the allocation-free norm2, whose reduction scratch is a file-scope __device__
array, against the existing lqx_norm2 (context-owned, cudaMalloc'ed scratch) on the same fields -- two calls in a row,
because all calls share the one array and it keeps the last call's contents.  Named test_zz_* so that pytest collects
it last: `pytest -x` stops at the first failure, and one here must not hide the parity tests.  Needs nothing from the
other tests (own contexts, own inputs): passes alone in a fresh process and after the rest of the suite."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle as orc

pytestmark = pytest.mark.gpu

# Both paths add the same fp64 squares of the same stored values and differ in the summation tree only (test_gpu_parity:
# "fused == two-call up to summation order" uses the same bound); against the oracle the suite's reduction tolerance holds.
TREE_TOL = 1e-13
RTOL = {"f32": 1e-4, "f64": 1e-10}


@pytest.fixture(scope="module")
def lqx():
    import paper_1105_2279_b200 as m

    return m


def _field(lat, seed, fid, dims, kind, prec):
    a = li.gaussian_field(seed, fid, dims, kind, prec).numpy()
    return a, lat.from_host(a)


# one CTA with a ragged tail (V = 1680 < 2048 sites per CTA), a full CTA plus a partly filled one (V = 2304), and
# 64 CTAs (16^3 x 32, BASELINE.json configs[1])
@pytest.mark.parametrize("dims", [(6, 5, 7, 8), (8, 6, 6, 8), (16, 16, 16, 32)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_noalloc_norm2_equals_the_existing_path_twice_in_a_row(lqx, dims, prec):
    import torch

    with lqx.Lattice(dims) as lat:
        a, fa = _field(lat, 31, 0, dims, "f", prec)
        b, fb = _field(lat, 31, 1, dims, "cm", prec)
        want_a, want_b = lqx.norm2(fa), lqx.norm2(fb)
        out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
        # first call, then a second one straight behind it on a DIFFERENT field (stale partials must not leak),
        # then the first field again: the shared scratch holds the previous call's contents each time
        lqx.norm2_noalloc(fa, out.data_ptr())
        lqx.norm2_noalloc(fb, out.data_ptr() + 8)
        got_a, got_b = (float(v) for v in out.cpu())
        lqx.norm2_noalloc(fa, out.data_ptr() + 8)
        got_a2 = float(out.cpu()[1])
        assert abs(got_a - want_a) <= TREE_TOL * want_a, (got_a, want_a)
        assert abs(got_b - want_b) <= TREE_TOL * want_b, (got_b, want_b)
        assert got_a2 == got_a  # fixed summation tree: bit-reproducible call to call
        # and against the oracle, at the tolerance of the suite's reduction tests
        tv = orc.truth_variant(prec)
        for got, arr in ((got_a, a), (got_b, b)):
            want = orc.norm2(dims, arr, tv)
            assert abs(got - want) / want < RTOL[prec]


def test_noalloc_norm2_all_kinds_and_full_size(lqx):
    """every field kind once, on a lattice of several hundred CTAs (32^3 x 64, BASELINE.json configs[2] geometry)"""
    import torch

    dims = (32, 32, 32, 64)
    with lqx.Lattice(dims) as lat:
        out = torch.zeros(1, dtype=torch.float64, device="cuda")
        for fid, kind in enumerate(["c", "cv", "cm", "f"]):
            _, f = _field(lat, 32, fid, dims, kind, "f32")
            want = lqx.norm2(f)
            for _ in range(2):
                out.fill_(-1.0)
                lqx.norm2_noalloc(f, out.data_ptr())
                got = float(out.cpu()[0])
                assert abs(got - want) <= TREE_TOL * want, (kind, got, want)


def test_noalloc_norm2_rejects_a_lattice_beyond_the_static_scratch(lqx):
    import torch

    dims = (64, 64, 64, 96)  # 25.2 M sites > LQX_NOALLOC_MAX_SITES = 2^24
    assert int(np.prod(dims)) > lqx.NOALLOC_MAX_SITES
    with lqx.Lattice(dims) as lat:
        f = lat.alloc(lqx.COMPLEX, lqx.F32)
        out = torch.full((1,), -7.0, dtype=torch.float64, device="cuda")
        with pytest.raises(lqx.LqxError) as e:
            lqx.norm2_noalloc(f, out.data_ptr())
        assert "static scratch" in str(e.value) and "LQX_NOALLOC_MAX_SITES" in str(e.value)
        torch.cuda.synchronize()
        assert float(out.cpu()[0]) == -7.0  # nothing was launched
        with pytest.raises(lqx.LqxError):
            lqx.norm2_noalloc(f, 0)  # null output
    # the entry point still works after the rejected calls
    small = (4, 4, 4, 4)
    with lqx.Lattice(small) as lat:
        _, g = _field(lat, 33, 0, small, "cv", "f64")
        o = torch.zeros(1, dtype=torch.float64, device="cuda")
        lqx.norm2_noalloc(g, o.data_ptr())
        assert abs(float(o.cpu()[0]) - lqx.norm2(g)) <= TREE_TOL * lqx.norm2(g)
