"""Pins of the oracle's generic expression evaluator (NEXT-2) and, without a GPU, of the code generator:
the evaluator must reduce to the already pinned oracle routines on the expressions they implement
(form i, form iii, the paper's hop written exactly as Listing 1 lines 25/27, the staple sum written with
nested shifts), and the CUDA source generated for those expressions must compile for sm_100a."""
import os
import re
import shutil
import subprocess

import numpy as np
import pytest

import lattice_inputs as li
import oracle as orc
from helpers import site_rel_err

L, ADJ, MUL, ADD, SUB, SCALE, SHIFT, TRACE = range(8)


def links(seed, dims, prec="f64"):
    return [t.numpy() for t in li.gauge_field(seed, dims, prec, "haar")]


def gauss(seed, fid, dims, kind, prec="f64"):
    return li.gaussian_field(seed, fid, dims, kind, prec).numpy()


def hop_nodes():
    """sum_mu u[mu]*shift(psi,FORWARD,mu) + shift(adj(u[mu])*psi,BACKWARD,mu); leaves u0..u3 = 0..3, psi = 4"""
    n = []
    for mu in range(4):
        n += [(L, mu, 0, 0), (L, 4, 0, 0), (SHIFT, +1, mu, 0), (MUL, 0, 0, 0)]
        n += [(L, mu, 0, 0), (ADJ, 0, 0, 0), (L, 4, 0, 0), (MUL, 0, 0, 0), (SHIFT, -1, mu, 0), (ADD, 0, 0, 0)]
        if mu:
            n += [(ADD, 0, 0, 0)]
    return n


def staple_nodes(mu):
    """sum_{nu != mu} u[nu]*shift(u[mu],F,nu)*adj(shift(u[nu],F,mu)) + shift(adj(u[nu])*u[mu]*shift(u[nu],F,mu), B, nu)"""
    n, first = [], True
    for nu in range(4):
        if nu == mu:
            continue
        n += [(L, nu, 0, 0), (L, mu, 0, 0), (SHIFT, +1, nu, 0), (MUL, 0, 0, 0), (L, nu, 0, 0), (SHIFT, +1, mu, 0), (ADJ, 0, 0, 0),
              (MUL, 0, 0, 0)]
        n += [(L, nu, 0, 0), (ADJ, 0, 0, 0), (L, mu, 0, 0), (MUL, 0, 0, 0), (L, nu, 0, 0), (SHIFT, +1, mu, 0), (MUL, 0, 0, 0),
              (SHIFT, -1, nu, 0), (ADD, 0, 0, 0)]
        if not first:
            n += [(ADD, 0, 0, 0)]
        first = False
    return n


FORM_I = [(L, 0, 0, 0), (L, 1, 0, 0), (MUL, 0, 0, 0), (L, 2, 0, 0), (L, 3, 0, 0), (ADJ, 0, 0, 0), (MUL, 0, 0, 0), (ADD, 0, 0, 0)]
FORM_III = [(L, 0, 0, 0), (SCALE, 0, 0, 2.5), (L, 1, 0, 0), (SHIFT, -1, 2, 0), (SUB, 0, 0, 0)]


@pytest.mark.parametrize("dims", [(4, 6, 2, 4), (3, 5, 2, 4)])
def test_evaluator_reduces_to_the_pinned_routines(dims):
    a, b, c, d = (gauss(7, k, dims, "cm") for k in range(4))
    assert site_rel_err(orc.eval_expr(dims, FORM_I, [a, b, c, d]), orc.mm_plus_madj(dims, a, b, c, d, "t64")) < 1e-14
    assert site_rel_err(orc.eval_expr(dims, FORM_III, [a, b]), orc.ax_minus_shift(dims, 2.5, a, b, -1, 2, "t64")) < 1e-15
    u = links(2, dims)
    for kind in ("f", "cv"):
        psi = gauss(2, 10, dims, kind)
        assert site_rel_err(orc.eval_expr(dims, hop_nodes(), u + [psi]), orc.hop(dims, u, psi, "t64")) < 1e-14
    for mu in range(4):
        assert site_rel_err(orc.eval_expr(dims, staple_nodes(mu), u), orc.staple_sum(dims, u, mu, "t64")) < 1e-14
    # form ii: trace(A*B) -> LatticeComplex
    tr = orc.eval_expr(dims, [(L, 0, 0, 0), (L, 1, 0, 0), (MUL, 0, 0, 0), (TRACE, 0, 0, 0)], [a, b])
    want = orc.trace_mm(dims, a, b, "t64")
    assert tr.shape == want.shape and np.abs(tr - want).max() < 1e-13
    # the plaquette written as an expression: Re of its per-site value is the pinned per-site plaquette integrand
    pl = orc.eval_expr(dims, plaquette_nodes(), u)
    v = int(np.prod(dims))
    want = orc.plaquette_sites(dims, u, np.arange(v, dtype=np.int64), "t64")
    got = np.asarray(pl).reshape(v, -1)
    re = got[:, 0].real if np.iscomplexobj(got) else got[:, 0]
    assert np.abs(re - want).max() < 1e-12


def test_evaluator_rejects_malformed_sequences():
    a = gauss(1, 0, (2, 2, 2, 2), "cm")
    with pytest.raises(ValueError):
        orc.eval_expr((2, 2, 2, 2), [(L, 0, 0, 0), (L, 0, 0, 0)], [a])
    with pytest.raises(ValueError):
        orc.eval_expr((2, 2, 2, 2), [(L, 0, 0, 0), (99, 0, 0, 0)], [a])


# ------------------------------------------------------------------ the code generator, without a GPU
def plaquette_nodes():
    """trace( sum_{mu<nu} (u[mu]*shift(u[nu],F,mu)) * adj(u[nu]*shift(u[mu],F,nu)) ); leaves u0..u3"""
    n, first = [], True
    for mu in range(3):
        for nu in range(mu + 1, 4):
            n += [(L, mu, 0, 0), (L, nu, 0, 0), (SHIFT, +1, mu, 0), (MUL, 0, 0, 0)]
            n += [(L, nu, 0, 0), (L, mu, 0, 0), (SHIFT, +1, nu, 0), (MUL, 0, 0, 0), (ADJ, 0, 0, 0), (MUL, 0, 0, 0)]
            if not first:
                n += [(ADD, 0, 0, 0)]
            first = False
    return n + [(TRACE, 0, 0, 0)]


def _source(nodes, leaf_kinds, dst_kind, prec, accumulate=False):
    import paper_1105_2279_b200 as lqx

    e = lqx.Expr(list(nodes), list(leaf_kinds))
    return lqx.expr_source(None, dst_kind, prec, e, accumulate)


def test_generated_source_is_one_fused_kernel():
    import paper_1105_2279_b200 as lqx

    src = _source(hop_nodes(), [lqx.COLORMAT] * 4 + [lqx.FERMION], lqx.FERMION, lqx.F32)
    assert src.count("__global__") == 1 and src.count("jstore<12>") == 1
    assert src.count("const int s") == 1 + 8 and "/ g.st" not in src  # eight neighbour sites, one select each, no division
    assert src.count("jload<9>") == 8 and src.count("jload<12>") == 8
    # scalars are arguments, not text: 2.5*A - shift(B) and 7*A - shift(B) generate the same source
    s1 = _source(FORM_III, [lqx.COLORMAT] * 2, lqx.COLORMAT, lqx.F64)
    s2 = _source([(L, 0, 0, 0), (SCALE, 0, 0, 7.0), (L, 1, 0, 0), (SHIFT, -1, 2, 0), (SUB, 0, 0, 0)], [lqx.COLORMAT] * 2,
                 lqx.COLORMAT, lqx.F64)
    assert s1 == s2 and "2.5" not in s1
    # accumulate ('+=', E2 of the Listing) reads the destination
    assert "jload<12, true>(dst, s0)" in _source(hop_nodes(), [lqx.COLORMAT] * 4 + [lqx.FERMION], lqx.FERMION, lqx.F32, True)


def test_generator_type_and_shape_errors():
    import paper_1105_2279_b200 as lqx

    with pytest.raises(lqx.LqxError):  # vector * matrix
        _source([(L, 0, 0, 0), (L, 1, 0, 0), (MUL, 0, 0, 0)], [lqx.COLORVEC, lqx.COLORMAT], lqx.COLORVEC, lqx.F32)
    with pytest.raises(lqx.LqxError):  # adj of a vector
        _source([(L, 0, 0, 0), (ADJ, 0, 0, 0)], [lqx.COLORVEC], lqx.COLORVEC, lqx.F32)
    with pytest.raises(lqx.LqxError):  # matrix + vector
        _source([(L, 0, 0, 0), (L, 1, 0, 0), (ADD, 0, 0, 0)], [lqx.COLORMAT, lqx.COLORVEC], lqx.COLORMAT, lqx.F32)
    with pytest.raises(lqx.LqxError):  # destination kind
        _source(FORM_I, [lqx.COLORMAT] * 4, lqx.COLORVEC, lqx.F32)
    with pytest.raises(lqx.LqxError):  # does not reduce to one value
        _source([(L, 0, 0, 0), (L, 0, 0, 0)], [lqx.COLORMAT], lqx.COLORMAT, lqx.F32)
    with pytest.raises(lqx.LqxError):  # shift direction
        _source([(L, 0, 0, 0), (SHIFT, 2, 0, 0)], [lqx.COLORMAT], lqx.COLORMAT, lqx.F32)


@pytest.mark.skipif(shutil.which("nvcc") is None and not os.path.exists("/usr/local/cuda/bin/nvcc"), reason="no nvcc")
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_generated_source_compiles_for_sm_100a(tmp_path, prec):
    import paper_1105_2279_b200 as lqx

    pc = lqx.F32 if prec == "f32" else lqx.F64
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    cases = {"hop": (hop_nodes(), [lqx.COLORMAT] * 4 + [lqx.FERMION], lqx.FERMION),
             "staple": (staple_nodes(1), [lqx.COLORMAT] * 4, lqx.COLORMAT),
             "form_iii": (FORM_III, [lqx.COLORMAT] * 2, lqx.COLORMAT)}
    sources = {name: _source(nodes, kinds, dk, pc) for name, (nodes, kinds, dk) in cases.items()}
    e = lqx.Expr([(L, 0, 0, 0), (L, 1, 0, 0), (MUL, 0, 0, 0), (TRACE, 0, 0, 0)], [lqx.COLORMAT] * 2)
    sources["trace_mm"] = lqx.expr_source(None, lqx.COMPLEX, pc, e)
    sources["norm2_hop"] = lqx.expr_source(None, lqx.FERMION, pc, lqx.Expr(hop_nodes(), [lqx.COLORMAT] * 4 + [lqx.FERMION]), reduce=1)
    sources["sum_form_i"] = lqx.expr_source(None, lqx.COLORMAT, pc, lqx.Expr(list(FORM_I), [lqx.COLORMAT] * 4), reduce=2)
    sources["sum_plaquette"] = lqx.expr_source(None, lqx.COMPLEX, pc, lqx.Expr(plaquette_nodes(), [lqx.COLORMAT] * 4), reduce=2)
    assert "jreduce<1>" in sources["norm2_hop"] and "jreduce<18>" in sources["sum_form_i"] and "jstore" not in sources["norm2_hop"].split("lqx_jit")[1]
    for name, text in sources.items():
        f = tmp_path / f"{name}_{prec}.cu"
        f.write_text(text)
        r = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-std=c++17", "-Xptxas", "-v", "-cubin", "-o",
                            str(f) + ".cubin", str(f)], capture_output=True, text=True)
        assert r.returncode == 0, r.stderr[-3000:]
        # the CTAs-per-SM bound follows the expression's register need: nothing beyond a few spilled words
        spill = [int(x) for x in re.findall(r"(\d+) bytes spill stores", r.stderr)]
        assert spill and max(spill) <= 64, (name, r.stderr[-600:])


def test_launch_bounds_follow_the_register_need():
    import paper_1105_2279_b200 as lqx

    def blocks(src):
        return int(re.search(r"__launch_bounds__\(128, (\d+)\)", src).group(1))

    cm4, f = [lqx.COLORMAT] * 4, lqx.FERMION
    # accumulator + one matrix + one fermion: six CTAs of 128 threads per SM in fp32 (85 registers), three in fp64
    assert blocks(_source(hop_nodes(), cm4 + [f], f, lqx.F32)) == 6
    assert blocks(_source(hop_nodes(), cm4 + [f], f, lqx.F64)) == 3
    # a product of products under a sum needs four matrices and the accumulator live: fewer CTAs, no spills
    assert blocks(lqx.expr_source(None, lqx.COMPLEX, lqx.F32, lqx.Expr(plaquette_nodes(), cm4), reduce=2)) <= 4
    assert blocks(lqx.expr_source(None, lqx.COMPLEX, lqx.F64, lqx.Expr(plaquette_nodes(), cm4), reduce=2)) == 2
