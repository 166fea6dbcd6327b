"""GPU parity: the CUDA path (through the C-ABI, via the thin binding) against the CPU oracle,
element by element on the same seeded inputs.  Index / copy work is bit-exact; floating point is
compared with the DESIGN.md A14 site-normalised error against the WIDE-arithmetic oracle variant
(t32 / t64), tolerance 1e-5 (fp32) and 1e-12 (fp64) as BASELINE.json north_star states; reductions
1e-4 / 1e-10 with the A15 normalisation."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle as orc
from helpers import cplx, site_rel_err

pytestmark = pytest.mark.gpu

TOL = {"f32": 1e-5, "f64": 1e-12}
RTOL = {"f32": 1e-4, "f64": 1e-10}
# several tiles + a ragged tail (V = 1680, not a multiple of 32 or 128), odd extents, L0 % 4 != 0
DIMS_RAGGED = (6, 5, 7, 8)
DIMS_EVEN = (8, 4, 6, 4)
ALL_DIMS = [(2, 2, 2, 2), (4, 4, 4, 4), DIMS_RAGGED, DIMS_EVEN, (3, 1, 2, 5)]


@pytest.fixture(scope="module")
def lqx():
    import paper_1105_2279_b200 as m

    return m


def _prec(lqx, prec):
    return {"f32": lqx.F32, "f64": lqx.F64}[prec]


def _np(t):
    return t.numpy()


def _gauss(seed, fid, dims, kind, prec):
    return _np(li.gaussian_field(seed, fid, dims, kind, prec))


def _links(seed, dims, prec, recipe="haar"):
    return [_np(t) for t in li.gauge_field(seed, dims, prec, recipe)]


# ------------------------------------------------------------------------------------------------
# a1 geometry
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", ALL_DIMS + [(16, 16, 16, 32), (32, 32, 32, 64), (48, 48, 48, 96)])
def test_neighbor_tables_bit_exact(lqx, dims):
    with lqx.Lattice(dims) as lat:
        for mu in range(4):
            for d in (+1, -1):
                got = lat.neighbor_table(d, mu)
                want = orc.neighbor_table(dims, d, mu)
                assert np.array_equal(got, want), (dims, mu, d)


# ------------------------------------------------------------------------------------------------
# a2 field store
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [DIMS_RAGGED, (4, 4, 4, 4)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("kind", ["c", "cv", "cm", "f"])
def test_push_pop_round_trip_bit_exact(lqx, dims, prec, kind):
    a = _gauss(11, 0, dims, kind, prec)
    with lqx.Lattice(dims) as lat:
        f = lat.from_host(a)
        assert np.array_equal(f.pop(), a)
        g = lat.alloc(f.kind, f.prec, torch_memory=False)  # library-owned memory path
        g.push(a)
        assert np.array_equal(g.pop(), a)
        lqx.copy(g, f)
        assert np.array_equal(g.pop(), a)


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("kind", ["c", "cv", "cm", "f"])
def test_internal_layout_is_blocked_site_fastest_soa(lqx, prec, kind):
    """include/lqx.h: blocks of 32 sites, 128-bit chunks of the site object, chunk q of the 32 sites
    contiguous.  The expected offsets are recomputed here from that sentence, not from the library."""
    import torch

    dims = (6, 2, 3, 2)  # V = 72: two full blocks and a ragged one
    a = _gauss(5, 0, dims, kind, prec)
    v = a.shape[0]
    nreal = a.reshape(v, -1).shape[1]
    w = 4 if prec == "f32" else 2
    nfull = nreal // w
    with lqx.Lattice(dims) as lat:
        f = lat.from_host(a)
        torch.cuda.synchronize()
        assert lat.padded_volume % 32 == 0 and lat.volume <= lat.padded_volume < lat.volume + 32
        assert lat.field_bytes(f.kind, f.prec) == lat.padded_volume * nreal * (4 if prec == "f32" else 8)
        raw = f._mem.view(torch.float32 if prec == "f32" else torch.float64).cpu().numpy()
        flat = a.reshape(v, nreal)
        expect = np.zeros(lat.padded_volume * nreal, dtype=flat.dtype)
        for s in range(v):
            for r in range(nreal):
                q = min(r // w, nfull)
                wq = w if q < nfull else nreal - nfull * w
                off = (s // 32) * 32 * nreal + q * 32 * w + (s % 32) * wq + (r - q * w)
                expect[off] = flat[s, r]
                assert lat.field_offset(f.kind, f.prec, s, r) == off
        assert np.array_equal(raw, expect)  # pad lanes of the last block are zero


# ------------------------------------------------------------------------------------------------
# a3 shift (bit-exact) and a5 form (iii)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [DIMS_RAGGED, DIMS_EVEN, (2, 2, 2, 2)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_shift_bit_exact_all_directions(lqx, dims, prec):
    with lqx.Lattice(dims) as lat:
        for kind in ("cm", "f", "c"):
            a = _gauss(3, 1, dims, kind, prec)
            fa = lat.from_host(a)
            fr = lat.alloc(fa.kind, fa.prec)
            for mu in range(4):
                for d in (+1, -1):
                    lqx.shift(fr, fa, d, mu)
                    assert np.array_equal(fr.pop(), orc.shift(dims, a, d, mu)), (kind, mu, d)
            # round trip
            fb = lat.alloc(fa.kind, fa.prec)
            lqx.shift(fr, fa, +1, 2)
            lqx.shift(fb, fr, -1, 2)
            assert np.array_equal(fb.pop(), a)


@pytest.mark.parametrize("dims", [DIMS_RAGGED, DIMS_EVEN])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_form_iii_ax_minus_shift(lqx, dims, prec):
    a, b = _gauss(7, 0, dims, "cm", prec), _gauss(7, 1, dims, "cm", prec)
    with lqx.Lattice(dims) as lat:
        fa, fb = lat.from_host(a), lat.from_host(b)
        fr = lat.alloc(lqx.COLORMAT, _prec(lqx, prec))
        for (d, mu) in [(-1, 2), (+1, 0), (-1, 0), (+1, 3), (-1, 1)]:
            lqx.ax_minus_shift(fr, 2.5, fa, fb, d, mu)
            got = fr.pop()
            # same operations in the same precision: bit-exact against the native oracle
            assert np.array_equal(got, orc.ax_minus_shift(dims, 2.5, a, b, d, mu, orc.native_variant(prec)))
            assert site_rel_err(got, orc.ax_minus_shift(dims, 2.5, a, b, d, mu, orc.truth_variant(prec))) < TOL[prec]


# ------------------------------------------------------------------------------------------------
# a4 site-local catalogue
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [DIMS_RAGGED, DIMS_EVEN])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_forms_i_ii_iv(lqx, dims, prec):
    tv = orc.truth_variant(prec)
    a, b, c, d = (_gauss(7, k, dims, "cm", prec) for k in range(4))
    v = _gauss(7, 4, dims, "cv", prec)
    psi = _gauss(7, 5, dims, "f", prec)
    with lqx.Lattice(dims) as lat:
        fa, fb, fc, fd, fv, fp = (lat.from_host(t) for t in (a, b, c, d, v, psi))
        r = lat.alloc(lqx.COLORMAT, fa.prec)
        lqx.mm_plus_madj(r, fa, fb, fc, fd)
        assert site_rel_err(r.pop(), orc.mm_plus_madj(dims, a, b, c, d, tv)) < TOL[prec]
        t = lat.alloc(lqx.COMPLEX, fa.prec)
        lqx.trace_mm(t, fa, fb)
        # form ii reduces nine products to ONE complex number per site: measured against the size of what was
        # summed, sum_ik |A_ik| |B_ki| (reading A14 with the summands as the site object), at the flat tolerance
        mag = np.einsum("xik,xki->x", np.abs(cplx(a)), np.abs(cplx(b)))
        assert float((np.abs(t.pop().astype(np.float64) - orc.trace_mm(dims, a, b, tv)).max(axis=1) / mag).max()) < TOL[prec]
        w = lat.alloc(lqx.COLORVEC, fa.prec)
        lqx.mat_vec(w, fa, fv)
        assert site_rel_err(w.pop(), orc.mat_vec(dims, a, v, tv)) < TOL[prec]
        wf = lat.alloc(lqx.FERMION, fa.prec)
        lqx.mat_vec(wf, fa, fp)
        assert site_rel_err(wf.pop(), orc.mat_vec(dims, a, psi, tv)) < TOL[prec]
        # in-place site-local evaluation is allowed (reading A21)
        lqx.mm_plus_madj(fa, fa, fb, fc, fd)
        assert site_rel_err(fa.pop(), orc.mm_plus_madj(dims, a, b, c, d, tv)) < TOL[prec]


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_axpy_scale_divide(lqx, prec):
    dims = DIMS_RAGGED
    tv = orc.truth_variant(prec)
    s0, h = _gauss(9, 0, dims, "f", prec), _gauss(9, 1, dims, "f", prec)
    with lqx.Lattice(dims) as lat:
        f0, fh = lat.from_host(s0), lat.from_host(h)
        r = lat.alloc(lqx.FERMION, f0.prec)
        lqx.axpy(r, f0, 0.37, fh)
        assert site_rel_err(r.pop(), orc.axpy(dims, s0, 0.37, h, tv)) < TOL[prec]
        lqx.scale(r, -1.75, f0)
        assert np.array_equal(r.pop(), orc.scale(dims, -1.75, s0, orc.native_variant(prec)))
        lqx.divide(r, f0, 3.3)
        assert site_rel_err(r.pop(), orc.divide(dims, 3.3, s0, tv)) < TOL[prec]


# ------------------------------------------------------------------------------------------------
# a9 reductions
# ------------------------------------------------------------------------------------------------
def _red_err(got, want, scale):
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    return float(np.abs(got - want).max() / max(np.abs(want).max(), scale))


@pytest.mark.parametrize("dims", [DIMS_RAGGED, (16, 8, 8, 8)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_reductions(lqx, dims, prec):
    tv = orc.truth_variant(prec)
    with lqx.Lattice(dims) as lat:
        for kind in ("c", "cv", "cm", "f"):
            a = _gauss(13, 2, dims, kind, prec)
            f = lat.from_host(a)
            rms = float(np.sqrt((a.astype(np.float64) ** 2).sum()))  # A15: sqrt(sum term^2)
            assert _red_err(lqx.sum(f), orc.sum_field(dims, a, tv), rms) < RTOL[prec]
            n2 = lqx.norm2(f)
            assert abs(n2 - orc.norm2(dims, a, tv)) / orc.norm2(dims, a, tv) < RTOL[prec]
            if kind == "cm":
                assert _red_err(lqx.trace(f), orc.trace(dims, a, tv), rms) < RTOL[prec]
            # deterministic: same bits on a second call
            assert lqx.norm2(f) == n2


# ------------------------------------------------------------------------------------------------
# a6 hop
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [DIMS_RAGGED, DIMS_EVEN, (2, 2, 2, 2)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_hop(lqx, dims, prec):
    tv = orc.truth_variant(prec)
    u = _links(2, dims, prec)
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        for kind in ("f", "cv"):
            psi = _gauss(2, 10, dims, kind, prec)
            fp = lat.from_host(psi)
            chi = lat.alloc(fp.kind, fp.prec)
            want = orc.hop(dims, u, psi, tv)
            lqx.hop(chi, fu, fp)
            assert site_rel_err(chi.pop(), want) < TOL[prec]
            n2 = lqx.hop_norm2(chi, fu, fp)
            assert site_rel_err(chi.pop(), want) < TOL[prec]
            want_n2 = float((want.astype(np.float64) ** 2).sum())
            assert abs(n2 - want_n2) / want_n2 < RTOL[prec]
            assert abs(n2 - lqx.norm2(chi)) / want_n2 < 1e-13  # fused == two-call up to summation order


def test_hop_and_smear_step_captured_in_a_cuda_graph(lqx):
    """The asynchronous calls do nothing but enqueue kernels on the context's stream, so a user can capture them
    into a CUDA graph (graph-amortised launches).  The replayed graph must reproduce the direct
    calls bit for bit -- and those are checked against the oracle here as well."""
    import torch

    dims, prec = DIMS_RAGGED, "f32"
    u = _links(2, dims, prec)
    psi = _gauss(2, 10, dims, "f", prec)
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        fo = [lat.alloc(lqx.COLORMAT, lqx.F32) for _ in range(4)]
        fp = lat.from_host(psi)
        chi = lat.alloc(fp.kind, fp.prec)
        lqx.hop(chi, fu, fp)
        lqx.smear_step(fo, fu, 0.5)
        direct_chi = chi.pop()
        direct_u = [f.pop() for f in fo]
        assert site_rel_err(direct_chi, orc.hop(dims, u, psi, "t32")) < TOL[prec]
        side = torch.cuda.Stream()
        lat.set_stream(side)
        try:
            with torch.cuda.stream(side):
                lqx.copy(chi, fp)            # overwrite the results so that only the replay can restore them
                for f, g in zip(fo, fu):
                    lqx.copy(f, g)
                n0 = lat.launch_count()
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=side):
                    lqx.hop(chi, fu, fp)
                    lqx.smear_step(fo, fu, 0.5)
                assert lat.launch_count() - n0 == 2
                side.synchronize()
                assert not np.array_equal(chi.pop(), direct_chi)  # capture enqueued nothing
                graph.replay()
                side.synchronize()
            assert np.array_equal(chi.pop(), direct_chi)
            for f, d in zip(fo, direct_u):
                assert np.array_equal(f.pop(), d)
        finally:
            torch.cuda.synchronize()
            lat.set_stream(torch.cuda.current_stream())


def test_c2_hop_full_size(lqx):
    """BASELINE.json configs[1]: 16^3x32 fp32, Haar links, Gaussian fermion; hop then norm2."""
    cfg = li.CONFIGS["c2"]
    dims = cfg["dims"]
    u = _links(cfg["seed"], dims, "f32")
    psi = _gauss(cfg["seed"], 10, dims, "f", "f32")
    want = orc.hop(dims, u, psi, "t32")
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        fp = lat.from_host(psi)
        chi = lat.alloc(lqx.FERMION, lqx.F32)
        n2 = lqx.hop_norm2(chi, fu, fp)
        got = chi.pop()
    assert site_rel_err(got, want) < TOL["f32"]
    want_n2 = float((want ** 2).sum())
    assert abs(n2 - want_n2) / want_n2 < RTOL["f32"]


# ------------------------------------------------------------------------------------------------
# a7 / a8 / a10 staple, smear, plaquette
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), DIMS_RAGGED, DIMS_EVEN, (2, 2, 2, 2), (3, 1, 2, 5)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_staple_smear_plaquette(lqx, dims, prec):
    tv = orc.truth_variant(prec)
    u = _links(1, dims, prec)
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        out = [lat.alloc(lqx.COLORMAT, fu[0].prec) for _ in range(4)]
        st = lat.alloc(lqx.COLORMAT, fu[0].prec)
        for mu in range(4):
            lqx.staple_sum(st, fu, mu)
            assert site_rel_err(st.pop(), orc.staple_sum(dims, u, mu, tv)) < TOL[prec]
        want = orc.smear_step(dims, u, 0.5, tv)
        psum_want = orc.plaquette_sum(dims, u, tv)
        scale = np.sqrt(18.0 * lat.volume)  # A15: size of a zero-mean Haar plaquette sum
        for want_plaq in (False, True):
            for o in out:
                lqx.scale(o, 0.0, o)
            p = lqx.smear_step(out, fu, 0.5, want_plaq_in=want_plaq)
            for mu in range(4):
                assert site_rel_err(out[mu].pop(), want[mu]) < TOL[prec], (mu, want_plaq)
            if want_plaq:
                assert abs(p - psum_want) / max(abs(psum_want), scale) < RTOL[prec]
        for variant in (0, 1, 2):  # option plaq_variant: automatic, rolled loops, the site's links held in registers
            lat.set_option("plaq_variant", variant)
            ps, pa = lqx.plaquette(fu)
            assert abs(ps - psum_want) / max(abs(psum_want), scale) < RTOL[prec], variant
            assert abs(pa - psum_want / (18.0 * lat.volume)) < RTOL[prec], variant
        lat.set_option("plaq_variant", 0)
        # plaquette of the smeared field (A11)
        ps2, _ = lqx.plaquette(out)
        w2 = orc.plaquette_sum(dims, want, "t64" if prec == "f64" else "n64")
        assert abs(ps2 - w2) / max(abs(w2), scale) < RTOL[prec]


# every smear kernel variant (option "smear_variant": 1 literal gather, 2 shared-corner with the lower
# staples exchanged through shared memory, 3 rolled literal = default, 4 four threads per site, 6 operands
# staged in shared memory, 7 the tile's own links in shared memory and the halo through L1, 8 plane-ordered 42-product evaluation on
# whole-x-row tiles in shared memory with persistent double-buffered CTAs, 9 the literal evaluation on row tiles, 10 the same
# with the upper staples' common factors kept in tensor memory: 42 products) and every
# CTA tile shape that divides the lattice, against the truth oracle; 16x8x4x4 spans several tiles in every
# direction for all shapes, 8x4x4x2 is exactly one 8x4x4x2 tile (every neighbour wraps into the same tile); 12x6x4x2 has
# row tiles of 96 threads and y-tiles of 2 and 3 rows, 6x4x2x4 has rows that are not whole warps (the row-tile kernels
# hand over to the rolled kernel there)
@pytest.mark.parametrize("dims", [(16, 8, 4, 4), (8, 4, 4, 2), (4, 4, 4, 4), (12, 6, 4, 2), (6, 4, 2, 4)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("variant", [1, 2, 3, 4, 6, 7, 8, 9, 10])
def test_smear_variants_and_tiles(lqx, dims, prec, variant):
    tv = orc.truth_variant(prec)
    u = _links(5, dims, prec)
    want = orc.smear_step(dims, u, 0.5, tv)
    psum_want = orc.plaquette_sum(dims, u, tv)
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        out = [lat.alloc(lqx.COLORMAT, fu[0].prec) for _ in range(4)]
        scale = np.sqrt(18.0 * lat.volume)
        lat.set_option("smear_variant", variant)
        first = None
        for tile in (-1, 0, 1, 2, 3, 4, 5, 6, 7):
            lat.set_option("tile", tile)
            for o in out:
                lqx.scale(o, 0.0, o)
            p = lqx.smear_step(out, fu, 0.5, want_plaq_in=True)
            got = [o.pop() for o in out]
            for mu in range(4):
                assert site_rel_err(got[mu], want[mu]) < TOL[prec], (variant, tile, mu)
            assert abs(p - psum_want) / max(abs(psum_want), scale) < RTOL[prec], (variant, tile)
            # run to run, and whatever the tile shape of a given variant, the per-site arithmetic is fixed
            lqx.smear_step(out, fu, 0.5, want_plaq_in=True)
            for mu in range(4):
                assert np.array_equal(out[mu].pop(), got[mu]), (variant, tile, mu)
            if variant in (1, 3, 6, 7, 9):  # variants 6 and 7 add their staples in variant 3's order; variant 2 sums in an order that depends on the tile faces; 2 and 4 fall back to 3 for tiles they lack
                if first is None:
                    first = got
                for mu in range(4):
                    assert np.array_equal(got[mu], first[mu]), (variant, tile, mu)


# option "bulk_fill": the row-tile kernel's tile filled by TMA bulk copies (cp.async.bulk + mbarrier) instead of per-thread
# cp.async, on lattices whose tile rows are whole 32-site blocks (16 and 32 sites per row; several tiles in z and t) --
# same bytes in shared memory, so the output must be bit-identical, and it must agree with the oracle
@pytest.mark.parametrize("dims", [(16, 8, 4, 4), (32, 4, 4, 6)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_smear_row_tile_bulk_fill(lqx, dims, prec):
    tv = orc.truth_variant(prec)
    u = _links(6, dims, prec)
    want = orc.smear_step(dims, u, 0.5, tv)
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        out = [lat.alloc(lqx.COLORMAT, fu[0].prec) for _ in range(4)]
        lat.set_option("smear_variant", 9)
        got = {}
        for bulk in (0, 1):
            lat.set_option("bulk_fill", bulk)
            for o in out:
                lqx.scale(o, 0.0, o)
            p = lqx.smear_step(out, fu, 0.5, want_plaq_in=True)
            assert lat.smear_info()[2].startswith("k_smear_rowlit")
            got[bulk] = ([o.pop() for o in out], p)
        for mu in range(4):
            assert site_rel_err(got[1][0][mu], want[mu]) < TOL[prec], mu
            assert np.array_equal(got[1][0][mu], got[0][0][mu]), mu
        assert got[1][1] == got[0][1]


# variant 10 (upper-staple factors kept in tensor memory): without the fused plaquette, on eight-row and four-row tiles
# (odd t-extent), and on ranges of time slices with even and odd boundaries -- every launch shape evaluates the same per-site
# arithmetic, so the ranges put together equal the whole-lattice step bit for bit; rows of 48, 16 and 8 sites
@pytest.mark.parametrize("dims", [(48, 4, 4, 6), (16, 4, 6, 5), (8, 4, 4, 4)])
def test_smear_variant_10_ranges_and_no_plaquette(lqx, dims):
    prec = "f32"
    tv = orc.truth_variant(prec)
    u = _links(7, dims, prec)
    want = orc.smear_step(dims, u, 0.5, tv)
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        out = [lat.alloc(lqx.COLORMAT, fu[0].prec) for _ in range(4)]
        lat.set_option("smear_variant", 10)
        lqx.smear_step(out, fu, 0.5, want_plaq_in=False)
        assert lat.smear_info()[2] == "k_smear_rowz"
        full = [o.pop() for o in out]
        for mu in range(4):
            assert site_rel_err(full[mu], want[mu]) < TOL[prec], mu
        lqx.smear_step(out, fu, 0.5, want_plaq_in=True)
        for mu in range(4):
            assert np.array_equal(out[mu].pop(), full[mu]), mu
        L3 = dims[3]
        for cuts in ([0, 2, L3], [0, 1, 3, L3], [0, L3 - 1, L3]):
            for o in out:
                lqx.scale(o, 0.0, o)
            for t0, t1 in zip(cuts[:-1], cuts[1:]):
                lqx.smear_step_range(out, fu, 0.5, t0, t1)
            for mu in range(4):
                assert np.array_equal(out[mu].pop(), full[mu]), (cuts, mu)


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_unit_gauge_is_a_fixed_point(lqx, prec):
    dims = DIMS_EVEN
    u = _links(0, dims, prec, "unit")
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        st = lat.alloc(lqx.COLORMAT, fu[0].prec)
        lqx.staple_sum(st, fu, 1)
        six = 6.0 * u[0]
        assert np.array_equal(st.pop(), six)  # every staple is the identity: S = 6*1 exactly
        out = [lat.alloc(lqx.COLORMAT, fu[0].prec) for _ in range(4)]
        p = lqx.smear_step(out, fu, 0.5, want_plaq_in=True)
        for mu in range(4):
            assert np.abs(out[mu].pop() - u[mu]).max() < (1e-7 if prec == "f32" else 1e-15)
        assert p == 18.0 * lat.volume
        assert lqx.plaquette(fu)[1] == 1.0


@pytest.mark.parametrize("prec,nsteps", [("f32", 4), ("f64", 3), ("f32", 1)])
def test_smear_iterate_trajectory(lqx, prec, nsteps):
    """configs[3] in miniature: near-unit links, iterated steps, plaquette after each (A23)."""
    dims = (8, 6, 4, 6)
    u = _links(4, dims, prec, "near_unit")
    want_u, want_p = orc.smear_iterate(dims, u, 0.5, nsteps, prec)
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        tmp = [lat.alloc(lqx.COLORMAT, fu[0].prec) for _ in range(4)]
        plaqs = lqx.smear_iterate(fu, tmp, 0.5, nsteps)
        for k in range(nsteps):
            assert abs(plaqs[k] - want_p[k]) < RTOL[prec], k
        for mu in range(4):
            assert site_rel_err(fu[mu].pop(), want_u[mu]) < TOL[prec] * nsteps
        # no projection back to SU(3) (reading A9): the links shrink, so nothing is asserted about
        # the direction in which the plaquette moves -- only agreement with the oracle's trajectory


def test_smear_iterate_host_end_to_end(lqx):
    dims = (4, 4, 4, 8)
    u = _links(4, dims, "f32", "near_unit")
    want_u, want_p = orc.smear_iterate(dims, u, 0.5, 2, "f32")
    out = [np.empty_like(t) for t in u]
    with lqx.Lattice(dims) as lat:
        plaqs = lqx.smear_iterate_host(lat, lqx.F32, u, out, 0.5, 2)
    for k in range(2):
        assert abs(plaqs[k] - want_p[k]) < RTOL["f32"]
    for mu in range(4):
        assert site_rel_err(out[mu], want_u[mu]) < TOL["f32"] * 2  # two iterated steps: reading A23


# The one-step host call streams the lattice through the GPU in slabs of time slices (upload, smear and download of
# different slabs overlap).  It must give exactly what the serial push / step / pop path gives -- same kernel, same
# per-site arithmetic -- on every tile map, including the wrap-around slabs, and agree with the oracle.
@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("dims,slabs", [((8, 8, 8, 16), 48), ((8, 8, 8, 16), 4), ((4, 4, 4, 8), 48),
                                        ((6, 6, 6, 12), 48), ((16, 4, 4, 6), 48), ((8, 4, 4, 24), 3)])
def test_smear_host_streamed_equals_serial_and_oracle(lqx, dims, slabs, prec):
    u = _links(11, dims, prec, "near_unit")
    code = lqx.F32 if prec == "f32" else lqx.F64
    serial = [np.empty_like(t) for t in u]
    streamed = [np.full_like(t, np.nan) for t in u]
    with lqx.Lattice(dims) as lat:
        lat.set_option("host_slabs", 0)
        p_serial = lqx.smear_iterate_host(lat, code, u, serial, 0.4, 1)
        lat.set_option("host_slabs", slabs)
        n0 = lat.launch_count()
        p_streamed = lqx.smear_iterate_host(lat, code, u, streamed, 0.4, 1)
        n_streamed = lat.launch_count() - n0
        # second call on the same context (events, streams and staging fields are reused), in place
        inplace = [t.copy() for t in u]
        p_inplace = lqx.smear_iterate_host(lat, code, inplace, inplace, 0.4, 1)
    # the serial path launches 4 + 1 + 4 + 2 + 4 kernels; a streamed call launches 9 per slab + 2
    assert n_streamed > 17, "the streamed path did not run for this lattice"
    for mu in range(4):
        assert np.array_equal(serial[mu], streamed[mu])
        assert np.array_equal(serial[mu], inplace[mu])
    assert p_serial == p_streamed == p_inplace
    want_u, want_p = orc.smear_iterate(dims, u, 0.4, 1, prec)
    assert abs(p_streamed[0] - want_p[0]) < RTOL[prec]
    for mu in range(4):
        assert site_rel_err(streamed[mu], want_u[mu]) < TOL[prec]


def test_smear_host_streams_by_default_at_production_slab_sizes(lqx):
    # automatic setting: 32^3 x 64 in fp32 has 4.7 MB per link in a two-slice slab -> 32 slabs
    dims = (32, 32, 32, 64)
    u = _links(13, dims, "f32", "near_unit")
    serial = [np.empty_like(t) for t in u]
    streamed = [np.empty_like(t) for t in u]
    with lqx.Lattice(dims) as lat:
        n0 = lat.launch_count()
        p_streamed = lqx.smear_iterate_host(lat, lqx.F32, u, streamed, 0.4, 1)
        assert lat.launch_count() - n0 == 32 * 9 + 2
        lat.set_option("host_slabs", 0)
        p_serial = lqx.smear_iterate_host(lat, lqx.F32, u, serial, 0.4, 1)
    assert p_serial == p_streamed
    for mu in range(4):
        assert np.array_equal(serial[mu], streamed[mu])


@pytest.mark.parametrize("slabs", [-1, 48])
def test_smear_host_falls_back_to_serial_when_slabs_do_not_fit(lqx, slabs):
    # 6^3 x 6: no even slab thickness gives a multiple of 32 sites and at least three slabs (and, on the automatic
    # setting, a lattice this small stays serial anyway)
    dims = (6, 6, 6, 6)
    u = _links(12, dims, "f32", "near_unit")
    out = [np.empty_like(t) for t in u]
    with lqx.Lattice(dims) as lat:
        lat.set_option("host_slabs", slabs)
        n0 = lat.launch_count()
        p = lqx.smear_iterate_host(lat, lqx.F32, u, out, 0.4, 1)
        assert lat.launch_count() - n0 <= 17
    want_u, want_p = orc.smear_iterate(dims, u, 0.4, 1, "f32")
    assert abs(p[0] - want_p[0]) < RTOL["f32"]
    for mu in range(4):
        assert site_rel_err(out[mu], want_u[mu]) < TOL["f32"]


# ------------------------------------------------------------------------------------------------
# error behaviour of the boundary
# ------------------------------------------------------------------------------------------------
def test_error_codes(lqx):
    dims = (4, 4, 4, 4)
    with lqx.Lattice(dims) as lat, lqx.Lattice((4, 4, 4, 2)) as lat2:
        a32 = lat.alloc(lqx.COLORMAT, lqx.F32)
        b32 = lat.alloc(lqx.COLORMAT, lqx.F32)
        a64 = lat.alloc(lqx.COLORMAT, lqx.F64)
        v32 = lat.alloc(lqx.COLORVEC, lqx.F32)
        other = lat2.alloc(lqx.COLORMAT, lqx.F32)

        def code(fn, *args):
            with pytest.raises(lqx.LqxError) as e:
                fn(*args)
            return e.value.code

        assert code(lqx.shift, a32, a32, +1, 0) == -4            # EALIAS
        assert code(lqx.shift, a32, b32, +1, 4) == -1            # EINVAL mu
        assert code(lqx.shift, a32, b32, 0, 1) == -1             # EINVAL dir
        assert code(lqx.shift, a32, a64, +1, 0) == -2            # ETYPE precision
        assert code(lqx.shift, a32, v32, +1, 0) == -2            # ETYPE kind
        assert code(lqx.shift, a32, other, +1, 0) == -3          # EGEOM
        assert code(lqx.ax_minus_shift, a32, 2.5, b32, a32, -1, 2) == -4
        assert code(lqx.mat_vec, v32, v32, v32) == -2
        u = [a32, b32, lat.alloc(lqx.COLORMAT, lqx.F32), lat.alloc(lqx.COLORMAT, lqx.F32)]
        assert code(lqx.smear_step, u, u, 0.5) == -4
        assert code(lqx.hop, v32, u, v32) == -4
        with pytest.raises(lqx.LqxError):
            lqx.Lattice((4, 0, 4, 4))


# Reading A21: a site-local form may overwrite one of its operands.  Those launches run the plain-load,
# non-__restrict__ instantiation of the kernel (ld.global.nc is undefined for memory the kernel writes): every in-place
# form, twice, on a ragged lattice, bit for bit against its out-of-place result.
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_in_place_forms_equal_out_of_place_bit_for_bit(lqx, prec):
    dims = DIMS_RAGGED
    a, b, c, d = (_gauss(7, k, dims, "cm", prec) for k in range(4))
    v = _gauss(7, 4, dims, "cv", prec)
    psi = _gauss(7, 5, dims, "f", prec)
    with lqx.Lattice(dims) as lat:
        P = _prec(lqx, prec)
        fa, fb, fc, fd = (lat.from_host(t) for t in (a, b, c, d))

        def fresh(t):
            return lat.from_host(t)

        for rep in range(2):
            # form i with the destination in each operand slot
            want = lat.alloc(lqx.COLORMAT, P)
            lqx.mm_plus_madj(want, fa, fb, fc, fd)
            w = want.pop()
            for slot in range(4):
                ops = [fa, fb, fc, fd]
                ops[slot] = fresh((a, b, c, d)[slot])
                lqx.mm_plus_madj(ops[slot], *ops)
                assert np.array_equal(ops[slot].pop(), w), ("form i", slot, rep)
            # the same matrix in two slots and as the destination
            x = fresh(a)
            lqx.mm_plus_madj(want, fa, fa, fc, fa)
            lqx.mm_plus_madj(x, x, x, fc, x)
            assert np.array_equal(x.pop(), want.pop())
            # E3 / E4 / scale / copy
            for fn, args in ((lqx.axpy, (1, 0.37, 2)), (lqx.axpy, (2, 0.37, 1))):
                r = lat.alloc(lqx.COLORMAT, P)
                fn(r, fa, args[1], fb)
                x = fresh(a if args[0] == 1 else b)
                fn(x, x if args[0] == 1 else fa, args[1], fb if args[0] == 1 else x)
                assert np.array_equal(x.pop(), r.pop()), ("axpy", args, rep)
            r = lat.alloc(lqx.COLORMAT, P)
            x = fresh(a)
            lqx.scale(r, -1.75, fa), lqx.scale(x, -1.75, x)
            assert np.array_equal(x.pop(), r.pop())
            x = fresh(a)
            lqx.divide(r, fa, 1.3), lqx.divide(x, x, 1.3)
            assert np.array_equal(x.pop(), r.pop())
            x = fresh(a)
            lqx.copy(x, x)
            assert np.array_equal(x.pop(), a)
            # form iv: v = M v
            for vec, kind in ((v, lqx.COLORVEC), (psi, lqx.FERMION)):
                r = lat.alloc(kind, P)
                x = fresh(vec)
                lqx.mat_vec(r, fa, x), lqx.mat_vec(x, fa, x)
                assert np.array_equal(x.pop(), r.pop()), ("form iv", kind, rep)
            # form iii may overwrite its UNshifted operand
            r = lat.alloc(lqx.COLORMAT, P)
            x = fresh(a)
            lqx.ax_minus_shift(r, 2.5, fa, fb, lqx.BACKWARD, 2), lqx.ax_minus_shift(x, 2.5, x, fb, lqx.BACKWARD, 2)
            assert np.array_equal(x.pop(), r.pop())
            # run-time expressions: dst as a leaf (site-local), and dst += e
            X = lqx.Expr.leaf
            r = lat.alloc(lqx.COLORMAT, P)
            x = fresh(a)
            lqx.expr_eval(r, X(fa) * X(fb) + X(fc) * lqx.adj(X(fa)))
            lqx.expr_eval(x, X(x) * X(fb) + X(fc) * lqx.adj(X(x)))
            assert np.array_equal(x.pop(), r.pop())
            r, x = fresh(d), fresh(d)
            lqx.expr_eval(r, X(fa) * lqx.shifted(X(fb), lqx.FORWARD, 1), accumulate=True)
            y = fresh(a)
            lqx.expr_eval(x, X(y) * lqx.shifted(X(fb), lqx.FORWARD, 1), accumulate=True)
            assert np.array_equal(x.pop(), r.pop())


def test_partial_overlap_and_misalignment_are_errors(lqx):
    """two attached views that overlap without sharing a base pointer are aliases too (byte ranges, not pointers);
    the device-to-device converters want 16-byte aligned buffers"""
    import ctypes as C

    import torch

    dims = (4, 4, 4, 4)
    with lqx.Lattice(dims) as lat:
        nbytes = lat.field_bytes(lqx.COLORMAT, lqx.F32)
        mem = torch.zeros(2 * nbytes, dtype=torch.uint8, device="cuda")

        def view(off):
            h = C.c_void_p()
            rc = lqx._lib.lqx_field_attach(lat.ctx, lqx.COLORMAT, lqx.F32, C.c_void_p(mem.data_ptr() + off), nbytes, C.byref(h))
            assert rc == 0
            return lqx.Field(lat, h, lqx.COLORMAT, lqx.F32, mem)

        f0, f1, f2 = view(0), view(256), view(nbytes)
        other = lat.alloc(lqx.COLORMAT, lqx.F32)

        def code(fn, *args):
            with pytest.raises(lqx.LqxError) as e:
                fn(*args)
            return e.value.code

        assert code(lqx.shift, f0, f1, +1, 0) == -4
        assert code(lqx.copy, f0, f1) == -4
        assert code(lqx.mm_plus_madj, f1, f0, other, other, other) == -4
        assert code(lqx.ax_minus_shift, f1, 2.5, f0, other, -1, 2) == -4
        u = [f1, other, lat.alloc(lqx.COLORMAT, lqx.F32), lat.alloc(lqx.COLORMAT, lqx.F32)]
        o = [f0] + [lat.alloc(lqx.COLORMAT, lqx.F32) for _ in range(3)]
        assert code(lqx.smear_step, o, u, 0.5) == -4
        lqx.copy(f0, f2)  # adjacent, not overlapping: fine
        lqx.shift(f0, f2, +1, 0)
        buf = torch.zeros(lat.volume * 18 + 4, dtype=torch.float32, device="cuda")
        with pytest.raises(lqx.LqxError) as e:
            other.import_dev(buf[1:])
        assert e.value.code == -1
        with pytest.raises(lqx.LqxError) as e:
            other.export_dev(buf[1:])
        assert e.value.code == -1
        other.import_dev(buf[4:])


# ------------------------------------------------------------------------------------------------
# NEXT-1: the paper's complete Jacobi smearing routine (Listing 1)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [DIMS_RAGGED, DIMS_EVEN, (2, 2, 2, 2)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("kind", ["f", "cv"])
def test_jacobi_smear(lqx, dims, prec, kind):
    tv = orc.truth_variant(prec)
    u = _links(2, dims, prec)
    chi0 = _gauss(2, 10, dims, kind, prec)
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        for (kappa, iters, skip, norm) in [(0.21, 5, -1, 1.7), (0.21, 4, 3, 1.7), (0.3, 1, 0, 0.5), (0.3, 0, -1, 2.0), (0.1, 2, 9, 1.0)]:
            chi = lat.from_host(chi0)
            tmp = [lat.alloc(chi.kind, chi.prec) for _ in range(2)]
            lqx.jacobi_smear(chi, fu, kappa, iters, skip, norm, tmp)
            want = orc.jacobi_smear(dims, u, chi0, kappa, iters, skip, norm, tv)
            assert site_rel_err(chi.pop(), want) < TOL[prec] * max(1, iters), (kappa, iters, skip)
        # error behaviour: scratch must not alias, iter >= 0, norm != 0
        chi = lat.from_host(chi0)
        t0 = lat.alloc(chi.kind, chi.prec)
        for bad in (lambda: lqx.jacobi_smear(chi, fu, 0.1, 2, -1, 1.0, [t0, t0]),
                    lambda: lqx.jacobi_smear(chi, fu, 0.1, 2, -1, 1.0, [chi, t0]),
                    lambda: lqx.jacobi_smear(chi, fu, 0.1, -1, -1, 1.0, [t0, lat.alloc(chi.kind, chi.prec)]),
                    lambda: lqx.jacobi_smear(chi, fu, 0.1, 2, -1, 0.0, [t0, lat.alloc(chi.kind, chi.prec)])):
            with pytest.raises(lqx.LqxError):
                bad()


# NEXT-3: every launch geometry the options (and the auto-tuner) can select -- N_threads x N_site of PAPER.md:117-126 --
# runs its own code path (grid-stride loop for N_site > 1, the last CTA ragged): each against the oracle, and all of
# them bit-identical to one another (the per-site arithmetic does not depend on the geometry)
@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("kind", ["f", "cv"])
def test_jacobi_smear_every_launch_geometry(lqx, prec, kind):
    dims = DIMS_RAGGED
    tv = orc.truth_variant(prec)
    u = _links(2, dims, prec)
    chi0 = _gauss(2, 10, dims, kind, prec)
    want = orc.jacobi_smear(dims, u, chi0, 0.21, 3, 3, 1.7, tv)
    first = None
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        for block in (32, 64, 128, 256):
            for nsite in (1, 2, 4):
                lat.set_option("jacobi_block", block)
                lat.set_option("jacobi_sites", nsite)
                chi = lat.from_host(chi0)
                tmp = [lat.alloc(chi.kind, chi.prec) for _ in range(2)]
                lqx.jacobi_smear(chi, fu, 0.21, 3, 3, 1.7, tmp)
                got = chi.pop()
                assert site_rel_err(got, want) < TOL[prec] * 3, (block, nsite)
                if first is None:
                    first = got
                assert np.array_equal(got, first), (block, nsite)
                for f in [chi] + tmp:
                    f.free()


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("dims", [(16, 8, 4, 4), DIMS_RAGGED])
def test_autotune_keeps_a_geometry_that_agrees_with_the_oracle(lqx, dims, prec):
    """lqx_autotune: the table lists every candidate with a time, exactly one is kept per kernel, an
    explicit option still overrides it, and the calls that follow -- now running the kept geometry -- agree with the oracle."""
    tv = orc.truth_variant(prec)
    P = _prec(lqx, prec)
    u = _links(5, dims, prec)
    psi = _gauss(5, 9, dims, "f", prec)
    with lqx.Lattice(dims) as lat:
        for cls, nkept in ((lqx.K_SMEAR, 1), (lqx.K_PLAQUETTE, 1), (lqx.K_HOP, 2)):
            rows = lat.autotune(cls, P, reps=2)
            assert rows and all(r["ms"] > 0 and r["kernel_class"] == cls and r["prec"] == P for r in rows)
            assert sum(r["chosen"] for r in rows) == nkept
        t = lat.tuned(lqx.K_SMEAR, P)
        assert t[0] in (3, 9, 10)
        hb, jb, js = lat.tuned(lqx.K_HOP, P)[:3]
        assert hb in (32, 64, 128, 256) and jb in (32, 64, 128, 256) and js in (1, 2, 4)
        assert lat.tuned(lqx.K_PLAQUETTE, P)[0] in (1, 2)
        fu = [lat.from_host(x) for x in u]
        out = [lat.alloc(lqx.COLORMAT, P) for _ in range(4)]
        p = lqx.smear_step(out, fu, 0.5, want_plaq_in=True)
        assert lat.smear_info()[0] == t[0]
        want = orc.smear_step(dims, u, 0.5, tv)
        for mu in range(4):
            assert site_rel_err(out[mu].pop(), want[mu]) < TOL[prec]
        psum = orc.plaquette_sum(dims, u, tv)
        scale = np.sqrt(18.0 * lat.volume)
        assert abs(p - psum) / max(abs(psum), scale) < RTOL[prec]
        assert abs(lqx.plaquette(fu)[0] - psum) / max(abs(psum), scale) < RTOL[prec]
        fpsi, chi = lat.from_host(psi), lat.alloc(lqx.FERMION, P)
        lqx.hop(chi, fu, fpsi)
        assert site_rel_err(chi.pop(), orc.hop(dims, u, psi, tv)) < TOL[prec]
        tmp = [lat.alloc(lqx.FERMION, P) for _ in range(2)]
        lqx.jacobi_smear(fpsi, fu, 0.21, 3, 3, 1.7, tmp)
        assert site_rel_err(fpsi.pop(), orc.jacobi_smear(dims, u, psi, 0.21, 3, 3, 1.7, tv)) < TOL[prec] * 3
        # an explicit option wins over the tuned choice
        lat.set_option("smear_variant", 1)
        lqx.smear_step(out, fu, 0.5)
        assert lat.smear_info()[0] == 1 and lat.smear_info()[2] == "k_smear_gather"


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_hop_every_block_size(lqx, prec):
    dims = DIMS_RAGGED
    u = _links(2, dims, prec)
    psi = _gauss(2, 10, dims, "f", prec)
    want = orc.hop(dims, u, psi, orc.truth_variant(prec))
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        fpsi, chi = lat.from_host(psi), lat.alloc(lqx.FERMION, _prec(lqx, prec))
        first = None
        for hb in (0, 32, 64, 128, 256):
            lat.set_option("hop_block", hb)
            lqx.scale(chi, 0.0, chi)
            lqx.hop(chi, fu, fpsi)
            got = chi.pop()
            assert site_rel_err(got, want) < TOL[prec], hb
            first = got if first is None else first
            assert np.array_equal(got, first), hb


def test_jacobi_smear_config2_size(lqx):
    """16^3x32 fp32 (the lattice of configs[1], a Table-1 size of the paper), 10 iterations, fermion."""
    cfg = li.CONFIGS["c2"]
    dims = cfg["dims"]
    u = _links(cfg["seed"], dims, "f32")
    chi0 = _gauss(cfg["seed"], 10, dims, "f", "f32")
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        chi = lat.from_host(chi0)
        tmp = [lat.alloc(chi.kind, chi.prec) for _ in range(2)]
        lqx.jacobi_smear(chi, fu, 0.05, 10, 3, 1.5, tmp)
        want = orc.jacobi_smear(dims, u, chi0, 0.05, 10, 3, 1.5, "t32")
        assert site_rel_err(chi.pop(), want) < TOL["f32"] * 10


# ------------------------------------------------------------------------------------------------
# BASELINE.json's full sizes, in the launch configuration bench.py times (default variant / tile):
# sampled outputs the oracle computes one by one, plus properties that hold at any size
# ------------------------------------------------------------------------------------------------
def _full_size_links(lqx, lat, cfgname, recipe, prec):
    """Same generator calls as bench.py: fields made on the GPU, imported, and copied to the host for the oracle."""
    import torch

    cfg = li.CONFIGS[cfgname]
    fields, host = [], []
    for mu in range(4):
        if recipe == "haar":
            z = li.haar_su3_complex(cfg["seed"], mu, lat.volume, "cuda")
        else:
            z = li.near_unit_su3_complex(cfg["seed"], mu, lat.volume, 0.1, "cuda")
        a = li._as_real(z, prec)
        del z
        fields.append(lat.alloc(lqx.COLORMAT, _prec(lqx, prec)).import_dev(a))
        torch.cuda.synchronize()
        host.append(a.cpu().numpy())
        del a
    torch.cuda.empty_cache()
    return fields, host


def _sample_sites(dims, n, seed):
    """Random sites plus the corners and faces where every kind of wrap-around happens."""
    rng = np.random.default_rng(seed)
    v = int(np.prod(dims))
    s = list(rng.integers(0, v, size=n))
    ext = [(0, d - 1, d // 2) for d in dims]
    for x0 in ext[0]:
        for x1 in ext[1]:
            for x2 in ext[2]:
                for x3 in ext[3]:
                    s.append(x0 + dims[0] * (x1 + dims[1] * (x2 + dims[2] * x3)))
    return np.unique(np.array(s, dtype=np.int64))


@pytest.mark.parametrize("cfgname,recipe", [("c4", "near_unit"), ("c3", "haar")])
def test_full_size_smear_step_sampled(lqx, cfgname, recipe):
    import torch

    cfg = li.CONFIGS[cfgname]
    dims, prec = cfg["dims"], cfg["prec"]
    tv = orc.truth_variant(prec)
    with lqx.Lattice(dims) as lat:
        fu, hu = _full_size_links(lqx, lat, cfgname, recipe, prec)
        out = [lat.alloc(lqx.COLORMAT, fu[0].prec) for _ in range(4)]
        p_fused = lqx.smear_step(out, fu, 0.5, want_plaq_in=True)
        sites = _sample_sites(dims, 3000, 17)
        dt = torch.float32 if prec == "f32" else torch.float64
        buf = torch.empty((lat.volume, 3, 3, 2), dtype=dt, device="cuda")
        idx = torch.from_numpy(sites).cuda()
        for mu in range(4):
            out[mu].export_dev(buf)
            got = buf[idx].cpu().numpy()
            want = orc.smear_links(dims, hu, 0.5, sites, np.full(sites.size, mu, dtype=np.int32), tv)
            assert site_rel_err(got, want) < TOL[prec], mu
        # plaquette: the fused sum equals the standalone kernel's (two code paths), and the per-site mean over
        # the sample agrees with the oracle's integrand within its statistical error
        p_alone, _ = lqx.plaquette(fu)
        scale = np.sqrt(18.0 * lat.volume)
        assert abs(p_fused - p_alone) / max(abs(p_alone), scale) < RTOL[prec]
        dens = orc.plaquette_sites(dims, hu, sites, tv)
        assert abs(p_alone / lat.volume - dens.mean()) < 6 * dens.std() / np.sqrt(sites.size) + 1e-6
        # ... and, not statistically: the GLOBAL plaquette sum of the whole lattice against the oracle's, for the
        # input field (fused and standalone) and for the output field (readings A11, A15)
        p_want = orc.plaquette_sum(dims, hu, tv)
        assert abs(p_alone - p_want) / max(abs(p_want), scale) < RTOL[prec]
        assert abs(p_fused - p_want) / max(abs(p_want), scale) < RTOL[prec]
        want_out = orc.smear_step(dims, hu, 0.5, tv)
        p_out_want = orc.plaquette_sum(dims, want_out, "t64" if prec == "f64" else "n64")
        del want_out
        p_out, _ = lqx.plaquette(out)
        assert abs(p_out - p_out_want) / max(abs(p_out_want), scale) < RTOL[prec]
        # property at any size: sum_{x,mu} Re tr[U S^dag] = 4 P, with S recovered from U' = (1-a) U + (a/6) S
        acc = 0.0
        for mu in range(4):
            out[mu].export_dev(buf)
            uin = torch.from_numpy(hu[mu]).cuda().to(torch.float64)
            stp = (buf.to(torch.float64) - 0.5 * uin) * 12.0
            acc += float((uin * stp).sum())
            del uin, stp
        # S is recovered as 12 (U' - U/2) from the ROUNDED output, which multiplies U's rounding error by 12: the
        # identity is checked at 4 x the reduction tolerance (reading A24)
        assert abs(acc - 4.0 * p_alone) / max(abs(4.0 * p_alone), scale) < RTOL[prec] * 4


def test_full_size_c4_ten_steps_properties(lqx):
    """configs[3]: ten iterated steps with the plaquette after each; the first step's plaquette equals the
    plaquette of a single smear_step output, and the trajectory is reproducible bit for bit."""
    cfg = li.CONFIGS["c4"]
    dims = cfg["dims"]
    with lqx.Lattice(dims) as lat:
        fu, _ = _full_size_links(lqx, lat, "c4", "near_unit", "f32")
        tmp = [lat.alloc(lqx.COLORMAT, lqx.F32) for _ in range(4)]
        keep = [lat.alloc(lqx.COLORMAT, lqx.F32) for _ in range(4)]
        for a, b in zip(keep, fu):
            lqx.copy(a, b)
        lqx.smear_step(tmp, fu, 0.5)
        _, p1 = lqx.plaquette(tmp)
        plaqs = lqx.smear_iterate(fu, tmp, 0.5, 10)
        assert len(plaqs) == 10 and all(np.isfinite(plaqs))
        assert abs(plaqs[0] - p1) < RTOL["f32"]
        assert all(0.0 < p < 1.0 for p in plaqs)
        n_a = lqx.norm2(fu[2])
        plaqs2 = lqx.smear_iterate(keep, tmp, 0.5, 10)
        assert plaqs2 == plaqs and lqx.norm2(keep[2]) == n_a
        # ten one-step calls walk the same links bit for bit; their plaquettes come from the standalone kernel
        # instead of the next step's fused pass (another summation order)
        for a, b in zip(keep, fu):
            lqx.copy(a, b)
        more = lqx.smear_iterate(fu, tmp, 0.5, 2)
        one = lqx.smear_iterate(keep, tmp, 0.5, 1) + lqx.smear_iterate(keep, tmp, 0.5, 1)
        assert lqx.norm2(keep[1]) == lqx.norm2(fu[1])
        assert all(abs(a - b) <= 1e-5 * abs(b) for a, b in zip(one, more))


def test_full_size_c4_trajectory_against_oracle(lqx):
    """configs[3] at full size, all TEN iterated steps (reading A23).  Primary check: the plaquette average after
    every step and the links after the last one (sampled sites) against the oracle's truth trajectory of the whole
    48^3x96 lattice (a few seconds per step on the host cores), link tolerance TOL * nsteps.  Secondary check, at the
    FLAT tolerance: every single step against the oracle restarted from the GPU's own previous output."""
    import torch

    cfg = li.CONFIGS["c4"]
    dims = cfg["dims"]
    nsteps = 10
    with lqx.Lattice(dims) as lat:
        fu, hu = _full_size_links(lqx, lat, "c4", "near_unit", "f32")
        tmp = [lat.alloc(lqx.COLORMAT, lqx.F32) for _ in range(4)]
        want_u, want_p = orc.smear_iterate(dims, hu, 0.5, nsteps, "f32")
        sites = _sample_sites(dims, 3000, 23)
        idx = torch.from_numpy(sites).cuda()
        buf = torch.empty((lat.volume, 3, 3, 2), dtype=torch.float32, device="cuda")
        plaqs = []
        prev = hu
        for k in range(nsteps):
            plaqs += lqx.smear_iterate(fu, tmp, 0.5, 1)
            now = []
            for mu in range(4):
                fu[mu].export_dev(buf)
                want = orc.smear_links(dims, prev, 0.5, sites, np.full(sites.size, mu, dtype=np.int32), "t32")
                assert site_rel_err(buf[idx].cpu().numpy(), want) < TOL["f32"], (k, mu)
                if k + 1 < nsteps:
                    now.append(buf.cpu().numpy())
            prev = now
        for k in range(nsteps):
            # absolute on the average as everywhere, and relative: the links shrink (no projection, A9) and the
            # plaquette falls from 0.49 to 2e-9 over the ten steps
            assert abs(plaqs[k] - want_p[k]) < RTOL["f32"], k
            assert abs(plaqs[k] - want_p[k]) < RTOL["f32"] * abs(want_p[k]) * (k + 1), k
        for mu in range(4):
            fu[mu].export_dev(buf)
            assert site_rel_err(buf[idx].cpu().numpy(), want_u[mu][sites]) < TOL["f32"] * nsteps, mu


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_full_size_c5_expression_sweep(lqx, prec):
    """configs[4]: 32^3x64, the four forms each followed by its reduction, against the truth oracle."""
    dims = li.CONFIGS["c5"]["dims"]
    tv = orc.truth_variant(prec)
    a, b, c, d = (_gauss(7, k, dims, "cm", prec) for k in range(4))
    v = _gauss(7, 4, dims, "cv", prec)
    with lqx.Lattice(dims) as lat:
        fa, fb, fc, fd, fv = (lat.from_host(t) for t in (a, b, c, d, v))
        r = lat.alloc(lqx.COLORMAT, fa.prec)
        cx = lat.alloc(lqx.COMPLEX, fa.prec)
        w = lat.alloc(lqx.COLORVEC, fa.prec)
        lqx.mm_plus_madj(r, fa, fb, fc, fd)
        want = orc.mm_plus_madj(dims, a, b, c, d, tv)
        assert site_rel_err(r.pop(), want) < TOL[prec]
        n2 = lqx.norm2(r)
        wn2 = orc.norm2(dims, want.astype(np.float64), "t64")
        assert abs(n2 - wn2) / wn2 < RTOL[prec]
        lqx.trace_mm(cx, fa, fb)
        want = orc.trace_mm(dims, a, b, tv)
        # form ii reduces nine products to ONE complex number per site: among 2 million sites some cancel
        # almost completely, so the error is measured against the size of what was summed,
        # sum_ik |A_ik| |B_ki| (reading A14 with the summands as the site object)
        mag = np.einsum("xik,xki->x", np.abs(cplx(a)), np.abs(cplx(b)))
        assert float((np.abs(cx.pop().astype(np.float64) - want).max(axis=1) / mag).max()) < TOL[prec]
        rms = float(np.sqrt((want.astype(np.float64) ** 2).sum()))
        assert _red_err(lqx.sum(cx), orc.sum_field(dims, want.astype(np.float64), "t64"), rms) < RTOL[prec]
        lqx.ax_minus_shift(r, 2.5, fa, fb, lqx.BACKWARD, 2)
        assert np.array_equal(r.pop(), orc.ax_minus_shift(dims, 2.5, a, b, -1, 2, orc.native_variant(prec)))
        want = orc.ax_minus_shift(dims, 2.5, a, b, -1, 2, tv).astype(np.float64)
        rms = float(np.sqrt((want ** 2).sum()))
        assert _red_err(lqx.trace(r), orc.trace(dims, want, "t64"), rms) < RTOL[prec]
        lqx.mat_vec(w, fa, fv)
        want = orc.mat_vec(dims, a, v, tv)
        assert site_rel_err(w.pop(), want) < TOL[prec]
        wn2 = float((want.astype(np.float64) ** 2).sum())
        assert abs(lqx.norm2(w) - wn2) / wn2 < RTOL[prec]


# ------------------------------------------------------------------------------------------------
# NEXT-2: run-time expression fusion (NVRTC) against the oracle's generic evaluator
# ------------------------------------------------------------------------------------------------
def _hop_expr(lqx, fu, fpsi):
    e = None
    for mu in range(4):
        t = lqx.Expr.leaf(fu[mu]) * lqx.shifted(fpsi, lqx.FORWARD, mu) + lqx.shifted(lqx.adj(fu[mu]) * lqx.Expr.leaf(fpsi), lqx.BACKWARD, mu)
        e = t if e is None else e + t
    return e


def _staple_expr(lqx, fu, mu):
    e = None
    for nu in range(4):
        if nu == mu:
            continue
        up = lqx.Expr.leaf(fu[nu]) * lqx.shifted(fu[mu], lqx.FORWARD, nu) * lqx.adj(lqx.shifted(fu[nu], lqx.FORWARD, mu))
        lo = lqx.shifted(lqx.adj(fu[nu]) * lqx.Expr.leaf(fu[mu]) * lqx.shifted(fu[nu], lqx.FORWARD, mu), lqx.BACKWARD, nu)
        e = up + lo if e is None else e + (up + lo)
    return e


@pytest.mark.parametrize("dims", [DIMS_RAGGED, (2, 2, 2, 2)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_expr_eval_against_oracle(lqx, dims, prec):
    u = _links(2, dims, prec)
    a, b, c, d = (_gauss(7, k, dims, "cm", prec) for k in range(4))
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        fa, fb, fc, fd = (lat.from_host(t) for t in (a, b, c, d))
        r = lat.alloc(lqx.COLORMAT, fa.prec)
        host = {id(f): h for f, h in zip(fu + [fa, fb, fc, fd], u + [a, b, c, d])}

        def want_of(e):  # the oracle on the expression's own postfix sequence and leaf order
            return orc.eval_expr(dims, e.nodes, [host[id(f)] for f in e.leaves])

        # form i and form iii as run-time expressions
        e = lqx.Expr.leaf(fa) * lqx.Expr.leaf(fb) + lqx.Expr.leaf(fc) * lqx.adj(fd)
        lqx.expr_eval(r, e)
        assert site_rel_err(r.pop(), want_of(e)) < TOL[prec]
        n0 = lat.expr_cache_size()
        e3 = 2.5 * lqx.Expr.leaf(fa) - lqx.shifted(fb, lqx.BACKWARD, 2)
        lqx.expr_eval(r, e3)
        got = r.pop()
        assert site_rel_err(got, want_of(e3)) < TOL[prec]
        lqx.ax_minus_shift(r, 2.5, fa, fb, lqx.BACKWARD, 2)
        assert site_rel_err(got, r.pop()) < TOL[prec]  # the hand-written kernel of the same expression
        assert lat.expr_cache_size() == n0 + 1
        lqx.expr_eval(r, 7.0 * lqx.Expr.leaf(fa) - lqx.shifted(fb, lqx.BACKWARD, 2))  # other scalar: same kernel
        assert lat.expr_cache_size() == n0 + 1
        assert site_rel_err(r.pop(), orc.eval_expr(dims, [(0, 0, 0, 0), (5, 0, 0, 7.0), (0, 1, 0, 0), (6, -1, 2, 0), (4, 0, 0, 0)], [a, b])) < TOL[prec]
        # the paper's E1/E2 expression, exactly as Listing 1 writes it, summed over mu; '=' then '+='
        for kind in ("f", "cv"):
            psi = _gauss(2, 10, dims, kind, prec)
            fpsi = lat.from_host(psi)
            host[id(fpsi)] = psi
            chi = lat.alloc(fpsi.kind, fpsi.prec)
            eh = _hop_expr(lqx, fu, fpsi)
            lqx.expr_eval(chi, eh)
            want = want_of(eh)
            assert site_rel_err(want, orc.hop(dims, u, psi, orc.truth_variant(prec))) < 1e-12
            assert site_rel_err(chi.pop(), want) < TOL[prec]
            lqx.expr_eval(chi, eh, accumulate=True)
            assert site_rel_err(chi.pop(), 2.0 * want) < TOL[prec]
            ref = lat.alloc(fpsi.kind, fpsi.prec)
            lqx.hop(ref, fu, fpsi)
            assert site_rel_err(ref.pop(), want) < TOL[prec]
        # nested shifts: the staple sum of one direction as ONE expression
        es = _staple_expr(lqx, fu, 1)
        lqx.expr_eval(r, es)
        assert site_rel_err(r.pop(), orc.staple_sum(dims, u, 1, orc.truth_variant(prec))) < TOL[prec]
        # in place where it is legal, refused where the destination is read through a shift
        lqx.expr_eval(fa, lqx.Expr.leaf(fa) * lqx.Expr.leaf(fb))
        assert site_rel_err(fa.pop(), orc.eval_expr(dims, [(0, 0, 0, 0), (0, 1, 0, 0), (2, 0, 0, 0)], [a, b])) < TOL[prec]
        with pytest.raises(lqx.LqxError):
            lqx.expr_eval(fb, lqx.Expr.leaf(fc) - lqx.shifted(fb, lqx.FORWARD, 0))
        with pytest.raises(lqx.LqxError):  # kind mismatch with the destination
            lqx.expr_eval(r, _hop_expr(lqx, fu, lat.from_host(_gauss(2, 10, dims, "cv", prec))))


@pytest.mark.parametrize("dims", [DIMS_RAGGED, (16, 8, 8, 8)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_expr_trace_and_reductions(lqx, dims, prec):
    """configs[4] through the run-time path: each form followed by its norm2 / sum / trace reduction, the
    reduction fused into the generated kernel (nothing is materialised)."""
    a, b, c, d = (_gauss(7, k, dims, "cm", prec) for k in range(4))
    v = _gauss(7, 4, dims, "cv", prec)
    with lqx.Lattice(dims) as lat:
        fa, fb, fc, fd, fv = (lat.from_host(t) for t in (a, b, c, d, v))
        host = {id(f): h for f, h in zip((fa, fb, fc, fd, fv), (a, b, c, d, v))}

        def want_of(e):
            return orc.eval_expr(dims, e.nodes, [host[id(f)] for f in e.leaves])

        L = lqx.Expr.leaf
        # form ii: trace(A*B) into a LatticeComplex, against the hand-written kernel and the oracle
        e2 = (L(fa) * L(fb)).trace()
        cx = lat.alloc(lqx.COMPLEX, fa.prec)
        lqx.expr_eval(cx, e2)
        got = cx.pop()
        mag = np.einsum("xik,xki->x", np.abs(cplx(a)), np.abs(cplx(b)))
        assert float((np.abs(got.astype(np.float64) - want_of(e2)).max(axis=1) / mag).max()) < TOL[prec]
        cx2 = lat.alloc(lqx.COMPLEX, fa.prec)
        lqx.trace_mm(cx2, fa, fb)
        assert float((np.abs(got.astype(np.float64) - cx2.pop()).max(axis=1) / mag).max()) < TOL[prec]
        for e in (L(fa) * L(fb) + L(fc) * lqx.adj(fd), 2.5 * L(fa) - lqx.shifted(fb, lqx.BACKWARD, 2), L(fa) * L(fv), e2):
            w = want_of(e)
            n2w = float((w ** 2).sum())
            assert abs(lqx.expr_reduce(lqx.R_NORM2, e) - n2w) / n2w < RTOL[prec]
            sw = w.sum(axis=0).ravel()
            rms = float(np.sqrt(n2w))
            assert _red_err(lqx.expr_reduce(lqx.R_SUM, e), sw, rms) < RTOL[prec]
        # global trace of a matrix expression = sum of its site-wise trace (reading A12)
        e1 = L(fa) * L(fb) + L(fc) * lqx.adj(fd)
        r = lat.alloc(lqx.COLORMAT, fa.prec)
        lqx.expr_eval(r, e1)
        tr_two_calls = np.asarray(lqx.trace(r))
        tr_fused = lqx.expr_reduce(lqx.R_SUM, e1.trace())
        rms = float(np.sqrt((want_of(e1) ** 2).sum()))
        assert _red_err(tr_fused, tr_two_calls, rms) < RTOL[prec]
        with pytest.raises(lqx.LqxError):
            lqx.expr_eval(cx, L(fv).trace())
        with pytest.raises(lqx.LqxError):
            lqx.expr_reduce(9, e1)


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("dims", [DIMS_RAGGED, (8, 8, 8, 8)])
def test_plaquette_as_a_runtime_expression(lqx, dims, prec):
    """sum_x trace( sum_{mu<nu} (U_mu * shift(U_nu,F,mu)) * adj(U_nu * shift(U_mu,F,nu)) ) written by the user and
    reduced inside one generated kernel: against the oracle's plaquette sum and the hand-written kernel."""
    u = _links(21, dims, prec, "near_unit")
    want = orc.plaquette_sum(dims, u, "t64" if prec == "f64" else "t32")
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        L = lqx.Expr.leaf
        e = None
        for mu in range(3):
            for nu in range(mu + 1, 4):
                t = (L(fu[mu]) * lqx.shifted(fu[nu], lqx.FORWARD, mu)) * lqx.adj(L(fu[nu]) * lqx.shifted(fu[mu], lqx.FORWARD, nu))
                e = t if e is None else e + t
        got = lqx.expr_reduce(lqx.R_SUM, e.trace())
        hand = lqx.plaquette(fu)[0]
        n = lat.expr_cache_size()
        lqx.expr_reduce(lqx.R_SUM, e.trace())
        assert lat.expr_cache_size() == n  # compiled once
    scale = 18.0 * np.prod(dims)
    assert abs(got[0] - want) / scale < RTOL[prec]
    assert abs(got[0] - hand) / scale < RTOL[prec]
    # the imaginary part (not zero: only its gauge average vanishes) against the oracle's evaluator
    w = orc.eval_expr(dims, e.trace().nodes, u)
    im = np.asarray(w).reshape(int(np.prod(dims)), -1)
    im_sum = float(im[:, 0].imag.sum()) if np.iscomplexobj(im) else float(im[:, 1].sum())
    assert abs(got[1] - im_sum) / scale < RTOL[prec]


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("fused", [True, False])
def test_jacobi_listing_through_runtime_expressions(lqx, prec, fused):
    """The paper's Listing 1 written as user code on the run-time expression path (bench.jacobi_listing), literally
    (E0..E4) and fused, against the oracle's routine and the hand-written lqx_jacobi_smear."""
    import bench

    dims = DIMS_RAGGED
    u = _links(2, dims, prec)
    chi0 = _gauss(2, 10, dims, "f", prec)
    kappa, iters, skip, norm = 0.21, 4, 3, 1.7
    with lqx.Lattice(dims) as lat:
        fu = [lat.from_host(t) for t in u]
        chi = lat.from_host(chi0)
        work = [lat.alloc(chi.kind, chi.prec) for _ in range(3)]
        bench.jacobi_listing(lqx, chi, fu, kappa, iters, skip, norm, work, fused)
        want = orc.jacobi_smear(dims, u, chi0, kappa, iters, skip, norm, orc.truth_variant(prec))
        got = chi.pop()
        assert site_rel_err(got, want) < TOL[prec] * iters
        ref = lat.from_host(chi0)
        lqx.jacobi_smear(ref, fu, kappa, iters, skip, norm, work[:2])
        assert site_rel_err(got, ref.pop()) < TOL[prec] * iters


# ------------------------------------------------------------------------------------------------
# bench.py: the JSON line the driver reads (a smaller workload than the default, same code path)
# ------------------------------------------------------------------------------------------------
def test_bench_line_contract():
    import json
    import os
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--workload", "c3", "--steps", "2", "--warmup", "3",
                          "--e2e-steps", "2", "--no-extras"], capture_output=True, text=True, cwd=root, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, "exactly one JSON line on stdout"
    line = json.loads(lines[0])
    assert line["metric"] == "smear-step site-updates/s" and line["unit"] == "site-updates/s"
    assert line["n_gpus"] == 1 and line["steps"] == 2 and line["warmup"] >= 3
    assert line["higher_is_better"] is True and line["scaling"] == "weak" and line["data"] == "synthetic"
    assert line["dtype"] == "f64" and line["vs_baseline"] is None
    assert "workload" in line["config"] and "model" not in line["config"]
    sites = line["config"]["sites"]
    assert abs(line["value"] - sites * 2 / (line["ms_per_step"] * 2 * 1e-3)) < 1e-6 * line["value"]
    assert line["gpu_launches"] >= 2 * 1  # at least one smear kernel per step
    r = line["roofline"]
    assert r["bound"] in ("hbm", "tensor", "alu") and r["unit"] in ("GB/s", "TFLOP/s")
    assert 0.0 < r["frac"] < 1.0 and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-9
    assert "traffic" in r and 0.0 < r["hbm"]["frac"] < 1.0
    e = line["e2e"]
    assert e["unit"] == line["unit"] and 0.0 < e["value"] < line["value"]
    assert e["h2d_bytes_per_step"] == sites * 4 * 18 * 8 and e["d2h_bytes_per_step"] >= e["h2d_bytes_per_step"]
    c = line["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and 0.0 < c["value"] < line["value"] and c["sample"]
    k = line["clocks"]
    assert k["sm_max_mhz"] > 0 and isinstance(k["reasons"], list)
    assert len(line["plaquette_avg_after_each_step"]) == 2 and all(abs(p) <= 1.0 for p in line["plaquette_avg_after_each_step"])


# ------------------------------------------------------------------------------------------------
# NEXT-4: decomposition along t (paper_1105_2279_b200/tsplit.py) on ONE GPU.  R ranks are emulated one after the other
# in this process (the profiling guide: never run ranks that wait on one another on one GPU): each has its own context
# on a local lattice of t-extent L3/R + 2, the halo exchange is a device copy between the ranks' fields.  The own slabs
# concatenated must equal lqx_smear_step on the whole lattice BIT FOR BIT, and the global plaquette must agree.
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("gdims,world", [((8, 4, 4, 8), 1), ((8, 4, 4, 8), 2), ((4, 4, 2, 12), 3), ((16, 4, 2, 8), 2)])
def test_tsplit_slabs_equal_the_single_gpu_step_bit_for_bit(lqx, gdims, world, prec):
    import torch

    from paper_1105_2279_b200 import tsplit
    from tsplit_helpers import EmulatedRanks, gather_own, scatter_no_halo

    P = _prec(lqx, prec)
    u = _links(6, gdims, prec, "near_unit")
    nsteps = 2
    with lqx.Lattice(gdims) as lat:  # the single-GPU answer
        fu = [lat.from_host(t) for t in u]
        tmp = [lat.alloc(lqx.COLORMAT, P) for _ in range(4)]
        want_plaqs = []
        for _ in range(nsteps):
            lqx.smear_step(tmp, fu, 0.5)
            fu, tmp = tmp, fu
            want_plaqs.append(lqx.plaquette(fu)[0])
        want = [f.pop() for f in fu]
    emu = EmulatedRanks(world)
    lats = [lqx.Lattice(tsplit.local_dims(gdims, world)) for _ in range(world)]
    try:
        comms = [tsplit.SelfComm() if world == 1 else emu.comm(r) for r in range(world)]
        ts = [tsplit.TSplit(tsplit.LqxBackend(lqx, lats[r]), comms[r], gdims) for r in range(world)]
        cur = [[lats[r].from_host(scatter_no_halo(f, gdims, r, world)) for f in u] for r in range(world)]  # NaN halos
        nxt = [[lats[r].alloc(lqx.COLORMAT, P) for _ in range(4)] for r in range(world)]
        for step in range(nsteps):
            if world == 1:
                ts[0].smear_step(nxt[0], cur[0], 0.5, overlap=(step == 0))
            else:
                for r in range(world):
                    comms[r].exchange(*ts[r]._halo_views(cur[r]))
                torch.cuda.synchronize()
                emu.flush()
                for r in range(world):
                    ts[r].smear_step(nxt[r], cur[r], 0.5, halos_fresh=True)
            cur, nxt = nxt, cur
            if world == 1:
                p = ts[0].plaquette_sum(cur[0])
            else:
                for r in range(world):
                    comms[r].exchange(*ts[r]._halo_views(cur[r]))
                torch.cuda.synchronize()
                emu.flush()
                p = sum(ts[r].plaquette_sum(cur[r], halos_fresh=True) for r in range(world))
            assert abs(p - want_plaqs[step]) <= RTOL[prec] * 1e-2 * max(abs(want_plaqs[step]), np.sqrt(18.0 * np.prod(gdims)))
        for mu in range(4):
            got = gather_own([cur[r][mu].pop() for r in range(world)], gdims)
            assert np.array_equal(got, want[mu]), mu
    finally:
        for l in lats:
            l.close()


def test_tsplit_geometry_errors(lqx):
    from paper_1105_2279_b200 import tsplit

    with pytest.raises(ValueError):
        tsplit.local_dims((4, 4, 4, 6), 4)
    with pytest.raises(ValueError):
        tsplit.local_dims((4, 4, 4, 4), 4)
    with lqx.Lattice((3, 3, 3, 4)) as lat:  # V3 = 27: a time slice is not a contiguous range
        f = lat.alloc(lqx.COLORMAT, lqx.F32)
        with pytest.raises(lqx.LqxError):
            f.slice_bytes(1)
        u = [lat.alloc(lqx.COLORMAT, lqx.F32) for _ in range(4)]
        o = [lat.alloc(lqx.COLORMAT, lqx.F32) for _ in range(4)]
        with pytest.raises(lqx.LqxError):
            lqx.smear_step_range(o, u, 0.5, 2, 2)
        lqx.smear_step_range(o, u, 0.5, 1, 3)  # ranges themselves need no contiguity
