"""Pins of the CPU oracle against what the paper and the mathematics fix (SURVEY.md 8(c) table
"What pins each part").  None of these re-types an oracle formula in the oracle's own form:
they are invariants, closed forms, special cases that reduce to numpy routines, and brute force
with explicitly enumerated coordinates on tiny lattices.  CPU only."""
import itertools
import math

import numpy as np
import pytest

import lattice_inputs as li
import oracle as orc
from helpers import cplx, gauge_transform_links, lat4, real2, roll_site, site_rel_err

DIMS_SMALL = [(2, 2, 2, 2), (4, 6, 2, 8), (3, 5, 2, 4), (4, 4, 4, 4)]


def vol(d):
    return int(np.prod(d))


def links(seed, dims, prec="f64", recipe="haar"):
    return [t.numpy() for t in li.gauge_field(seed, dims, prec, recipe)]


def gauss(seed, fid, dims, kind, prec="f64"):
    return li.gaussian_field(seed, fid, dims, kind, prec).numpy()


# ------------------------------------------------------------------------------- geometry (a1)
@pytest.mark.parametrize("dims", DIMS_SMALL)
def test_neighbor_table_brute_force(dims):
    """all 8*V entries against coordinates recomputed by numpy unravel/ravel (x0 fastest)."""
    v = vol(dims)
    coords = np.array(np.unravel_index(np.arange(v), dims, order="F")).T  # [V,4]
    for mu in range(4):
        for sign in (+1, -1):
            c = coords.copy()
            c[:, mu] = (c[:, mu] + sign) % dims[mu]
            want = np.ravel_multi_index(tuple(c.T), dims, order="F")
            got = orc.neighbor_table(dims, sign, mu)
            assert got.dtype == np.int32
            assert np.array_equal(got, want)


@pytest.mark.parametrize("dims", DIMS_SMALL)
def test_neighbor_table_is_permutation_with_inverse_and_period(dims):
    v = vol(dims)
    ident = np.arange(v)
    for mu in range(4):
        f = orc.neighbor_table(dims, +1, mu)
        b = orc.neighbor_table(dims, -1, mu)
        assert np.array_equal(np.sort(f), ident)
        assert np.array_equal(b[f], ident) and np.array_equal(f[b], ident)
        p = ident.copy()
        for _ in range(dims[mu]):
            p = f[p]
        assert np.array_equal(p, ident)


def test_site_index_and_coords_worked_example():
    """site(x) = x0 + L0*(x1 + L1*(x2 + L2*x3)) on a hand-computed case."""
    dims = (4, 6, 2, 8)
    assert orc.site_index(dims, (3, 5, 1, 7)) == 3 + 4 * (5 + 6 * (1 + 2 * 7))
    assert orc.site_coords(dims, 3 + 4 * (5 + 6 * (1 + 2 * 7))) == (3, 5, 1, 7)
    assert orc.site_index(dims, (1, 0, 0, 0)) == 1 and orc.site_index(dims, (0, 1, 0, 0)) == 4


# ------------------------------------------------------------------------------- shift (a3)
@pytest.mark.parametrize("dims", DIMS_SMALL)
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_shift_round_trip_bit_exact(dims, dtype):
    f = gauss(5, 0, dims, "f").astype(dtype)
    for mu in range(4):
        g = orc.shift(dims, orc.shift(dims, f, +1, mu), -1, mu)
        assert np.array_equal(g.view(np.uint8), f.view(np.uint8))


def test_shift_convention_delta_function():
    """shift(f,FORWARD,mu)(x) = f(x+mu^)  (Listing 1 l.25 vs Eq. 2):
    a delta at x0 appears, after a FORWARD shift, at x0 - mu^."""
    dims = (4, 6, 2, 8)
    x0 = (2, 0, 1, 7)
    f = np.zeros((vol(dims), 2))
    f[orc.site_index(dims, x0), 0] = 1.0
    for mu in range(4):
        for sign in (+1, -1):
            g = orc.shift(dims, f, sign, mu)
            x = list(x0)
            x[mu] = (x[mu] - sign) % dims[mu]
            want = np.zeros_like(f)
            want[orc.site_index(dims, x), 0] = 1.0
            assert np.array_equal(g, want)


@pytest.mark.parametrize("dims", DIMS_SMALL)
def test_shift_equals_array_roll(dims):
    f = gauss(6, 1, dims, "cm")
    for mu in range(4):
        for sign in (+1, -1):
            assert np.array_equal(orc.shift(dims, f, sign, mu), roll_site(f, dims, sign, mu))


# ------------------------------------------------------------------------------- site algebra (a4)
@pytest.mark.parametrize("variant", orc.VARIANTS)
def test_form_i_against_numpy_matmul(variant):
    dims = (3, 5, 2, 4)
    dt = np.float32 if variant.endswith("32") else np.float64
    a, b, c, d = (gauss(7, k, dims, "cm").astype(dt) for k in range(4))
    r = orc.mm_plus_madj(dims, a, b, c, d, variant)
    A, B, Cm, D = (cplx(t) for t in (a, b, c, d))
    want = A @ B + Cm @ D.conj().transpose(0, 2, 1)
    tol = 2e-6 if variant == "n32" else 1e-14
    assert site_rel_err(r, real2(want)) < tol


def test_form_i_special_cases_identity_and_zero():
    dims = (2, 2, 2, 2)
    a = gauss(7, 0, dims, "cm")
    one = real2(np.broadcast_to(np.eye(3), (vol(dims), 3, 3)))
    zero = np.zeros_like(a)
    # A*1 + 0 = A bit for bit; 0 + 1*adj(D) = adj(D); adj(adj(A)) = A bit for bit
    assert np.array_equal(orc.mm_plus_madj(dims, a, one, zero, zero, "n64"), a)
    adj_a = orc.mm_plus_madj(dims, zero, zero, one, a, "n64")
    assert np.array_equal(cplx(adj_a), cplx(a).conj().transpose(0, 2, 1))
    assert np.array_equal(orc.mm_plus_madj(dims, zero, zero, one, adj_a, "n64"), a)


def test_su3_products_stay_unitary():
    """products of SU(3) matrices stay unitary to 1e-12 and det = 1 (BASELINE.json north_star)."""
    dims = (4, 4, 4, 4)
    u = links(1, dims)
    zero = np.zeros_like(u[0])
    p = u[0]
    for k in range(1, 4):
        p = orc.mm_plus_madj(dims, p, u[k], zero, zero, "n64")
    for _ in range(8):
        p = orc.mm_plus_madj(dims, p, u[1], zero, zero, "n64")
    P = cplx(p)
    assert np.abs(P @ P.conj().transpose(0, 2, 1) - np.eye(3)).max() < 1e-12
    assert np.abs(np.linalg.det(P) - 1).max() < 1e-12
    assert abs(orc.norm2(dims, p, "n64") - 3 * vol(dims)) < 1e-9


def test_adj_of_product_and_trace_cyclic():
    dims = (3, 5, 2, 4)
    a, b = gauss(7, 0, dims, "cm"), gauss(7, 1, dims, "cm")
    zero = np.zeros_like(a)
    one = real2(np.broadcast_to(np.eye(3), (vol(dims), 3, 3)))
    ab = orc.mm_plus_madj(dims, a, b, zero, zero, "n64")
    adj_ab = orc.mm_plus_madj(dims, zero, zero, one, ab, "n64")
    adj_a = orc.mm_plus_madj(dims, zero, zero, one, a, "n64")
    adj_b = orc.mm_plus_madj(dims, zero, zero, one, b, "n64")
    bdag_adag = orc.mm_plus_madj(dims, adj_b, adj_a, zero, zero, "n64")
    assert site_rel_err(adj_ab, bdag_adag) < 1e-15
    t1, t2 = orc.trace_mm(dims, a, b, "t64"), orc.trace_mm(dims, b, a, "t64")
    assert np.abs(t1 - t2).max() < 1e-13
    assert np.abs(cplx(t1) - np.einsum("xij,xji->x", cplx(a), cplx(b))).max() < 1e-13
    # two code paths: sum_x trace_mm(A, adj A) = norm2(A)
    tt = orc.trace_mm(dims, a, adj_a, "n64")
    s = orc.sum_field(dims, tt, "n64")
    assert abs(s[0] - orc.norm2(dims, a, "n64")) < 1e-9 * s[0] and abs(s[1]) < 1e-9


@pytest.mark.parametrize("dtype,variant", [(np.float32, "n32"), (np.float64, "n64")])
def test_form_iii_exact_zero(dtype, variant):
    """with B = 2.5*shift(A,FORWARD,2): 2.5*A - shift(B,BACKWARD,2) == 0 exactly (native
    arithmetic only: the wide-arithmetic truth keeps the bits B lost when it was rounded)."""
    dims = (4, 6, 4, 2)
    a = gauss(7, 0, dims, "cm").astype(dtype)
    b = orc.shift(dims, (dtype(2.5) * a).astype(dtype), +1, 2)
    r = orc.ax_minus_shift(dims, 2.5, a, b, -1, 2, variant)
    assert np.count_nonzero(r) == 0


def test_form_iii_against_roll():
    dims = (4, 6, 2, 8)
    a, b = gauss(7, 0, dims, "cm"), gauss(7, 1, dims, "cm")
    for mu in range(4):
        for sign in (+1, -1):
            r = orc.ax_minus_shift(dims, 2.5, a, b, sign, mu, "n64")
            assert np.array_equal(r, 2.5 * a - roll_site(b, dims, sign, mu))


def test_form_iv_mat_vec():
    dims = (3, 5, 2, 4)
    u = links(2, dims)[0]
    for kind in ("cv", "f"):
        v = gauss(7, 4, dims, kind)
        w = orc.mat_vec(dims, u, v, "n64")
        # unitary M preserves the norm
        assert abs(orc.norm2(dims, w, "n64") - orc.norm2(dims, v, "n64")) < 1e-10 * orc.norm2(dims, v, "n64")
        if kind == "cv":
            want = np.einsum("xij,xj->xi", cplx(u), cplx(v))
        else:
            want = np.einsum("xij,xaj->xai", cplx(u), cplx(v))
        assert site_rel_err(w, real2(want)) < 1e-14


# ------------------------------------------------------------------------------- hop (a6)
def test_hop_unit_links_constant_psi():
    dims = (4, 4, 2, 6)
    u = links(0, dims, recipe="unit")
    psi = np.broadcast_to(gauss(3, 0, (1, 1, 1, 1), "f"), (vol(dims), 4, 3, 2)).copy()
    chi = orc.hop(dims, u, psi, "n64")
    assert np.array_equal(chi, 8.0 * psi)


@pytest.mark.parametrize("variant", ["n64", "t64"])
def test_hop_u1_plane_wave_eigenvalue(variant):
    """U_mu = exp(i theta_mu) 1, psi = v exp(i p.x): chi = sum_mu 2cos(p_mu+theta_mu) psi.
    A swapped FORWARD/BACKWARD or a missing adj misses by O(1)."""
    dims = (4, 6, 2, 8)
    v_ = vol(dims)
    theta = np.array([0.3, -1.1, 0.7, 2.0])
    n = np.array([1, 2, 1, 3])
    p = 2 * np.pi * n / np.array(dims)
    coords = np.array(np.unravel_index(np.arange(v_), dims, order="F")).T
    phase = np.exp(1j * (coords @ p))
    vec = cplx(gauss(3, 1, (1, 1, 1, 1), "f"))[0]
    psi = real2(phase[:, None, None] * vec[None])
    u = [real2(np.broadcast_to(np.exp(1j * theta[mu]) * np.eye(3), (v_, 3, 3))) for mu in range(4)]
    chi = orc.hop(dims, u, psi, variant)
    lam = np.sum(2 * np.cos(p + theta))
    assert site_rel_err(chi, lam * psi) < 1e-13


def test_hop_point_source():
    """chi(x0 - mu^) = U_mu(x0 - mu^) v ; chi(x0 + mu^) = U_mu(x0)^dagger v ; zero elsewhere."""
    dims = (4, 6, 4, 8)
    u = links(2, dims)
    x0 = (1, 5, 0, 7)
    s0 = orc.site_index(dims, x0)
    vec = gauss(3, 2, (1, 1, 1, 1), "cv")[0]
    psi = np.zeros((vol(dims), 3, 2))
    psi[s0] = vec
    chi = cplx(orc.hop(dims, u, psi, "n64"))
    want = np.zeros_like(chi)
    for mu in range(4):
        xm = list(x0); xm[mu] = (xm[mu] - 1) % dims[mu]
        xp = list(x0); xp[mu] = (xp[mu] + 1) % dims[mu]
        sm, sp = orc.site_index(dims, xm), orc.site_index(dims, xp)
        want[sm] += cplx(u[mu])[sm] @ cplx(vec)
        want[sp] += cplx(u[mu])[s0].conj().T @ cplx(vec)
    assert np.abs(chi - want).max() < 1e-14


def test_hop_gauge_covariance():
    """chi[g U g^dag, g psi] = g chi[U, psi]; the transformation is applied with numpy."""
    dims = (4, 4, 2, 6)
    u = links(2, dims)
    psi = gauss(2, 9, dims, "f")
    g = li.random_gauge_rotation(11, dims).numpy()
    ug = [real2(t) for t in gauge_transform_links([cplx(t) for t in u], g, dims)]
    psig = real2(np.einsum("xij,xaj->xai", g, cplx(psi)))
    chi = cplx(orc.hop(dims, u, psi, "n64"))
    chig = cplx(orc.hop(dims, ug, psig, "n64"))
    assert np.abs(chig - np.einsum("xij,xaj->xai", g, chi)).max() < 1e-13


@pytest.mark.parametrize("variant", ["n32", "n64"])
def test_hop_listing_form_bit_for_bit(variant):
    """Listing 1's shift(adj(u)*psi,BACKWARD,mu) == BASELINE's adj(shift(u,B,mu))*shift(psi,B,mu)."""
    dims = (4, 4, 2, 6)
    dt = np.float32 if variant == "n32" else np.float64
    u = [t.astype(dt) for t in links(2, dims)]
    psi = gauss(2, 9, dims, "f").astype(dt)
    a = orc.hop(dims, u, psi, variant)
    b = orc.hop(dims, u, psi, variant, listing_form=True)
    assert np.array_equal(a.view(np.uint8), b.view(np.uint8))


# ------------------------------------------------------------------------------- staple / smear (a7)
@pytest.mark.parametrize("variant", orc.VARIANTS)
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 4, 4, 4), (3, 5, 2, 4)])
def test_unit_gauge_staple_is_six_and_smear_is_identity(variant, dims):
    prec = "f32" if variant.endswith("32") else "f64"
    u = links(0, dims, prec, "unit")
    for mu in range(4):
        s = orc.staple_sum(dims, u, mu, variant)
        assert np.array_equal(cplx(s), np.broadcast_to(6.0 * np.eye(3), (vol(dims), 3, 3)))
    out = orc.smear_step(dims, u, 0.5, variant)
    for mu in range(4):
        if variant == "t32":   # (float)(a/6) * 6 is not exactly a in fp64 arithmetic: 1 fp32 ulp
            assert np.abs(out[mu] - u[mu]).max() < 1e-7
        else:
            assert np.array_equal(out[mu].astype(np.float64), u[mu].astype(np.float64))


def _brute_force_staple(U, dims, x, mu):
    """explicit coordinates, numpy matmul, dictionary lookup -- tiny lattices only."""
    def at(nu, y):
        return U[nu][tuple(c % L for c, L in zip(y, dims))]
    def sh(y, d, k):
        y = list(y); y[d] += k; return tuple(y)
    acc = np.zeros((3, 3), dtype=complex)
    for nu in range(4):
        if nu == mu:
            continue
        acc += at(nu, x) @ at(mu, sh(x, nu, 1)) @ at(nu, sh(x, mu, 1)).conj().T
        y = sh(x, nu, -1)
        acc += at(nu, y).conj().T @ at(mu, y) @ at(nu, sh(y, mu, 1))
    return acc


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (3, 2, 4, 2)])
def test_staple_brute_force_tiny(dims):
    u = links(1, dims)
    # U[mu][(x0,x1,x2,x3)] lookup built from the QDP site order by explicit enumeration
    U = []
    for mu in range(4):
        c = cplx(u[mu])
        d = {}
        for x in itertools.product(*[range(L) for L in dims]):
            d[x] = c[x[0] + dims[0] * (x[1] + dims[1] * (x[2] + dims[2] * x[3]))]
        U.append(d)
    for mu in range(4):
        s = cplx(orc.staple_sum(dims, u, mu, "t64"))
        for x in itertools.product(*[range(L) for L in dims]):
            sidx = x[0] + dims[0] * (x[1] + dims[1] * (x[2] + dims[2] * x[3]))
            assert np.abs(s[sidx] - _brute_force_staple(U, dims, x, mu)).max() < 1e-14


@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (4, 6, 2, 4), (3, 5, 2, 4)])
def test_staple_sum_equals_the_42_product_order(dims):
    """The evaluation order of the GPU kernels k_smear_rows / k_smear_rowz (DESIGN.md sec.6.1 items 5 and 16) against the
    literal oracle: for a plane a < b the ONE product Z' = U_a(x+b) adj(U_b(x+a)) gives the upper staple of link a,
    U_b(x) Z', and of link b, U_a(x) adj(Z'); the lower staples stay literal.  42 products per site instead of 48, the
    same staple sums (to rounding)."""
    u = links(8, dims)
    U = [cplx(t) for t in u]
    sh = lambda f, sign, mu: cplx(orc.shift(dims, real2(f), sign, mu))
    adj = lambda m: np.conj(np.swapaxes(m, -1, -2))
    S = [np.zeros_like(U[0]) for _ in range(4)]
    nprod = 0
    for a in range(4):
        for b in range(a + 1, 4):
            z = sh(U[a], +1, b) @ adj(sh(U[b], +1, a))  # Z'_ab(x)
            S[a] += U[b] @ z
            S[b] += U[a] @ adj(z)
            nprod += 3
    for mu in range(4):
        for nu in range(4):
            if nu == mu:
                continue
            # lower staple of link mu in plane nu: adj(U_nu(x-nu)) U_mu(x-nu) U_nu(x-nu+mu)
            t = adj(sh(U[nu], -1, nu)) @ sh(U[mu], -1, nu)
            S[mu] += t @ sh(sh(U[nu], -1, nu), +1, mu)
            nprod += 2
    assert nprod == 42
    for mu in range(4):
        want = cplx(orc.staple_sum(dims, u, mu, "t64"))
        assert np.abs(S[mu] - want).max() < 1e-13, mu


def test_staple_abelian_closed_form():
    """diagonal U(1)^3 links with random phases: every staple is a sum/difference of phases."""
    dims = (4, 6, 2, 4)
    v_ = vol(dims)
    rng = np.random.default_rng(5)
    phi = rng.uniform(-np.pi, np.pi, size=(4, v_, 3))
    u = []
    for mu in range(4):
        m = np.zeros((v_, 3, 3), dtype=complex)
        for a in range(3):
            m[:, a, a] = np.exp(1j * phi[mu, :, a])
        u.append(real2(m))
    for mu in range(4):
        want = np.zeros((v_, 3), dtype=complex)
        for nu in range(4):
            if nu == mu:
                continue
            up = phi[nu] + roll_site(phi[mu], dims, +1, nu) - roll_site(phi[nu], dims, +1, mu)
            lo_at_y = -phi[nu] + phi[mu] + roll_site(phi[nu], dims, +1, mu)   # lives at y = x - nu^
            want += np.exp(1j * up) + np.exp(1j * roll_site(lo_at_y, dims, -1, nu))
        s = cplx(orc.staple_sum(dims, u, mu, "n64"))
        assert np.abs(s[:, [0, 1, 2], [0, 1, 2]] - want).max() < 1e-13
        off = s.copy(); off[:, [0, 1, 2], [0, 1, 2]] = 0
        assert np.abs(off).max() == 0


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 4, 2, 6)])
def test_smear_step_gauge_covariance(dims):
    """U'_mu[g U g^dag](x) = g(x) U'_mu[U](x) g(x+mu^)^dag  (non-abelian: catches operand order)."""
    u = links(1, dims)
    g = li.random_gauge_rotation(12, dims).numpy()
    ug = [real2(t) for t in gauge_transform_links([cplx(t) for t in u], g, dims)]
    out = [cplx(t) for t in orc.smear_step(dims, u, 0.5, "n64")]
    outg = [cplx(t) for t in orc.smear_step(dims, ug, 0.5, "n64")]
    want = gauge_transform_links(out, g, dims)
    for mu in range(4):
        assert np.abs(outg[mu] - want[mu]).max() < 1e-13


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (3, 5, 2, 4)])
def test_staple_plaquette_identity(dims):
    """sum_{x,mu} Re tr[U_mu(x) S_mu(x)^dag] = 4 * plaquette sum (two oracle code paths)."""
    u = links(1, dims)
    lhs = 0.0
    for mu in range(4):
        s = cplx(orc.staple_sum(dims, u, mu, "n64"))
        lhs += np.einsum("xij,xij->", cplx(u[mu]), s.conj()).real
    p = orc.plaquette_sum(dims, u, "n64")
    assert abs(lhs - 4 * p) < 1e-10 * max(1.0, abs(lhs))


def test_smear_coefficients_and_alpha_limits():
    """alpha = 0 returns the input; U' - (1-a)U = (a/6) S."""
    dims = (2, 4, 2, 4)
    u = links(3, dims)
    out0 = orc.smear_step(dims, u, 0.0, "n64")
    for mu in range(4):
        assert np.array_equal(out0[mu], u[mu])
    a = 0.3
    out = orc.smear_step(dims, u, a, "t64")
    for mu in range(4):
        s = orc.staple_sum(dims, u, mu, "t64")
        assert site_rel_err(out[mu], (1 - a) * u[mu] + (a / 6) * s) < 1e-15


def test_smear_links_matches_smear_step():
    dims = (4, 4, 4, 4)
    u = links(1, dims)
    rng = np.random.default_rng(0)
    sites = rng.integers(0, vol(dims), size=50)
    mus = rng.integers(0, 4, size=50)
    full = orc.smear_step(dims, u, 0.5, "t64")
    got = orc.smear_links(dims, u, 0.5, sites, mus, "t64")
    for k in range(50):
        assert np.array_equal(got[k], full[mus[k]][sites[k]])


def test_smear_output_leaves_su3():
    """reading A9: no projection -- U' is not unitary for Haar input, and that is expected."""
    dims = (4, 4, 4, 4)
    u = links(1, dims)
    out = cplx(orc.smear_step(dims, u, 0.5, "n64")[0])
    dev = np.abs(out @ out.conj().transpose(0, 2, 1) - np.eye(3)).max()
    assert dev > 0.1


# ------------------------------------------------------------------------------- plaquette (a8)
@pytest.mark.parametrize("variant", orc.VARIANTS)
def test_plaquette_unit_links_is_one(variant):
    dims = (4, 2, 6, 4)
    prec = "f32" if variant.endswith("32") else "f64"
    u = links(0, dims, prec, "unit")
    assert orc.plaquette_avg(dims, u, variant) == 1.0
    assert orc.plaquette_sum(dims, u, variant) == 18.0 * vol(dims)


def test_plaquette_gauge_invariance_and_haar_mean():
    dims = (4, 4, 4, 4)
    u = links(1, dims)
    g = li.random_gauge_rotation(13, dims).numpy()
    ug = [real2(t) for t in gauge_transform_links([cplx(t) for t in u], g, dims)]
    p, pg = orc.plaquette_sum(dims, u, "t64"), orc.plaquette_sum(dims, ug, "t64")
    assert abs(p - pg) < 1e-11 * 18 * vol(dims)
    # Haar links: E[Re tr P] = 0, Var = 1/2 per plaquette -> avg within 5 sigma of 0
    sigma = math.sqrt(0.5 * 6 * vol(dims)) / (18 * vol(dims))
    assert abs(p / (18 * vol(dims))) < 5 * sigma


def test_plaquette_against_numpy_roll():
    dims = (3, 5, 2, 4)
    u = links(2, dims)
    U = [cplx(t) for t in u]
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            m = U[mu] @ roll_site(U[nu], dims, +1, mu) @ roll_site(U[mu], dims, +1, nu).conj().transpose(0, 2, 1) \
                @ U[nu].conj().transpose(0, 2, 1)
            tot += np.trace(m, axis1=1, axis2=2).real.sum()
    assert abs(orc.plaquette_sum(dims, u, "n64") - tot) < 1e-11 * 18 * vol(dims)
    sites = np.arange(vol(dims))
    per = orc.plaquette_sites(dims, u, sites, "n64")
    assert abs(math.fsum(per) - orc.plaquette_sum(dims, u, "t64")) < 1e-10


def test_plaquette_near_unit_recipe_is_close_to_one():
    dims = (4, 4, 4, 4)
    u = links(4, dims, "f32", "near_unit")
    p = orc.plaquette_avg(dims, u, "t32")
    assert 0.8 < p < 1.0


# ------------------------------------------------------------------------------- reductions (a9)
@pytest.mark.parametrize("variant", orc.VARIANTS)
def test_reductions_against_fsum(variant):
    dims = (4, 6, 2, 8)
    dt = np.float32 if variant.endswith("32") else np.float64
    f = gauss(9, 0, dims, "cm").astype(dt)
    s = orc.sum_field(dims, f, variant)
    f64 = f.astype(np.float64).reshape(vol(dims), -1)
    want = np.array([math.fsum(f64[:, k]) for k in range(18)]).reshape(3, 3, 2)
    assert np.abs(s - want).max() < 1e-12 * np.abs(f64).sum(axis=0).max()
    n2 = orc.norm2(dims, f, variant)
    assert abs(n2 - math.fsum((f64 ** 2).ravel())) < 1e-13 * n2
    t = orc.trace(dims, f, variant)
    c = cplx(f)
    wt = [math.fsum(np.trace(c, axis1=1, axis2=2).real), math.fsum(np.trace(c, axis1=1, axis2=2).imag)]
    assert np.abs(t - wt).max() < 1e-12 * np.abs(f64).sum(axis=0).max()


def test_sum_of_constant_field():
    dims = (4, 4, 2, 2)
    one = gauss(1, 0, (1, 1, 1, 1), "cv")
    f = np.broadcast_to(one, (vol(dims), 3, 2)).copy()
    assert np.allclose(orc.sum_field(dims, f, "t64"), vol(dims) * one[0], rtol=1e-15, atol=0)


# ------------------------------------------------------------------------------- E0/E3/E4 pieces
@pytest.mark.parametrize("variant", ["n32", "n64"])
@pytest.mark.parametrize("kind", ["f", "cv"])
def test_axpy_and_divide_compose_to_one_jacobi_iteration(variant, kind):
    """Two code paths of the oracle: Listing 1 with iter = 1 (orc_jacobi_smear) is, line by line, E1/E2 (the hop),
    E3 `chi = s_0 + kappa*h` and E4 `chi /= norm`.  Built from the separate routines hop, axpy
    and divide it must give the same numbers BIT FOR BIT in the native variants; a wrong operand order or sign in
    axpy (s_0 and h swapped, kappa on the wrong term) or a multiply in divide misses by O(1)."""
    dims = (4, 2, 6, 2)
    dt = np.float32 if variant == "n32" else np.float64
    u = [t.astype(dt) for t in links(6, dims)]
    chi = gauss(6, 3, dims, kind).astype(dt)
    kappa, norm = 0.23, 1.9
    whole = orc.jacobi_smear(dims, u, chi, kappa, 1, -1, norm, variant)
    pieces = orc.divide(dims, norm, orc.axpy(dims, chi, kappa, orc.hop(dims, u, chi, variant), variant), variant)
    assert np.array_equal(whole, pieces)
    # iter = 0 is E4 alone
    assert np.array_equal(orc.jacobi_smear(dims, u, chi, kappa, 0, -1, norm, variant), orc.divide(dims, norm, chi, variant))


@pytest.mark.parametrize("variant", ["n32", "n64", "t32", "t64"])
def test_scale_against_divide_and_linearity(variant):
    """scale(1/n) and divide(n) are the same map up to one rounding of 1/n and one of the product (reading A22);
    divide by a power of two is exact; axpy is linear in kappa: axpy(a, 2k, b) - axpy(a, k, b) = k*b up to rounding,
    axpy(a, 0, b) = a exactly, axpy(0, 1, b) = b exactly."""
    dims = (2, 4, 2, 4)
    a, b = (gauss(8, k, dims, "f").astype(np.float32 if variant.endswith("32") else np.float64) for k in (0, 1))
    # scalars are rounded once to the FIELD precision in every variant, so 1/n and n carry fp32 roundings in t32 too
    eps = 2.0 ** -23 if variant.endswith("32") else 2.0 ** -52
    n = 1.7
    s, d = orc.scale(dims, 1.0 / n, a, variant).astype(np.float64), orc.divide(dims, n, a, variant).astype(np.float64)
    assert np.abs(s - d).max() <= 2.5 * eps * np.abs(d).max()
    assert np.array_equal(orc.divide(dims, 4.0, a, variant), orc.scale(dims, 0.25, a, variant))
    assert np.array_equal(orc.divide(dims, 4.0, a, variant).astype(np.float64), a.astype(np.float64) / 4.0)
    assert np.array_equal(orc.axpy(dims, a, 0.0, b, variant).astype(np.float64), a.astype(np.float64))
    assert np.array_equal(orc.axpy(dims, np.zeros_like(a), 1.0, b, variant).astype(np.float64), b.astype(np.float64))
    k = 0.375  # exactly representable, so k*b is one rounding
    diff = orc.axpy(dims, a, 2 * k, b, variant).astype(np.float64) - orc.axpy(dims, a, k, b, variant).astype(np.float64)
    assert np.abs(diff - k * b.astype(np.float64)).max() <= 4 * eps * (np.abs(a).max() + np.abs(b).max())


# ------------------------------------------------------------------------------- a10: the trajectory driver
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_smear_iterate_on_unit_links_is_constant(prec):
    """unit links are a fixed point of the step (S = 6, U' = U): every plaquette average is exactly 1 and the
    field never changes, however many steps."""
    dims = (4, 2, 4, 2)
    u = links(0, dims, prec, "unit")
    out, plaqs = orc.smear_iterate(dims, u, 0.5, 4, prec)
    if prec == "f64":
        assert plaqs == [1.0, 1.0, 1.0, 1.0]
        for mu in range(4):
            assert np.array_equal(out[mu], u[mu])
    else:
        # Step 1 runs in the truth variant of fp32, whose a/6 is rounded to fp32 (reading A10): 6 * c1 = 0.5 (1 + 3e-8),
        # so the links become 1 + d with d = 6 c1 - 0.5.  The later steps run in fp64 with the exact coefficient (A23),
        # where U = 1 + d maps to 1 + 2 d (the fixed point has eigenvalue 2): d doubles per step.  This pins the
        # driver's switch of variant after the first step -- without it d would grow as 2^k - 1.
        d1 = 6.0 * float(np.float32(0.5 / 6.0)) - 0.5
        for k, p in enumerate(plaqs):
            assert abs(p - (1.0 + d1 * 2 ** k) ** 4) < 1e-12, k
        for mu in range(4):
            assert np.abs(out[mu] - (1.0 + d1 * 8) * u[mu]).max() < 1e-12


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_smear_iterate_with_alpha_zero_is_constant(prec):
    """alpha = 0: U' = U, so the trajectory is constant and every reported plaquette is the input's."""
    dims = (2, 4, 2, 4)
    u = links(3, dims, prec)
    out, plaqs = orc.smear_iterate(dims, u, 0.0, 3, prec)
    p0 = orc.plaquette_avg(dims, u, orc.truth_variant(prec))
    assert all(abs(p - p0) < 1e-14 for p in plaqs)
    for mu in range(4):
        assert np.array_equal(out[mu].astype(np.float64), u[mu].astype(np.float64))


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_smear_iterate_equals_explicit_steps(prec):
    """The driver is n explicit smear_step calls with the plaquette of each OUTPUT (reading A11 for configs[3]):
    the plaquette reported for step k is that of the field AFTER step k, not before it, and the links returned are
    those after the last step.  Rebuilt here from smear_step / plaquette_avg calls written out one by one; the first
    step starts from the storage-precision field with wide arithmetic, the later ones stay in fp64 (A23)."""
    dims = (4, 4, 2, 6)
    u0 = links(4, dims, prec, "near_unit")
    out, plaqs = orc.smear_iterate(dims, u0, 0.5, 3, prec)
    tv = orc.truth_variant(prec)
    later = "t64" if prec == "f64" else "n64"
    u1 = orc.smear_step(dims, u0, 0.5, tv)
    u2 = orc.smear_step(dims, u1, 0.5, later)
    u3 = orc.smear_step(dims, u2, 0.5, later)
    want = [orc.plaquette_avg(dims, u1, later), orc.plaquette_avg(dims, u2, later), orc.plaquette_avg(dims, u3, later)]
    assert plaqs == want
    for mu in range(4):
        assert np.array_equal(out[mu], u3[mu])
    # and none of the reported values is the plaquette BEFORE its step
    before = [orc.plaquette_avg(dims, u0, tv), want[0], want[1]]
    assert all(abs(p - b) > 1e-3 for p, b in zip(plaqs, before))
    # one step of the driver = smear_step + plaquette_avg of its output
    out1, p1 = orc.smear_iterate(dims, u0, 0.5, 1, prec)
    assert p1 == [want[0]] and all(np.array_equal(a, b) for a, b in zip(out1, u1))


def test_smear_iterate_plaquette_is_gauge_invariant_and_matches_numpy():
    """the whole trajectory of plaquettes is invariant under a gauge transformation of the start (the step is gauge
    covariant), and the first value equals a numpy-roll evaluation of the plaquette of smear_step's output."""
    dims = (4, 2, 2, 4)
    u = links(5, dims, "f64", "near_unit")
    g = cplx(li.gauge_field(9, dims, "f64", "haar")[0].numpy())
    ug = [real2(t) for t in gauge_transform_links([cplx(t) for t in u], g, dims)]
    _, p = orc.smear_iterate(dims, u, 0.5, 3, "f64")
    _, pg = orc.smear_iterate(dims, ug, 0.5, 3, "f64")
    assert np.allclose(p, pg, rtol=0, atol=1e-13)
    u1 = [cplx(t) for t in orc.smear_step(dims, u, 0.5, "t64")]
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            a = np.einsum("xij,xjk->xik", u1[mu], roll_site(u1[nu], dims, +1, mu))
            b = np.einsum("xij,xjk->xik", u1[nu], roll_site(u1[mu], dims, +1, nu))
            tot += np.einsum("xij,xij->", a, b.conj()).real
    assert abs(p[0] - tot / (18.0 * vol(dims))) < 1e-13


# ------------------------------------------------------------------------------- variants agree
def test_native_and_truth_variants_agree_within_fair_tolerance():
    """shows BASELINE's tolerances are fair: native fp64 vs x87 truth ~1e-15, native fp32 vs
    fp64-arithmetic truth ~1e-6 (site-normalised, reading A14)."""
    dims = (4, 4, 4, 4)
    u64 = links(1, dims, "f64")
    u32 = links(1, dims, "f32")
    o_n64, o_t64 = orc.smear_step(dims, u64, 0.5, "n64"), orc.smear_step(dims, u64, 0.5, "t64")
    o_n32, o_t32 = orc.smear_step(dims, u32, 0.5, "n32"), orc.smear_step(dims, u32, 0.5, "t32")
    for mu in range(4):
        assert site_rel_err(o_n64[mu], o_t64[mu]) < 5e-15
        assert site_rel_err(o_n32[mu], o_t32[mu]) < 3e-6
