"""Pins of the oracle's Jacobi smearing routine (Listing 1) against
what the paper fixes: it is the power series in kappa of the inverse of K = 1 - kappa*H truncated at
N_smear, i.e. chi = sum_{n<=N} kappa^n H^n s_0 / norm.  H is built here from numpy
rolls and einsum (helpers.roll_site), never from the oracle.  CPU only."""
import numpy as np
import pytest

import lattice_inputs as li
import oracle as orc
from helpers import cplx, gauge_transform_links, real2, roll_site, site_rel_err


def vol(d):
    return int(np.prod(d))


def links(seed, dims, prec="f64", recipe="haar"):
    return [t.numpy() for t in li.gauge_field(seed, dims, prec, recipe)]


def gauss(seed, fid, dims, kind, prec="f64"):
    return li.gaussian_field(seed, fid, dims, kind, prec).numpy()


def hop_numpy(u, psi, dims, skip=-1):
    """H psi with array rolls: sum_mu U_mu(x) psi(x+mu) + U_mu(x-mu)^dag psi(x-mu); psi complex [V,a,3]."""
    out = np.zeros_like(psi)
    for mu in range(4):
        if mu == skip:
            continue
        um = cplx(u[mu])
        out += np.einsum("xij,xaj->xai", um, roll_site(psi, dims, +1, mu))
        ub = roll_site(um, dims, -1, mu)
        out += np.einsum("xji,xaj->xai", ub.conj(), roll_site(psi, dims, -1, mu))
    return out


@pytest.mark.parametrize("variant", ["n64", "t64"])
@pytest.mark.parametrize("skip", [-1, 3, 0])
def test_jacobi_is_the_truncated_power_series(variant, skip):
    dims = (4, 6, 2, 4)
    u = links(2, dims)
    chi0 = gauss(2, 10, dims, "f")
    kappa, iters, norm = 0.21, 5, 1.7
    got = orc.jacobi_smear(dims, u, chi0, kappa, iters, skip, norm, variant)
    s0 = cplx(chi0)
    term, want = s0.copy(), s0.copy()
    for n in range(1, iters + 1):
        term = kappa * hop_numpy(u, term, dims, skip)
        want = want + term
    assert site_rel_err(got, real2(want / norm)) < 1e-13


def test_jacobi_zero_iterations_and_zero_kappa():
    dims = (2, 4, 2, 2)
    u = links(1, dims)
    chi0 = gauss(1, 3, dims, "cv")
    assert np.array_equal(orc.jacobi_smear(dims, u, chi0, 0.3, 0, -1, 2.0, "n64"), chi0 / 2.0)
    assert np.array_equal(orc.jacobi_smear(dims, u, chi0, 0.0, 4, -1, 1.0, "n64"), chi0)


@pytest.mark.parametrize("skip,ndir", [(-1, 4), (3, 3), (7, 4)])
def test_jacobi_unit_links_constant_source_is_a_geometric_series(skip, ndir):
    """H s = 2*ndir*s on unit links and a constant field: chi = sum_n (2 ndir kappa)^n s / norm."""
    dims = (4, 4, 2, 6)
    u = links(0, dims, recipe="unit")
    s = np.broadcast_to(gauss(3, 0, (1, 1, 1, 1), "f"), (vol(dims), 4, 3, 2)).copy()
    kappa, iters, norm = 0.0625, 6, 3.0
    got = orc.jacobi_smear(dims, u, s, kappa, iters, skip, norm, "n64")
    q = 2 * ndir * kappa
    assert site_rel_err(got, s * sum(q ** n for n in range(iters + 1)) / norm) < 1e-14


def test_jacobi_u1_plane_wave_eigenvalue():
    """A plane wave on U(1) links is an eigenvector of H with lambda = sum_mu 2cos(p_mu + theta_mu), so
    the routine multiplies it by sum_n (kappa lambda)^n / norm; a wrong shift sign misses by O(1)."""
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
    lam = np.sum(2 * np.cos(p + theta))
    kappa, iters = 0.11, 7
    got = orc.jacobi_smear(dims, u, psi, kappa, iters, -1, 1.0, "t64")
    assert site_rel_err(got, psi * sum((kappa * lam) ** k for k in range(iters + 1))) < 1e-13


def test_jacobi_gauge_covariance():
    dims = (4, 4, 2, 4)
    u = links(2, dims)
    chi0 = gauss(2, 9, dims, "f")
    g = li.random_gauge_rotation(11, dims).numpy()
    ug = [real2(t) for t in gauge_transform_links([cplx(t) for t in u], g, dims)]
    chig = real2(np.einsum("xij,xaj->xai", g, cplx(chi0)))
    a = cplx(orc.jacobi_smear(dims, u, chi0, 0.2, 3, -1, 1.3, "n64"))
    b = cplx(orc.jacobi_smear(dims, ug, chig, 0.2, 3, -1, 1.3, "n64"))
    assert np.abs(b - np.einsum("xij,xaj->xai", g, a)).max() < 1e-12


def test_jacobi_native_fp32_tracks_truth():
    dims = (4, 4, 4, 4)
    u = links(2, dims, "f32")
    chi0 = gauss(2, 5, dims, "f", "f32")
    a = orc.jacobi_smear(dims, u, chi0, 0.15, 8, -1, 2.0, "n32")
    b = orc.jacobi_smear(dims, u, chi0, 0.15, 8, -1, 2.0, "t32")
    assert site_rel_err(a, b) < 8 * 1e-6
