"""Test-side helpers (numpy only): views of QDP-order arrays, gauge transformations, error
norms.  Nothing here is used by the product path or by the oracle."""
import numpy as np


def cplx(a):
    """QDP-order real array [..., 2] -> complex array [...] (fp64)."""
    a = np.asarray(a, dtype=np.float64)
    return a[..., 0] + 1j * a[..., 1]


def real2(z, dtype=np.float64):
    z = np.asarray(z)
    return np.ascontiguousarray(np.stack((z.real, z.imag), axis=-1).astype(dtype))


def lat4(field, dims):
    """[V, ...] site-major (x0 fastest) -> [L3, L2, L1, L0, ...]"""
    return field.reshape(tuple(reversed(dims)) + field.shape[1:])


def roll_site(field, dims, sign, mu):
    """f(x + sign*mu^) as an array op: independent of any neighbour table."""
    f4 = lat4(field, dims)
    return np.roll(f4, -sign, axis=3 - mu).reshape(field.shape)


def gauge_transform_links(u, g, dims):
    """U_mu(x) -> g(x) U_mu(x) g(x+mu^)^dagger ; u: list of complex [V,3,3], g complex [V,3,3]"""
    out = []
    for mu in range(4):
        gf = roll_site(g, dims, +1, mu)
        out.append(np.einsum("xij,xjk,xlk->xil", g, u[mu], gf.conj()))
    return out


def site_rel_err(got, want):
    """DESIGN.md reading A14: max_i |g_i - o_i| / max(|o_i|, m_site(i)), m_site = largest
    component magnitude of the oracle's site object containing i.  Arrays are [V, ...]."""
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    v = want.shape[0]
    w = np.abs(want.reshape(v, -1))
    m = w.max(axis=1, keepdims=True)
    m = np.where(m == 0.0, 1.0, m)
    d = np.abs(got.reshape(v, -1) - want.reshape(v, -1))
    return float((d / np.maximum(w, m)).max()) if d.size else 0.0


def strict_rel_err(got, want):
    got = np.asarray(got, dtype=np.float64).ravel()
    want = np.asarray(want, dtype=np.float64).ravel()
    nz = want != 0
    return float((np.abs(got - want)[nz] / np.abs(want[nz])).max()) if nz.any() else 0.0
