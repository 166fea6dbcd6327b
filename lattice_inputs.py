"""Seeded synthetic lattice inputs (the ONLY module shared by the oracle side and the CUDA side).

Holds no arithmetic of the method (no shift, no staple, no hop, no reduction) -- only the input
recipes of BASELINE.json `configs` as read in DESIGN.md section 4:

* a counter-based generator: 64-bit mix of (seed, field id, site, complex index) -> two uniforms
  -> Box-Muller -> one complex Gaussian with N(0,1) real and imaginary parts.  Order- and
  thread-count-independent, identical on CPU and GPU up to libm rounding of log/sin/cos;
* Haar-random SU(3): modified Gram-Schmidt on the columns of a complex Gaussian 3x3 (R diagonal
  real positive = the phase fix), then det^(-1/3) (principal branch) multiplied in;
* near-unit SU(3): exp(i*eps*H), H traceless Hermitian from a Gaussian matrix, Taylor series,
  then row-wise reunitarisation.

All fields are returned in the external "QDP++ order": site-major, sites
lexicographic with x0 fastest, inside a site [row][col][re,im] (matrix), [spin][colour][re,im]
(fermion), [colour][re,im] (vector), [re,im] (complex) -- as a real tensor whose last dim is 2.
Everything is computed in fp64 and only then rounded to the requested precision, so the oracle
and the CUDA path consume bit-identical arrays.
"""
from __future__ import annotations

import math

import torch

# BASELINE.json configs -> geometry, precision, seed (seeds: SURVEY.md 8(c) A19)
CONFIGS = {
    "c1": {"dims": (4, 4, 4, 4), "prec": "f64", "seed": 1},
    "c2": {"dims": (16, 16, 16, 32), "prec": "f32", "seed": 2},
    "c3": {"dims": (32, 32, 32, 64), "prec": "f64", "seed": 3},
    "c4": {"dims": (48, 48, 48, 96), "prec": "f32", "seed": 4},
    "c5": {"dims": (32, 32, 32, 64), "prec": "f32+f64", "seed": 7},
}

_MASK64 = (1 << 64) - 1


def _i64(c: int) -> int:
    """Python int (mod 2^64) -> the int64 with the same bit pattern."""
    c &= _MASK64
    return c - (1 << 64) if c >= (1 << 63) else c


_GOLDEN = _i64(0x9E3779B97F4A7C15)
_M1 = _i64(0xBF58476D1CE4E5B9)
_M2 = _i64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    """Logical shift right on int64 bit patterns."""
    return (x >> k) & ((1 << (64 - k)) - 1)


def _mix64(x: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser on int64 tensors (wrapping arithmetic = arithmetic mod 2^64)."""
    x = x + _GOLDEN
    x = (x ^ _lsr(x, 30)) * _M1
    x = (x ^ _lsr(x, 27)) * _M2
    return x ^ _lsr(x, 31)


def _mix64_int(x: int) -> int:
    x = (x + 0x9E3779B97F4A7C15) & _MASK64
    x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
    x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & _MASK64
    return x ^ (x >> 31)


def volume(dims) -> int:
    v = 1
    for d in dims:
        v *= int(d)
    return v


def gaussian_complex(seed: int, field_id: int, nsites: int, ncomplex: int,
                     device="cpu", site_offset: int = 0) -> torch.Tensor:
    """[nsites, ncomplex] complex128, re and im i.i.d. N(0,1); element (s,k) depends only on
    (seed, field_id, s + site_offset, k)."""
    key = _i64(_mix64_int(_mix64_int(seed & _MASK64) ^ ((field_id + 1) * 0xD1342543DE82EF95 & _MASK64)))
    s = torch.arange(site_offset, site_offset + nsites, dtype=torch.int64, device=device)
    k = torch.arange(ncomplex, dtype=torch.int64, device=device)
    ctr = (s[:, None] * ncomplex + k[None, :]) * 2
    z1 = _mix64(ctr + key)
    z2 = _mix64(ctr + 1 + key)
    two53 = float(1 << 53)
    u1 = (_lsr(z1, 11).to(torch.float64) + 0.5) / two53
    u2 = (_lsr(z2, 11).to(torch.float64) + 0.5) / two53
    r = torch.sqrt(-2.0 * torch.log(u1))
    th = (2.0 * math.pi) * u2
    return torch.complex(r * torch.cos(th), r * torch.sin(th))


def _as_real(z: torch.Tensor, prec: str) -> torch.Tensor:
    out = torch.view_as_real(z.contiguous())
    if prec == "f32":
        return out.to(torch.float32).contiguous()
    if prec == "f64":
        return out.contiguous()
    raise ValueError(prec)


def gaussian_field(seed, field_id, dims, kind: str, prec: str, device="cpu") -> torch.Tensor:
    """Gaussian LatticeColorMatrix 'cm' [V,3,3,2], LatticeColorVector 'cv' [V,3,2],
    LatticeFermion 'f' [V,4,3,2] or LatticeComplex 'c' [V,2] in QDP order."""
    shape = {"cm": (3, 3), "cv": (3,), "f": (4, 3), "c": ()}[kind]
    n = 1
    for d in shape:
        n *= d
    v = volume(dims)
    z = gaussian_complex(seed, field_id, v, n, device).reshape((v,) + shape)
    return _as_real(z, prec)


def _gram_schmidt_columns(g: torch.Tensor) -> torch.Tensor:
    """Modified Gram-Schmidt on the columns of g [V,3,3] (complex128); R diagonal real > 0."""
    c0, c1, c2 = g[:, :, 0], g[:, :, 1], g[:, :, 2]
    q0 = c0 / torch.linalg.vector_norm(c0, dim=1, keepdim=True)
    c1 = c1 - q0 * (q0.conj() * c1).sum(dim=1, keepdim=True)
    q1 = c1 / torch.linalg.vector_norm(c1, dim=1, keepdim=True)
    c2 = c2 - q0 * (q0.conj() * c2).sum(dim=1, keepdim=True)
    c2 = c2 - q1 * (q1.conj() * c2).sum(dim=1, keepdim=True)
    q2 = c2 / torch.linalg.vector_norm(c2, dim=1, keepdim=True)
    return torch.stack((q0, q1, q2), dim=2)


def _det3(m: torch.Tensor) -> torch.Tensor:
    return (m[:, 0, 0] * (m[:, 1, 1] * m[:, 2, 2] - m[:, 1, 2] * m[:, 2, 1])
            - m[:, 0, 1] * (m[:, 1, 0] * m[:, 2, 2] - m[:, 1, 2] * m[:, 2, 0])
            + m[:, 0, 2] * (m[:, 1, 0] * m[:, 2, 1] - m[:, 1, 1] * m[:, 2, 0]))


def haar_su3_complex(seed, field_id, nsites, device="cpu") -> torch.Tensor:
    """[nsites,3,3] complex128 Haar-random SU(3) (BASELINE.json configs[0] recipe, A16)."""
    g = gaussian_complex(seed, field_id, nsites, 9, device).reshape(nsites, 3, 3)
    q = _gram_schmidt_columns(g)
    phi = torch.angle(_det3(q))
    ph = torch.polar(torch.ones_like(phi), -phi / 3.0)
    return q * ph[:, None, None]


def near_unit_su3_complex(seed, field_id, nsites, eps=0.1, device="cpu") -> torch.Tensor:
    """[nsites,3,3] complex128: exp(i*eps*H) reunitarised (BASELINE.json configs[3] recipe, A17)."""
    g = gaussian_complex(seed, field_id, nsites, 9, device).reshape(nsites, 3, 3)
    h = 0.5 * (g + g.conj().transpose(1, 2))
    tr = (h[:, 0, 0] + h[:, 1, 1] + h[:, 2, 2]) / 3.0
    eye = torch.eye(3, dtype=torch.complex128, device=g.device)
    h = h - tr[:, None, None] * eye
    x = (1j * eps) * h
    term = eye.expand(nsites, 3, 3).clone()
    acc = term.clone()
    for n in range(1, 25):  # |x| ~ 0.5 -> 0.5^24/24! far below 1e-17
        term = torch.matmul(term, x) / n
        acc = acc + term
    # reunitarise: normalise row 0, Gram-Schmidt row 1, row 2 = conj(row0 x row1)
    r0 = acc[:, 0, :]
    r0 = r0 / torch.linalg.vector_norm(r0, dim=1, keepdim=True)
    r1 = acc[:, 1, :]
    r1 = r1 - r0 * (r0.conj() * r1).sum(dim=1, keepdim=True)
    r1 = r1 / torch.linalg.vector_norm(r1, dim=1, keepdim=True)
    r2 = torch.stack((r0[:, 1] * r1[:, 2] - r0[:, 2] * r1[:, 1],
                      r0[:, 2] * r1[:, 0] - r0[:, 0] * r1[:, 2],
                      r0[:, 0] * r1[:, 1] - r0[:, 1] * r1[:, 0]), dim=1).conj()
    return torch.stack((r0, r1, r2), dim=1)


def gauge_field(seed, dims, prec: str, recipe="haar", device="cpu", eps=0.1):
    """multi1d<LatticeColorMatrix> u(Nd): list of 4 tensors [V,3,3,2] in QDP order.
    Field ids 0..3 are the link directions."""
    v = volume(dims)
    out = []
    for mu in range(4):
        if recipe == "haar":
            z = haar_su3_complex(seed, mu, v, device)
        elif recipe == "near_unit":
            z = near_unit_su3_complex(seed, mu, v, eps, device)
        elif recipe == "unit":
            z = torch.eye(3, dtype=torch.complex128, device=device).expand(v, 3, 3).clone()
        else:
            raise ValueError(recipe)
        out.append(_as_real(z, prec))
    return out


def random_gauge_rotation(seed, dims, device="cpu") -> torch.Tensor:
    """g(x): [V,3,3] complex128 Haar SU(3), field id 100 (used by gauge-covariance pins)."""
    return haar_su3_complex(seed, 100, volume(dims), device)
