"""ctypes binding of the CPU oracle (oracle/lattice_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It imports nothing from the CUDA package.  All fields are numpy arrays in QDP order
(see lattice_oracle.cpp header); `variant` selects the instantiation:

    n32  fp32 in, fp32 arithmetic, fp32 out   (native, timed)
    t32  fp32 in, fp64 arithmetic, fp64 out   (truth for fp32 configs)
    n64  fp64 in, fp64 arithmetic, fp64 out   (native, timed)
    t64  fp64 in, x87 long double arithmetic, fp64 out (truth for fp64 configs)
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_IN = {"n32": np.float32, "t32": np.float32, "n64": np.float64, "t64": np.float64}
_OUT = {"n32": np.float32, "t32": np.float64, "n64": np.float64, "t64": np.float64}
VARIANTS = tuple(_IN)

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_norm2_n32.restype = C.c_double
        for v in VARIANTS:
            getattr(_lib, f"orc_norm2_{v}").restype = C.c_double
            getattr(_lib, f"orc_plaquette_sum_{v}").restype = C.c_double
        _lib.orc_site_index.restype = C.c_long
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def truth_variant(prec: str) -> str:
    return {"f32": "t32", "f64": "t64"}[prec]


def native_variant(prec: str) -> str:
    return {"f32": "n32", "f64": "n64"}[prec]


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> None:
    lib().orc_set_num_threads(int(n))


def _dims(dims):
    return (C.c_int * 4)(*[int(d) for d in dims])


def _vol(dims):
    return int(np.prod([int(d) for d in dims]))


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _inp(a, variant):
    a = np.ascontiguousarray(a)
    if a.dtype != _IN[variant]:
        raise TypeError(f"variant {variant} wants {_IN[variant]}, got {a.dtype}")
    return a


def _out(shape, variant):
    return np.empty(shape, dtype=_OUT[variant])


# ---------------------------------------------------------------- geometry
def site_index(dims, x) -> int:
    return int(lib().orc_site_index(_dims(dims), _dims(x)))


def site_coords(dims, s):
    x = (C.c_int * 4)()
    lib().orc_site_coords(_dims(dims), C.c_long(int(s)), x)
    return tuple(x)


def neighbor_table(dims, sign, mu):
    out = np.empty(_vol(dims), dtype=np.int32)
    lib().orc_neighbor_table(_dims(dims), C.c_int(sign), C.c_int(mu), _p(out))
    return out


# ---------------------------------------------------------------- shift
def shift(dims, f, sign, mu):
    f = np.ascontiguousarray(f)
    v = _vol(dims)
    nreal = f.size // v
    out = np.empty_like(f)
    fn = {np.dtype(np.float32): lib().orc_shift_f32, np.dtype(np.float64): lib().orc_shift_f64}[f.dtype]
    fn(_dims(dims), C.c_int(nreal), _p(f), _p(out), C.c_int(sign), C.c_int(mu))
    return out


# ---------------------------------------------------------------- catalogue
def mm_plus_madj(dims, a, b, c, d, variant):
    a, b, c, d = (_inp(t, variant) for t in (a, b, c, d))
    r = _out(a.shape, variant)
    getattr(lib(), f"orc_mm_plus_madj_{variant}")(_dims(dims), _p(a), _p(b), _p(c), _p(d), _p(r))
    return r


def trace_mm(dims, a, b, variant):
    a, b = _inp(a, variant), _inp(b, variant)
    r = _out((_vol(dims), 2), variant)
    getattr(lib(), f"orc_trace_mm_{variant}")(_dims(dims), _p(a), _p(b), _p(r))
    return r


def ax_minus_shift(dims, alpha, a, b, sign, mu, variant):
    a, b = _inp(a, variant), _inp(b, variant)
    r = _out(a.shape, variant)
    getattr(lib(), f"orc_ax_minus_shift_{variant}")(_dims(dims), C.c_double(alpha), _p(a), _p(b),
                                                     C.c_int(sign), C.c_int(mu), _p(r))
    return r


def _nspin(v, dims):
    ncx = v.size // (_vol(dims) * 2)
    if ncx not in (3, 12):
        raise ValueError("vector operand must be a colour vector (3) or fermion (12)")
    return ncx // 3


def mat_vec(dims, m, v, variant):
    m, v = _inp(m, variant), _inp(v, variant)
    w = _out(v.shape, variant)
    getattr(lib(), f"orc_mat_vec_{variant}")(_dims(dims), C.c_int(_nspin(v, dims)), _p(m), _p(v), _p(w))
    return w


def axpy(dims, s0, kappa, h, variant):
    s0, h = _inp(s0, variant), _inp(h, variant)
    r = _out(s0.shape, variant)
    ncx = s0.size // (_vol(dims) * 2)
    getattr(lib(), f"orc_axpy_{variant}")(_dims(dims), C.c_int(ncx), _p(s0), C.c_double(kappa), _p(h), _p(r))
    return r


def scale(dims, sc, a, variant):
    a = _inp(a, variant)
    r = _out(a.shape, variant)
    ncx = a.size // (_vol(dims) * 2)
    getattr(lib(), f"orc_scale_{variant}")(_dims(dims), C.c_int(ncx), C.c_double(sc), _p(a), _p(r))
    return r


def divide(dims, nrm, a, variant):
    a = _inp(a, variant)
    r = _out(a.shape, variant)
    ncx = a.size // (_vol(dims) * 2)
    getattr(lib(), f"orc_divide_{variant}")(_dims(dims), C.c_int(ncx), C.c_double(nrm), _p(a), _p(r))
    return r


def hop(dims, u, psi, variant, listing_form=False):
    u = [_inp(t, variant) for t in u]
    psi = _inp(psi, variant)
    chi = _out(psi.shape, variant)
    name = "orc_hop_listing_" if listing_form else "orc_hop_"
    getattr(lib(), name + variant)(_dims(dims), C.c_int(_nspin(psi, dims)), _p(u[0]), _p(u[1]), _p(u[2]),
                                   _p(u[3]), _p(psi), _p(chi))
    return chi


def jacobi_smear(dims, u, chi, kappa, iters, no_smear_dir, norm, variant):
    """Listing 1 of the paper, step by step: power series in kappa of the hopping term
    applied to chi, divided by norm.  no_smear_dir outside 0..3 smears in all four directions."""
    u = [_inp(t, variant) for t in u]
    chi = _inp(chi, variant)
    out = _out(chi.shape, variant)
    getattr(lib(), f"orc_jacobi_smear_{variant}")(_dims(dims), C.c_int(_nspin(chi, dims)), _p(u[0]), _p(u[1]), _p(u[2]),
                                                  _p(u[3]), _p(chi), C.c_double(kappa), C.c_int(iters),
                                                  C.c_int(no_smear_dir), C.c_double(norm), _p(out))
    return out


# ---------------------------------------------------------------- generic expressions (NEXT-2)
X_LEAF, X_ADJ, X_MUL, X_ADD, X_SUB, X_SCALE, X_SHIFT, X_TRACE = range(8)


def eval_expr(dims, nodes, leaves):
    """Plain per-site evaluation of a QDP++-style expression given in postfix order (the whole
    expression per site; :101: shift reads its operand at the periodic neighbour; Listing 1 operators * + -
    adj shift).  nodes: sequence of (op, a, b, s) with the operator codes above;
    leaves: QDP-order real arrays [V, ..., 2].  Arithmetic in complex128 (the truth for both precisions);
    returns a QDP-order float64 array.  A shift of a sub-expression is the sub-expression's field gathered
    through the oracle's neighbour table: shift(e, sign, mu)(x) = e(x + sign*mu^)."""
    stack = []
    for (op, a, b, s) in nodes:
        if op == X_LEAF:
            f = np.asarray(leaves[a], dtype=np.float64)
            stack.append(f[..., 0] + 1j * f[..., 1])
        elif op == X_ADJ:
            m = stack.pop()
            stack.append(np.conj(np.swapaxes(m, -1, -2)))
        elif op == X_MUL:
            r, l = stack.pop(), stack.pop()
            if r.ndim == 3 and r.shape[1:] == (3, 3):
                stack.append(np.einsum("xik,xkj->xij", l, r))
            elif r.ndim == 2:
                stack.append(np.einsum("xij,xj->xi", l, r))
            else:
                stack.append(np.einsum("xij,xaj->xai", l, r))
        elif op == X_ADD:
            r, l = stack.pop(), stack.pop()
            stack.append(l + r)
        elif op == X_SUB:
            r, l = stack.pop(), stack.pop()
            stack.append(l - r)
        elif op == X_SCALE:
            stack.append(float(s) * stack.pop())
        elif op == X_SHIFT:
            stack.append(stack.pop()[neighbor_table(dims, int(a), int(b))])
        elif op == X_TRACE:
            m = stack.pop()
            stack.append(m[:, 0, 0] + m[:, 1, 1] + m[:, 2, 2])
        else:
            raise ValueError(f"unknown operator {op}")
    if len(stack) != 1:
        raise ValueError("the postfix sequence does not reduce to one value")
    z = stack[0]
    return np.ascontiguousarray(np.stack((z.real, z.imag), axis=-1))


# ---------------------------------------------------------------- reductions
def sum_field(dims, f, variant):
    f = _inp(f, variant)
    ncx = f.size // (_vol(dims) * 2)
    out = np.empty(2 * ncx, dtype=np.float64)
    getattr(lib(), f"orc_sum_{variant}")(_dims(dims), C.c_int(ncx), _p(f), _p(out))
    return out.reshape(f.shape[1:])


def norm2(dims, f, variant) -> float:
    f = _inp(f, variant)
    ncx = f.size // (_vol(dims) * 2)
    return float(getattr(lib(), f"orc_norm2_{variant}")(_dims(dims), C.c_int(ncx), _p(f)))


def trace(dims, m, variant):
    m = _inp(m, variant)
    out = np.empty(2, dtype=np.float64)
    getattr(lib(), f"orc_trace_{variant}")(_dims(dims), _p(m), _p(out))
    return out


def plaquette_sum(dims, u, variant) -> float:
    u = [_inp(t, variant) for t in u]
    return float(getattr(lib(), f"orc_plaquette_sum_{variant}")(_dims(dims), _p(u[0]), _p(u[1]), _p(u[2]), _p(u[3])))


def plaquette_avg(dims, u, variant) -> float:
    return plaquette_sum(dims, u, variant) / (18.0 * _vol(dims))


def plaquette_sites(dims, u, sites, variant):
    u = [_inp(t, variant) for t in u]
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty(sites.size, dtype=np.float64)
    getattr(lib(), f"orc_plaquette_sites_{variant}")(_dims(dims), _p(u[0]), _p(u[1]), _p(u[2]), _p(u[3]),
                                                     C.c_long(sites.size), _p(sites), _p(out))
    return out


# ---------------------------------------------------------------- staple / smear
def staple_sum(dims, u, mu, variant):
    u = [_inp(t, variant) for t in u]
    out = _out(u[0].shape, variant)
    getattr(lib(), f"orc_staple_sum_{variant}")(_dims(dims), _p(u[0]), _p(u[1]), _p(u[2]), _p(u[3]),
                                                C.c_int(mu), _p(out))
    return out


def smear_step(dims, u, alpha, variant):
    u = [_inp(t, variant) for t in u]
    r = [_out(u[0].shape, variant) for _ in range(4)]
    getattr(lib(), f"orc_smear_step_{variant}")(_dims(dims), _p(u[0]), _p(u[1]), _p(u[2]), _p(u[3]),
                                                C.c_double(alpha), _p(r[0]), _p(r[1]), _p(r[2]), _p(r[3]))
    return r


def smear_links(dims, u, alpha, sites, mus, variant):
    u = [_inp(t, variant) for t in u]
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    mus = np.ascontiguousarray(mus, dtype=np.int32)
    out = _out((sites.size, 3, 3, 2), variant)
    getattr(lib(), f"orc_smear_links_{variant}")(_dims(dims), _p(u[0]), _p(u[1]), _p(u[2]), _p(u[3]),
                                                 C.c_double(alpha), C.c_long(sites.size), _p(sites), _p(mus), _p(out))
    return out


def smear_iterate(dims, u, alpha, nsteps, prec):
    """Truth trajectory (reading A23): step 1 from the storage-precision start with wide
    arithmetic, later steps stay in fp64 (no rounding back to the storage precision).
    Returns (list of link fields after the last step, [plaquette_avg after each step])."""
    variant = truth_variant(prec)
    plaqs = []
    for _ in range(nsteps):
        u = smear_step(dims, u, alpha, variant)
        variant = "t64" if prec == "f64" else "n64"
        plaqs.append(plaquette_avg(dims, u, variant))
    return u, plaqs
