"""paper_1105_2279_b200 -- thin Python binding of the lqx C-ABI library (include/lqx.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of liblqx.so.
The raw layer mirrors the C names without the `lqx_` prefix (`init`, `field_alloc`, `smear_step`,
...) and raises `LqxError` on a non-zero status.  `Lattice` / `Field` are small conveniences on
top (torch supplies device memory and the stream; numpy/torch arrays in QDP order go in and out).

There is no CPU fallback: if liblqx.so cannot be loaded or built, importing this package raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

F32, F64 = 4, 8
COMPLEX, COLORVEC, COLORMAT, FERMION = 1, 3, 9, 12
BACKWARD, FORWARD = -1, +1
K_SMEAR, K_PLAQUETTE, K_HOP, K_CATALOGUE, K_REDUCE = range(5)
KIND_SHAPE = {COMPLEX: (), COLORVEC: (3,), COLORMAT: (3, 3), FERMION: (4, 3)}
_NP = {F32: np.float32, F64: np.float64}


class TuneRow(C.Structure):
    _fields_ = [("kernel_class", C.c_int), ("prec", C.c_int), ("param", C.c_int * 2), ("ms", C.c_double), ("chosen", C.c_int)]


class LqxError(RuntimeError):
    def __init__(self, code, detail=""):
        self.code = int(code)
        msg = _lib.lqx_strerror(int(code)).decode()
        super().__init__(f"lqx status {code} ({msg})" + (f": {detail}" if detail else ""))


def _load():
    path = _build.LIB
    if not os.path.exists(path) or _build._stale(path, [os.path.join(_build.CSRC, s) for s in _build.SOURCES] + _build.HEADERS):
        try:
            path = _build.build()
        except Exception as e:
            # never run kernels that do not match the sources under review without saying so: a stale library is
            # loaded only on explicit request (LQX_ALLOW_STALE=1), and then loudly
            if not os.path.exists(_build.LIB):
                raise ImportError(f"liblqx.so is missing and could not be built: {e}") from e
            if os.environ.get("LQX_ALLOW_STALE") != "1":
                raise ImportError(f"liblqx.so is older than csrc/ and could not be rebuilt ({e}); "
                                  "set LQX_ALLOW_STALE=1 to load it anyway") from e
            import time
            import warnings

            warnings.warn("loading a STALE liblqx.so (built %s) although csrc/ is newer: %s"
                          % (time.ctime(os.path.getmtime(_build.LIB)), e))
            path = _build.LIB
    return C.CDLL(path)


_lib = _load()
_vp, _i, _d, _i64 = C.c_void_p, C.c_int, C.c_double, C.c_int64
_pvp = C.POINTER(C.c_void_p)
_pd = C.POINTER(C.c_double)

# name -> (restype, argtypes); every symbol include/lqx.h declares
SIGNATURES = {
    "lqx_init": (_i, [C.POINTER(C.c_int), _i, _vp, _pvp]),
    "lqx_finalize": (_i, [_vp]),
    "lqx_set_stream": (_i, [_vp, _vp]),
    "lqx_volume": (_i64, [_vp]),
    "lqx_padded_volume": (_i64, [_vp]),
    "lqx_field_offset": (_i64, [_vp, _i, _i, _i64, _i]),
    "lqx_field_bytes": (_i64, [_vp, _i, _i]),
    "lqx_neighbor_table": (_i, [_vp, _i, _i, _vp]),
    "lqx_field_alloc": (_i, [_vp, _i, _i, _pvp]),
    "lqx_field_attach": (_i, [_vp, _i, _i, _vp, C.c_size_t, _pvp]),
    "lqx_field_free": (_i, [_vp]),
    "lqx_field_data": (_vp, [_vp]),
    "lqx_field_kind": (_i, [_vp]),
    "lqx_field_prec": (_i, [_vp]),
    "lqx_field_push": (_i, [_vp, _vp]),
    "lqx_field_pop": (_i, [_vp, _vp]),
    "lqx_field_import_dev": (_i, [_vp, _vp]),
    "lqx_field_export_dev": (_i, [_vp, _vp]),
    "lqx_copy": (_i, [_vp, _vp]),
    "lqx_shift": (_i, [_vp, _vp, _i, _i]),
    "lqx_mm_plus_madj": (_i, [_vp, _vp, _vp, _vp, _vp]),
    "lqx_trace_mm": (_i, [_vp, _vp, _vp]),
    "lqx_ax_minus_shift": (_i, [_vp, _d, _vp, _vp, _i, _i]),
    "lqx_mat_vec": (_i, [_vp, _vp, _vp]),
    "lqx_hop": (_i, [_vp, _pvp, _vp]),
    "lqx_hop_norm2": (_i, [_vp, _pvp, _vp, _pd]),
    "lqx_jacobi_smear": (_i, [_vp, _pvp, _d, _i, _i, _d, _pvp]),
    "lqx_expr_eval": (_i, [_vp, _i, _vp, _i, _pvp, _i]),
    "lqx_expr_reduce": (_i, [_i, _vp, _i, _pvp, _i, _pd, C.POINTER(C.c_int)]),
    "lqx_expr_source": (_i, [_vp, _i, _i, _i, _vp, _i, C.POINTER(C.c_int), _i, C.c_char_p, C.c_size_t]),
    "lqx_expr_cache_size": (_i, [_vp]),
    "lqx_axpy": (_i, [_vp, _vp, _d, _vp]),
    "lqx_scale": (_i, [_vp, _d, _vp]),
    "lqx_divide": (_i, [_vp, _vp, _d]),
    "lqx_sum": (_i, [_vp, _pd]),
    "lqx_norm2": (_i, [_vp, _pd]),
    "lqx_norm2_noalloc": (_i, [_vp, _vp]),
    "lqx_trace": (_i, [_vp, _pd]),
    "lqx_plaquette": (_i, [_pvp, _pd, _pd]),
    "lqx_staple_sum": (_i, [_vp, _pvp, _i]),
    "lqx_smear_step": (_i, [_pvp, _pvp, _d, _pd]),
    "lqx_smear_iterate": (_i, [_pvp, _pvp, _d, _i, _pd]),
    "lqx_smear_iterate_host": (_i, [_vp, _i, _pvp, _pvp, _d, _i, _pd]),
    "lqx_bench_fma_peak": (_i, [_vp, _i, _pd]),
    "lqx_bench_copy_peak": (_i, [_vp, C.c_size_t, _pd]),
    "lqx_kernel_time": (_i, [_vp, _i, _pd, C.POINTER(C.c_int)]),
    "lqx_launch_count": (_i64, [_vp]),
    "lqx_smear_step_range": (_i, [_pvp, _pvp, _d, _i, _i]),
    "lqx_plaquette_range": (_i, [_pvp, _i, _i, _pd]),
    "lqx_field_slice": (_i, [_vp, _i, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]),
    "lqx_smear_info": (_i, [_vp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.c_char_p, _i]),
    "lqx_autotune": (_i, [_vp, _i, _i, _i, _vp, _i, C.POINTER(C.c_int)]),
    "lqx_tuned": (_i, [_vp, _i, _i, C.POINTER(C.c_int)]),
    "lqx_set_option": (_i, [_vp, C.c_char_p, _i]),
    "lqx_strerror": (C.c_char_p, [_i]),
    "lqx_last_error": (C.c_char_p, [_vp]),
    "lqx_version": (C.c_char_p, []),
}
for _name, (_res, _args) in SIGNATURES.items():
    _fn = getattr(_lib, _name)
    _fn.restype = _res
    _fn.argtypes = _args


def library_path() -> str:
    return _lib._name


def version() -> str:
    return _lib.lqx_version().decode()


def _check(rc, ctx=None):
    if rc != 0:
        detail = _lib.lqx_last_error(ctx).decode() if ctx else ""
        raise LqxError(rc, detail)


def _h(f):
    return f.handle if isinstance(f, Field) else f


def _arr4(fields):
    return (C.c_void_p * 4)(*[_h(f) for f in fields])


def _ctx_of(f):
    return f.lat.ctx if isinstance(f, Field) else None


# ------------------------------------------------------------------------------------------------
# conveniences
# ------------------------------------------------------------------------------------------------
class Lattice:
    """A context (lqx_init) bound to a CUDA device and to torch's current stream."""

    def __init__(self, dims, device: int = 0, stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("lqx needs a CUDA device (there is no CPU fallback)")
        self.dims = tuple(int(d) for d in dims)
        self.device = int(device)
        torch.cuda.set_device(self.device)
        torch.cuda.init()
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        out = C.c_void_p()
        _check(_lib.lqx_init((C.c_int * 4)(*self.dims), self.device, C.c_void_p(stream.cuda_stream), C.byref(out)))
        self.ctx = out
        self.volume = int(_lib.lqx_volume(self.ctx))
        self.padded_volume = int(_lib.lqx_padded_volume(self.ctx))
        self._fields = []

    def close(self):
        if self.ctx:
            for f in self._fields:
                f.handle = None
                f._mem = None
            _check(_lib.lqx_finalize(self.ctx))
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def field_bytes(self, kind, prec) -> int:
        return int(_lib.lqx_field_bytes(self.ctx, kind, prec))

    def field_offset(self, kind, prec, site: int, real_index: int) -> int:
        """Element offset of (site, QDP-order real index) in the internal blocked-SoA layout."""
        r = int(_lib.lqx_field_offset(self.ctx, kind, prec, int(site), int(real_index)))
        if r < 0:
            raise LqxError(r)
        return r

    def alloc(self, kind, prec, torch_memory: bool = True) -> "Field":
        """New zero field.  torch_memory=True: a torch uint8 tensor owns the bytes and the library
        borrows them (lqx_field_attach); False: the library allocates (lqx_field_alloc)."""
        out = C.c_void_p()
        mem = None
        if torch_memory:
            import torch

            nbytes = self.field_bytes(kind, prec)
            with torch.cuda.stream(self.stream):
                mem = torch.zeros(nbytes, dtype=torch.uint8, device=f"cuda:{self.device}")
            _check(_lib.lqx_field_attach(self.ctx, kind, prec, C.c_void_p(mem.data_ptr()), nbytes, C.byref(out)), self.ctx)
        else:
            _check(_lib.lqx_field_alloc(self.ctx, kind, prec, C.byref(out)), self.ctx)
        f = Field(self, out, kind, prec, mem)
        self._fields.append(f)
        return f

    def from_host(self, array, kind=None) -> "Field":
        """Push a QDP-order host array ([V, *shape, 2], float32/float64, numpy or torch CPU)."""
        a = _as_numpy(array)
        if kind is None:
            kind = {(): COMPLEX, (3,): COLORVEC, (3, 3): COLORMAT, (4, 3): FERMION}[tuple(a.shape[1:-1])]
        prec = {np.dtype(np.float32): F32, np.dtype(np.float64): F64}[a.dtype]
        f = self.alloc(kind, prec)
        f.push(a)
        return f

    def neighbor_table(self, direction, mu):
        out = np.empty(self.volume, dtype=np.int32)
        _check(_lib.lqx_neighbor_table(self.ctx, direction, mu, out.ctypes.data_as(C.c_void_p)), self.ctx)
        return out

    def set_stream(self, stream):
        """lqx_set_stream: later calls are enqueued on `stream` (a torch.cuda.Stream); the old one is synchronised
        first.  With a non-default stream the asynchronous calls can be captured into a CUDA graph."""
        _check(_lib.lqx_set_stream(self.ctx, C.c_void_p(stream.cuda_stream)), self.ctx)
        self.stream = stream

    def set_option(self, key: str, value: int):
        _check(_lib.lqx_set_option(self.ctx, key.encode(), int(value)), self.ctx)

    def kernel_time(self, kernel_class: int):
        """-> (total_ms, count) of one kernel class since the last read (needs set_option('time_kernels', 1))."""
        ms, n = C.c_double(), C.c_int()
        _check(_lib.lqx_kernel_time(self.ctx, kernel_class, C.byref(ms), C.byref(n)), self.ctx)
        return ms.value, n.value

    def expr_cache_size(self) -> int:
        return int(_lib.lqx_expr_cache_size(self.ctx))

    def smear_info(self):
        """(variant, FMA lane-ops per site, kernel name) of the last smear launch."""
        v, n = C.c_int(), C.c_int()
        name = C.create_string_buffer(64)
        _check(_lib.lqx_smear_info(self.ctx, C.byref(v), C.byref(n), name, 64), self.ctx)
        return v.value, n.value, name.value.decode()

    def autotune(self, kernel_class, prec, reps=5):
        """Time every launch geometry of a kernel class on this lattice, keep the fastest; returns the table rows."""
        rows = (TuneRow * 64)()
        n = C.c_int()
        _check(_lib.lqx_autotune(self.ctx, kernel_class, prec, reps, C.cast(rows, C.c_void_p), 64, C.byref(n)), self.ctx)
        return [{"kernel_class": r.kernel_class, "prec": r.prec, "param": [r.param[0], r.param[1]], "ms": r.ms, "chosen": bool(r.chosen)}
                for r in rows[:min(n.value, 64)]]

    def tuned(self, kernel_class, prec):
        out = (C.c_int * 4)()
        _check(_lib.lqx_tuned(self.ctx, kernel_class, prec, out), self.ctx)
        return list(out)

    def launch_count(self) -> int:
        return int(_lib.lqx_launch_count(self.ctx))

    def bench_fma_peak(self, kind: int) -> float:
        out = C.c_double()
        _check(_lib.lqx_bench_fma_peak(self.ctx, kind, C.byref(out)), self.ctx)
        return out.value

    def bench_copy_peak(self, nbytes: int) -> float:
        out = C.c_double()
        _check(_lib.lqx_bench_copy_peak(self.ctx, nbytes, C.byref(out)), self.ctx)
        return out.value


def _as_numpy(array):
    if hasattr(array, "detach"):
        array = array.detach().cpu().numpy()
    return np.ascontiguousarray(array)


class Field:
    def __init__(self, lat, handle, kind, prec, mem=None):
        self.lat, self.handle, self.kind, self.prec, self._mem = lat, handle, kind, prec, mem

    @property
    def host_shape(self):
        return (self.lat.volume,) + KIND_SHAPE[self.kind] + (2,)

    def push(self, array):
        a = _as_numpy(array)
        if a.dtype != _NP[self.prec] or a.size != int(np.prod(self.host_shape)):
            raise TypeError(f"push wants {_NP[self.prec].__name__} with {self.host_shape}, got {a.dtype} {a.shape}")
        _check(_lib.lqx_field_push(self.handle, a.ctypes.data_as(C.c_void_p)), self.lat.ctx)
        return self

    def pop(self):
        out = np.empty(self.host_shape, dtype=_NP[self.prec])
        _check(_lib.lqx_field_pop(self.handle, out.ctypes.data_as(C.c_void_p)), self.lat.ctx)
        return out

    def slice_bytes(self, t):
        """(offset, nbytes) of time slice t inside this field's device storage (lqx_field_slice)."""
        off, n = C.c_int64(), C.c_int64()
        _check(_lib.lqx_field_slice(self.handle, int(t), C.byref(off), C.byref(n)), self.lat.ctx)
        return off.value, n.value

    def slice_view(self, t):
        """Time slice t of the device storage as a torch uint8 view (torch-owned fields only): what a halo
        exchange sends and receives."""
        if self._mem is None:
            raise ValueError("slice_view needs a field whose memory torch owns (Lattice.alloc(torch_memory=True))")
        off, n = self.slice_bytes(t)
        return self._mem[off:off + n]

    def import_dev(self, dev_tensor):
        """AoS QDP-order torch CUDA tensor -> this field (device to device)."""
        _check(_lib.lqx_field_import_dev(self.handle, C.c_void_p(dev_tensor.data_ptr())), self.lat.ctx)
        return self

    def export_dev(self, dev_tensor):
        _check(_lib.lqx_field_export_dev(self.handle, C.c_void_p(dev_tensor.data_ptr())), self.lat.ctx)
        return dev_tensor

    def free(self):
        if self.handle:
            _check(_lib.lqx_field_free(self.handle), self.lat.ctx)
            self.handle = None
            self._mem = None
            if self in self.lat._fields:
                self.lat._fields.remove(self)


# ------------------------------------------------------------------------------------------------
# raw layer: the C names without the prefix
# ------------------------------------------------------------------------------------------------
def copy(r, a):
    _check(_lib.lqx_copy(_h(r), _h(a)), _ctx_of(r))


def shift(r, a, direction, mu):
    _check(_lib.lqx_shift(_h(r), _h(a), direction, mu), _ctx_of(r))


def mm_plus_madj(r, a, b, c, d):
    _check(_lib.lqx_mm_plus_madj(_h(r), _h(a), _h(b), _h(c), _h(d)), _ctx_of(r))


def trace_mm(c, a, b):
    _check(_lib.lqx_trace_mm(_h(c), _h(a), _h(b)), _ctx_of(c))


def ax_minus_shift(r, alpha, a, b, direction, mu):
    _check(_lib.lqx_ax_minus_shift(_h(r), float(alpha), _h(a), _h(b), direction, mu), _ctx_of(r))


def mat_vec(w, m, v):
    _check(_lib.lqx_mat_vec(_h(w), _h(m), _h(v)), _ctx_of(w))


def hop(chi, u, psi):
    _check(_lib.lqx_hop(_h(chi), _arr4(u), _h(psi)), _ctx_of(chi))


def hop_norm2(chi, u, psi) -> float:
    out = C.c_double()
    _check(_lib.lqx_hop_norm2(_h(chi), _arr4(u), _h(psi), C.byref(out)), _ctx_of(chi))
    return out.value


def jacobi_smear(chi, u, kappa, iters, no_smear_dir, norm, tmp):
    """chi <- sum_{n<=iters} kappa^n H^n chi / norm (Listing 1 of the paper); tmp = two scratch fields."""
    arr = (C.c_void_p * 2)(_h(tmp[0]), _h(tmp[1]))
    _check(_lib.lqx_jacobi_smear(_h(chi), _arr4(u), float(kappa), int(iters), int(no_smear_dir), float(norm), arr), _ctx_of(chi))


# ---- run-time expression fusion: a tiny builder for the flattened postfix tree of lqx_expr_eval
X_LEAF, X_ADJ, X_MUL, X_ADD, X_SUB, X_SCALE, X_SHIFT, X_TRACE = range(8)
R_NORM2, R_SUM = 1, 2


class _XNode(C.Structure):
    _fields_ = [("op", C.c_int32), ("a", C.c_int32), ("b", C.c_int32), ("s", C.c_double)]


class Expr:
    """Expression over fields with the paper's operators: `*`, `+`, `-`, real `scalar * e`, adj(e),
    shift(e, direction, mu).  Leaves are Field objects (or, for expr_source, bare kind codes)."""

    def __init__(self, nodes, leaves):
        self.nodes, self.leaves = nodes, leaves  # nodes: list of (op, a, b, s); leaves: list of fields

    @staticmethod
    def leaf(field):
        return Expr([(X_LEAF, 0, 0, 0.0)], [field])

    def _merge(self, other):
        """Postfix of other re-indexed onto this expression's leaf list (identical fields share a slot)."""
        leaves = list(self.leaves)
        remap = {}
        for i, f in enumerate(other.leaves):
            for j, g in enumerate(leaves):
                if g is f:
                    remap[i] = j
                    break
            else:
                remap[i] = len(leaves)
                leaves.append(f)
        nodes = [(op, remap[a] if op == X_LEAF else a, b, s) for (op, a, b, s) in other.nodes]
        return nodes, leaves

    def _binary(self, other, op):
        if not isinstance(other, Expr):
            other = Expr.leaf(other)
        nodes, leaves = self._merge(other)
        return Expr(self.nodes + nodes + [(op, 0, 0, 0.0)], leaves)

    def __mul__(self, other):
        if isinstance(other, (int, float)):
            return Expr(self.nodes + [(X_SCALE, 0, 0, float(other))], self.leaves)
        return self._binary(other, X_MUL)

    def __rmul__(self, other):
        return Expr(self.nodes + [(X_SCALE, 0, 0, float(other))], self.leaves)

    def __add__(self, other):
        return self._binary(other, X_ADD)

    def __sub__(self, other):
        return self._binary(other, X_SUB)

    def adj(self):
        return Expr(self.nodes + [(X_ADJ, 0, 0, 0.0)], self.leaves)

    def shift(self, direction, mu):
        return Expr(self.nodes + [(X_SHIFT, int(direction), int(mu), 0.0)], self.leaves)

    def trace(self):
        return Expr(self.nodes + [(X_TRACE, 0, 0, 0.0)], self.leaves)

    def _c_nodes(self):
        arr = (_XNode * len(self.nodes))()
        for i, (op, a, b, s) in enumerate(self.nodes):
            arr[i].op, arr[i].a, arr[i].b, arr[i].s = op, a, b, s
        return arr


def adj(e):
    return (e if isinstance(e, Expr) else Expr.leaf(e)).adj()


def shifted(e, direction, mu):
    return (e if isinstance(e, Expr) else Expr.leaf(e)).shift(direction, mu)


def expr_eval(dst, expr, accumulate=False):
    """dst = expr (or dst += expr): one fused kernel, NVRTC-compiled on first use and cached."""
    leaves = (C.c_void_p * max(1, len(expr.leaves)))(*[_h(f) for f in expr.leaves])
    _check(_lib.lqx_expr_eval(_h(dst), 1 if accumulate else 0, expr._c_nodes(), len(expr.nodes), leaves, len(expr.leaves)),
           _ctx_of(dst))


def expr_reduce(what, expr):
    """norm2 (what = R_NORM2 -> float) or sum (R_SUM -> array of 2*kind doubles, QDP order) of an expression,
    evaluated and reduced in one generated kernel."""
    leaves = (C.c_void_p * len(expr.leaves))(*[_h(f) for f in expr.leaves])
    out = (C.c_double * 24)()
    n = C.c_int()
    _check(_lib.lqx_expr_reduce(int(what), expr._c_nodes(), len(expr.nodes), leaves, len(expr.leaves), out, C.byref(n)),
           _ctx_of(expr.leaves[0]))
    return out[0] if what == R_NORM2 else np.array(out[: n.value])


def expr_source(lat, dst_kind, prec, expr, accumulate=False, reduce=0) -> str:
    """The CUDA source generated for expr; leaves may be Field objects or kind codes."""
    kinds = (C.c_int * max(1, len(expr.leaves)))(*[f.kind if isinstance(f, Field) else int(f) for f in expr.leaves])
    buf = C.create_string_buffer(1 << 16)
    n = _lib.lqx_expr_source(lat.ctx if isinstance(lat, Lattice) else lat, dst_kind, prec, (1 + reduce) if reduce else (1 if accumulate else 0), expr._c_nodes(),
                             len(expr.nodes), kinds, len(expr.leaves), buf, len(buf))
    if n < 0:
        raise LqxError(n, _lib.lqx_last_error(lat.ctx if isinstance(lat, Lattice) else lat).decode())
    return buf.value.decode()


def axpy(r, s0, kappa, h):
    _check(_lib.lqx_axpy(_h(r), _h(s0), float(kappa), _h(h)), _ctx_of(r))


def scale(r, s, a):
    _check(_lib.lqx_scale(_h(r), float(s), _h(a)), _ctx_of(r))


def divide(r, a, nrm):
    _check(_lib.lqx_divide(_h(r), _h(a), float(nrm)), _ctx_of(r))


def sum(f):  # noqa: A001 - mirrors the C name
    n = 2 * f.kind
    out = (C.c_double * n)()
    _check(_lib.lqx_sum(_h(f), out), _ctx_of(f))
    return np.array(out[:], dtype=np.float64).reshape(KIND_SHAPE[f.kind] + (2,))


def norm2(f) -> float:
    out = C.c_double()
    _check(_lib.lqx_norm2(_h(f), C.byref(out)), _ctx_of(f))
    return out.value


NOALLOC_MAX_SITES = 1 << 24  # include/lqx.h LQX_NOALLOC_MAX_SITES


def norm2_noalloc(f, out_dev_ptr: int) -> None:
    """lqx_norm2_noalloc: norm2(f) written to one double at DEVICE address `out_dev_ptr` (e.g. a torch float64
    tensor's data_ptr()); allocates nothing, asynchronous on the lattice's stream (include/lqx.h)."""
    _check(_lib.lqx_norm2_noalloc(_h(f), C.c_void_p(int(out_dev_ptr))), _ctx_of(f))


def trace(m):
    out = (C.c_double * 2)()
    _check(_lib.lqx_trace(_h(m), out), _ctx_of(m))
    return np.array(out[:], dtype=np.float64)


def plaquette(u):
    """-> (plaq_sum, plaq_avg)"""
    s, a = C.c_double(), C.c_double()
    _check(_lib.lqx_plaquette(_arr4(u), C.byref(s), C.byref(a)), _ctx_of(u[0]))
    return s.value, a.value


def staple_sum(out, u, mu):
    _check(_lib.lqx_staple_sum(_h(out), _arr4(u), mu), _ctx_of(out))


def smear_step(uout, uin, alpha, want_plaq_in: bool = False):
    """One smearing step; returns the plaquette SUM of the input field if want_plaq_in."""
    p = C.c_double()
    _check(_lib.lqx_smear_step(_arr4(uout), _arr4(uin), float(alpha), C.byref(p) if want_plaq_in else None), _ctx_of(uin[0]))
    return p.value if want_plaq_in else None


def smear_step_range(uout, uin, alpha, t0, t1):
    """The smear step of the time slices [t0, t1) only (asynchronous); see lqx_smear_step_range."""
    _check(_lib.lqx_smear_step_range(_arr4(uout), _arr4(uin), float(alpha), int(t0), int(t1)), _ctx_of(uin[0]))


def plaquette_range(u, t0, t1):
    """Plaquette SUM over the sites of the time slices [t0, t1)."""
    s = C.c_double()
    _check(_lib.lqx_plaquette_range(_arr4(u), int(t0), int(t1), C.byref(s)), _ctx_of(u[0]))
    return s.value


def smear_iterate(u, tmp, alpha, nsteps, want_plaq: bool = True):
    """nsteps steps in place (tmp = ping-pong scratch); returns plaquette averages after each step."""
    out = (C.c_double * max(1, nsteps))()
    _check(_lib.lqx_smear_iterate(_arr4(u), _arr4(tmp), float(alpha), int(nsteps), out if want_plaq else None), _ctx_of(u[0]))
    return list(out[:nsteps]) if want_plaq else None


def smear_iterate_host(lat: Lattice, prec, host_u_in, host_u_out, alpha, nsteps):
    """End-to-end call with HOST buffers in QDP order (numpy or pinned torch CPU tensors)."""
    def ptr(a):
        return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data

    pin = (C.c_void_p * 4)(*[ptr(a) for a in host_u_in])
    pout = (C.c_void_p * 4)(*[ptr(a) for a in host_u_out])
    out = (C.c_double * max(1, nsteps))()
    _check(_lib.lqx_smear_iterate_host(lat.ctx, prec, pin, pout, float(alpha), int(nsteps), out), lat.ctx)
    return list(out[:nsteps])
