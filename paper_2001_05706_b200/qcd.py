"""Thin ctypes binding of libqcd_b200.so (include/qcd.h) -- argument marshalling only.

Every function here has the name of the C entry point it calls (minus the ``qcd_``
prefix) and does nothing but turn torch tensors into device pointers and sizes.  All
arithmetic of the hot path runs in the CUDA kernels of the library; there is no CPU
fallback: if the library is missing or no CUDA device is present the calls raise.

PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqcd_b200.so")

OK, NOCONV, EINVAL, EALLOC, ECUDA, EBREAKDOWN = 0, 1, -1, -2, -3, -4
DAGGER = 1
PARITY_EVEN, PARITY_ODD, PARITY_FULL = 0, 1, 2


class QcdError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("qcd error %d: %s" % (code, text))
        self.code = code


class Stats(C.Structure):
    _fields_ = [("iters", C.c_int), ("reliable_updates", C.c_int), ("converged", C.c_int),
                ("breakdown", C.c_int), ("r_iter", C.c_double), ("r_true", C.c_double),
                ("seconds", C.c_double), ("flops", C.c_double), ("bytes", C.c_double)]


_lib = None
_vp, _i, _d, _sz = C.c_void_p, C.c_int, C.c_double, C.c_size_t
_dims_t = C.c_int * 4

# name -> (restype, argtypes); mirrors include/qcd.h one to one
SIGNATURES = {
    "qcd_last_error": (C.c_char_p, []),
    "qcd_version": (_i, []),
    "qcd_init": (_i, [_i, _vp, C.POINTER(_vp)]),
    "qcd_finalize": (_i, [_vp]),
    "qcd_gauge_bytes": (_sz, [_dims_t, _i, _i]),
    "qcd_gauge_load": (_i, [_vp, C.POINTER(_vp), _vp, _i, _vp, _dims_t, _i, _i, _i]),
    "qcd_gauge_free": (_i, [_vp]),
    "qcd_clover_bytes": (_sz, [_dims_t, _i]),
    "qcd_clover_build": (_i, [_vp, C.POINTER(_vp), _vp, _vp, _d, _d, _i]),
    "qcd_clover_free": (_i, [_vp]),
    "qcd_clover_unpack": (_i, [_vp, _vp, _vp, _i]),
    "qcd_spinor_bytes": (_sz, [_dims_t, _i]),
    "qcd_spinor_pack": (_i, [_vp, _vp, _vp, _dims_t, _i]),
    "qcd_spinor_unpack": (_i, [_vp, _vp, _vp, _dims_t, _i]),
    "qcd_convert": (_i, [_vp, _vp, _i, _vp, _i, _dims_t, _i]),
    "qcd_hop": (_i, [_vp, _vp, _vp, _i, _i, _dims_t, _i]),
    "qcd_hop_xpay": (_i, [_vp, _vp, _vp, _d, _d, _vp, _i, _i]),
    "qcd_dslash": (_i, [_vp, _vp, _vp, _vp, _d, _d, _i, _dims_t, _i]),
    "qcd_dslash_ex": (_i, [_vp, _vp, _vp, _vp, _d, _d, _i, _i, _vp]),
    "qcd_half_spinor_bytes": (_sz, [_dims_t]),
    "qcd_spinor_to_half": (_i, [_vp, _vp, _vp, _dims_t, _i]),
    "qcd_spinor_from_half": (_i, [_vp, _vp, _vp, _dims_t, _i]),
    "qcd_dslash_half": (_i, [_vp, _i, _vp, _vp, _vp, _d, _d, _i, _i, _vp]),
    "qcd_wilson_multi": (_i, [_vp, _vp, _vp, _i, _vp, _d, _i]),
    "qcd_dslash_host_batch": (_i, [_vp, _vp, _vp, _i, _sz, _sz, _vp, _vp, _d, _d, _i, _i]),
    "qcd_workspace_bytes": (_sz, [_dims_t, _i]),
    "qcd_set_workspace": (_i, [_vp, _vp, _sz]),
    "qcd_axpy": (_i, [_vp, _d, _vp, _vp, _sz, _i]),
    "qcd_xpay": (_i, [_vp, _vp, _d, _vp, _sz, _i]),
    "qcd_axpby": (_i, [_vp, _d, _vp, _d, _vp, _sz, _i]),
    "qcd_norm2": (_i, [_vp, _vp, _sz, _i, C.POINTER(_d)]),
    "qcd_redot": (_i, [_vp, _vp, _vp, _sz, _i, C.POINTER(_d)]),
    "qcd_cg_update": (_i, [_vp, _d, _vp, _vp, _vp, _vp, _sz, _i, C.POINTER(_d)]),
    "qcd_set_operator": (_i, [_vp, _vp, _vp, _vp, _vp, _d, _d, _i, _d]),
    "qcd_cg_solve": (_i, [_vp, _vp, _d, _i]),
    "qcd_cg_solve_ex": (_i, [_vp, _vp, _vp, _d, _i, C.POINTER(Stats)]),
    "qcd_cg_multishift": (_i, [_vp, _vp, _vp, C.POINTER(_d), _i, _d, _i, C.POINTER(Stats), C.POINTER(_d)]),
    "qcd_apply_operator": (_i, [_vp, _vp, _vp, _i]),
    "qcd_noalloc_max_bytes": (_sz, []),
    "qcd_noalloc_setup": (_i, [_i]),
    "qcd_norm2_noalloc": (_i, [_i, _vp, _vp, _sz, _i, _vp]),
    "qcd_eo_prepare": (_i, [_vp, _vp, _vp]),
    "qcd_eo_reconstruct": (_i, [_vp, _vp, _vp]),
    "qcd_clover_apply": (_i, [_vp, _vp, _vp, _vp, _i, _i]),
    "qcd_cheb_apply": (_i, [_vp, _vp, _vp, _vp, _d, C.POINTER(_d), _i, _d]),
    "qcd_cheb_apply_multi": (_i, [_vp, _vp, _vp, _i, _vp, _d, C.POINTER(_d), _i, _d]),
    "qcd_hop_host": (_i, [_vp, _vp, _vp, _vp, _i, _i]),
    "qcd_dslash_host": (_i, [_vp, _vp, _vp, _vp, _vp, _d, _d, _i, _i]),
    "qcd_launch_count": (C.c_longlong, [_vp]),
}


def lib():
    """Load libqcd_b200.so; fails loudly when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s is missing: run `python -m paper_2001_05706_b200.build` "
                              "(there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _check(rc, soft=False):
    if rc < 0 or (rc > 0 and not soft):
        raise QcdError(rc, lib().qcd_last_error().decode())
    return rc


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        assert t.is_contiguous()
        return C.c_void_p(t.data_ptr())
    return C.c_void_p(int(t))


def _prec(t: torch.Tensor) -> int:
    return {torch.float32: 4, torch.float64: 8}[t.dtype]


def _dtype(precision: int):
    return {4: torch.float32, 8: torch.float64}[precision]


def noalloc_max_bytes() -> int:
    return int(lib().qcd_noalloc_max_bytes())


def noalloc_setup(device: int = 0):
    _check(lib().qcd_noalloc_setup(device))


def norm2_noalloc(x: torch.Tensor, result_dev: torch.Tensor, nreal=None, device: int = 0, stream=None):
    """result_dev[0] = |x|^2 on `stream` (default: torch's current stream); no ctx, nothing allocated."""
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    _check(lib().qcd_norm2_noalloc(device, C.c_void_p(st), _ptr(x), x.numel() if nreal is None else int(nreal), _prec(x), _ptr(result_dev)))


def _dims(dims):
    return _dims_t(*[int(d) for d in dims])


class Context:
    """qcd_ctx bound to a device and (by default) torch's current stream on it."""

    def __init__(self, device: int = 0, stream=None):
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: libqcd_b200 has no CPU fallback")
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = _vp()
        _check(lib().qcd_init(device, C.c_void_p(self.stream.cuda_stream), C.byref(h)))
        self.h = h
        self._ws = None

    def close(self):
        if self.h:
            lib().qcd_finalize(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def empty(self, nbytes: int) -> torch.Tensor:
        return torch.empty(max(int(nbytes), 16), dtype=torch.uint8, device=self.device)

    # ---- workspace -------------------------------------------------------------
    def workspace_bytes(self, dims, precision) -> int:
        return int(lib().qcd_workspace_bytes(_dims(dims), precision))

    def set_workspace(self, ws: torch.Tensor | None):
        self._ws = ws
        if ws is None:
            _check(lib().qcd_set_workspace(self.h, None, 0))
        else:
            _check(lib().qcd_set_workspace(self.h, _ptr(ws), ws.numel() * ws.element_size()))

    def ensure_workspace(self, nbytes: int):
        if self._ws is None or self._ws.numel() * self._ws.element_size() < nbytes:
            self.set_workspace(self.empty(nbytes))

    # ---- fields ------------------------------------------------------------------
    def gauge_load(self, links: torch.Tensor, dims, precision: int, reconstruct: int, t_boundary: int = -1):
        """links: device tensor, boundary layout [T][Z][Y][X][4][3][3][2]."""
        storage = self.empty(lib().qcd_gauge_bytes(_dims(dims), precision, reconstruct))
        g = _vp()
        _check(lib().qcd_gauge_load(self.h, C.byref(g), _ptr(links), _prec(links), _ptr(storage), _dims(dims),
                                    precision, reconstruct, t_boundary))
        return Gauge(g, storage, tuple(int(d) for d in dims), precision, reconstruct)

    def clover_build(self, gauge: "Gauge", kappa: float, csw: float, precision: int):
        storage = self.empty(lib().qcd_clover_bytes(_dims(gauge.dims), precision))
        c = _vp()
        _check(lib().qcd_clover_build(self.h, C.byref(c), gauge.h, _ptr(storage), kappa, csw, precision))
        return Clover(c, storage, gauge.dims, precision, kappa, csw)

    def clover_unpack(self, clover: "Clover", which: int) -> torch.Tensor:
        X, Y, Z, T = clover.dims
        out = torch.empty((T, Z, Y, X, 12, 12, 2), dtype=torch.float64, device=self.device)
        _check(lib().qcd_clover_unpack(self.h, _ptr(out), clover.h, which))
        return out

    def spinor_pack(self, boundary: torch.Tensor, dims) -> torch.Tensor:
        internal = torch.empty(boundary.numel(), dtype=boundary.dtype, device=self.device)
        _check(lib().qcd_spinor_pack(self.h, _ptr(internal), _ptr(boundary), _dims(dims), _prec(boundary)))
        return internal

    def spinor_unpack(self, internal: torch.Tensor, dims) -> torch.Tensor:
        X, Y, Z, T = (int(d) for d in dims)
        boundary = torch.empty((T, Z, Y, X, 4, 3, 2), dtype=internal.dtype, device=self.device)
        _check(lib().qcd_spinor_unpack(self.h, _ptr(boundary), _ptr(internal), _dims(dims), _prec(internal)))
        return boundary

    def convert(self, src: torch.Tensor, precision: int, dims, nblocks: int) -> torch.Tensor:
        dst = torch.empty(src.numel(), dtype=_dtype(precision), device=self.device)
        _check(lib().qcd_convert(self.h, _ptr(dst), precision, _ptr(src), _prec(src), _dims(dims), nblocks))
        return dst

    # ---- stencil -------------------------------------------------------------------
    def hop(self, out, inp, gauge: "Gauge", out_parity: int, dagger: bool = False):
        _check(lib().qcd_hop(_ptr(out), _ptr(inp), gauge.h, out_parity, int(dagger), _dims(gauge.dims), gauge.precision))

    def hop_xpay(self, out, inp, z, a: float, b: float, gauge: "Gauge", out_parity: int, dagger: bool = False):
        _check(lib().qcd_hop_xpay(_ptr(out), _ptr(inp), _ptr(z), a, b, gauge.h, out_parity, int(dagger)))

    def dslash(self, out, inp, gauge: "Gauge", clover, kappa: float, csw: float, parity: int):
        _check(lib().qcd_dslash(_ptr(out), _ptr(inp), gauge.h, clover.h if clover else None, kappa, csw, parity,
                                _dims(gauge.dims), gauge.precision))

    def dslash_ex(self, out, inp, gauge: "Gauge", clover, kappa: float, csw: float, parity: int, flags: int = 0, tmp=None):
        _check(lib().qcd_dslash_ex(_ptr(out), _ptr(inp), gauge.h, clover.h if clover else None, kappa, csw, parity,
                                   flags, _ptr(tmp)))

    # ---- 16-bit storage ---------------------------------------------------------------
    def spinor_to_half(self, f32: torch.Tensor, dims, nblocks: int) -> torch.Tensor:
        half = self.empty(lib().qcd_half_spinor_bytes(_dims(dims)) // 2 * nblocks)
        _check(lib().qcd_spinor_to_half(self.h, _ptr(half), _ptr(f32), _dims(dims), nblocks))
        return half

    def spinor_from_half(self, half: torch.Tensor, dims, nblocks: int) -> torch.Tensor:
        X, Y, Z, T = (int(d) for d in dims)
        f32 = torch.empty(nblocks * (X * Y * Z * T // 2) * 24, dtype=torch.float32, device=self.device)
        _check(lib().qcd_spinor_from_half(self.h, _ptr(f32), _ptr(half), _dims(dims), nblocks))
        return f32

    def dslash_half(self, out, out_precision: int, in_half, gauge: "Gauge", clover, kappa: float, csw: float, parity: int,
                    flags: int = 0, tmp_half=None):
        _check(lib().qcd_dslash_half(_ptr(out), out_precision, _ptr(in_half), gauge.h, clover.h if clover else None,
                                     kappa, csw, parity, flags, _ptr(tmp_half)))

    def hop_host(self, out_host, in_host, gauge: "Gauge", out_parity: int, dagger: bool = False):
        """out_host / in_host: pinned (or pageable) HOST tensors, one-parity internal blocks."""
        _check(lib().qcd_hop_host(self.h, _ptr(out_host), _ptr(in_host), gauge.h, out_parity, int(dagger)))

    def dslash_host(self, out_host, in_host, gauge: "Gauge", clover, kappa: float, csw: float, parity: int, flags: int = 0):
        _check(lib().qcd_dslash_host(self.h, _ptr(out_host), _ptr(in_host), gauge.h, clover.h if clover else None,
                                     kappa, csw, parity, flags))

    def wilson_multi(self, out, inp, nvec: int, gauge: "Gauge", kappa: float, gamma5: bool = False):
        _check(lib().qcd_wilson_multi(self.h, _ptr(out), _ptr(inp), nvec, gauge.h, kappa, int(gamma5)))

    def dslash_host_batch(self, out_host, in_host, nvec: int, gauge: "Gauge", clover, kappa: float, csw: float,
                          parity: int, flags: int = 0, out_stride=None, in_stride=None):
        """nvec vectors held consecutively in (pinned) HOST tensors, pipelined H2D / operator / D2H."""
        es = out_host.element_size()
        ostr = out_host.numel() // max(nvec, 1) * es if out_stride is None else out_stride
        istr = in_host.numel() // max(nvec, 1) * es if in_stride is None else in_stride
        _check(lib().qcd_dslash_host_batch(self.h, _ptr(out_host), _ptr(in_host), nvec, ostr, istr, gauge.h,
                                           clover.h if clover else None, kappa, csw, parity, flags))

    # ---- BLAS ------------------------------------------------------------------------
    def axpy(self, a, x, y):
        _check(lib().qcd_axpy(self.h, a, _ptr(x), _ptr(y), x.numel(), _prec(x)))

    def xpay(self, x, a, y):
        _check(lib().qcd_xpay(self.h, _ptr(x), a, _ptr(y), x.numel(), _prec(x)))

    def axpby(self, a, x, b, y):
        _check(lib().qcd_axpby(self.h, a, _ptr(x), b, _ptr(y), x.numel(), _prec(x)))

    def norm2(self, x, fetch: bool = True):
        r = _d()
        _check(lib().qcd_norm2(self.h, _ptr(x), x.numel(), _prec(x), C.byref(r) if fetch else None))
        return r.value if fetch else None

    def redot(self, x, y, fetch: bool = True):
        r = _d()
        _check(lib().qcd_redot(self.h, _ptr(x), _ptr(y), x.numel(), _prec(x), C.byref(r) if fetch else None))
        return r.value if fetch else None

    def cg_update(self, a, p, q, x, r, fetch: bool = True):
        res = _d()
        _check(lib().qcd_cg_update(self.h, a, _ptr(p), _ptr(q), _ptr(x), _ptr(r), x.numel(), _prec(x),
                                   C.byref(res) if fetch else None))
        return res.value if fetch else None

    # ---- solvers -----------------------------------------------------------------------
    def set_operator(self, g_hi, g_lo=None, c_hi=None, c_lo=None, kappa=0.0, csw=0.0, parity=2, delta=0.1):
        self._op = (g_hi, g_lo, c_hi, c_lo)  # keep the handles alive
        _check(lib().qcd_set_operator(self.h, g_hi.h, g_lo.h if g_lo else None, c_hi.h if c_hi else None,
                                      c_lo.h if c_lo else None, kappa, csw, parity, delta))

    def apply_operator(self, out, inp, flags: int = 0):
        _check(lib().qcd_apply_operator(self.h, _ptr(out), _ptr(inp), flags))

    def eo_prepare(self, bhat, b):
        _check(lib().qcd_eo_prepare(self.h, _ptr(bhat), _ptr(b)))

    def eo_reconstruct(self, x, b):
        _check(lib().qcd_eo_reconstruct(self.h, _ptr(x), _ptr(b)))

    def clover_apply(self, out, inp, clover, inverse: bool, parity: int):
        _check(lib().qcd_clover_apply(self.h, _ptr(out), _ptr(inp), clover.h, int(bool(inverse)), parity))

    def cg_solve(self, x, b, tol: float, maxiter: int):
        """Returns (return code, Stats). QCD_NOCONV (1) is returned, not raised."""
        st = Stats()
        rc = _check(lib().qcd_cg_solve_ex(self.h, _ptr(x), _ptr(b), tol, maxiter, C.byref(st)), soft=True)
        return rc, st

    def cg_multishift(self, x, b, shifts, tol: float, maxiter: int):
        """x: len(shifts) consecutive fields.  Returns (return code, Stats, [r_true_i])."""
        ns = len(shifts)
        sh = (_d * ns)(*[float(v) for v in shifts])
        rt = (_d * ns)()
        st = Stats()
        rc = _check(lib().qcd_cg_multishift(self.h, _ptr(x), _ptr(b), sh, ns, tol, maxiter, C.byref(st), rt), soft=True)
        return rc, st, [rt[i] for i in range(ns)]

    def cheb_apply(self, y, v, gauge: "Gauge", kappa: float, coeff, scale: float):
        n = len(coeff)
        arr = (_d * n)(*[float(c) for c in coeff])
        _check(lib().qcd_cheb_apply(self.h, _ptr(y), _ptr(v), gauge.h, kappa, arr, n - 1, scale))

    def cheb_apply_multi(self, y, v, nvec: int, gauge: "Gauge", kappa: float, coeff, scale: float):
        """y, v: nvec consecutive full internal fields."""
        n = len(coeff)
        arr = (_d * n)(*[float(c) for c in coeff])
        _check(lib().qcd_cheb_apply_multi(self.h, _ptr(y), _ptr(v), nvec, gauge.h, kappa, arr, n - 1, scale))

    def launch_count(self) -> int:
        return int(lib().qcd_launch_count(self.h))


class Gauge:
    def __init__(self, h, storage, dims, precision, reconstruct):
        self.h, self.storage, self.dims, self.precision, self.reconstruct = h, storage, dims, precision, reconstruct

    def __del__(self):
        try:
            if self.h:
                lib().qcd_gauge_free(self.h)
                self.h = None
        except Exception:
            pass


class Clover:
    def __init__(self, h, storage, dims, precision, kappa, csw):
        self.h, self.storage, self.dims, self.precision, self.kappa, self.csw = h, storage, dims, precision, kappa, csw

    def __del__(self):
        try:
            if self.h:
                lib().qcd_clover_free(self.h)
                self.h = None
        except Exception:
            pass
