"""ctypes loader for the CPU oracle (oracle/qcd_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  Nothing under
paper_2001_05706_b200/ imports this module, and this module imports nothing
from the CUDA path.

All fields are numpy float64 arrays in the boundary layout
  gauge  [T][Z][Y][X][4][3][3][2]      spinor [T][Z][Y][X][4][3][2]
``dims`` is (X, Y, Z, T).  Arithmetic is done in C (fp64, OpenMP over sites).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = [os.path.join(_HERE, "qcd_oracle.c"), os.path.join(_HERE, "qcd_oracle_impl.h")]
_lib = None


def build(force: bool = False) -> str:
    """Compile liboracle.so with gcc (idempotent)."""
    stale = force or not os.path.exists(_SO) or any(
        os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if stale:
        cmd = ["gcc", "-O2", "-fopenmp", "-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", _SO, _SRC[0], "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_invert_12.restype = C.c_int
        for n in ("orc_apply_M", "orc_cg", "orc_cg_mixed", "orc_cheb", "orc_cg_multishift", "orc_apply_M_q16",
                  "orc_apply_N_q16"):
            getattr(_lib, n).restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def _dims(dims):
    return (C.c_int * 4)(*[int(d) for d in dims])


def _vol(dims):
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def _spinor_like(dims):
    X, Y, Z, T = (int(d) for d in dims)
    return np.empty((T, Z, Y, X, 4, 3, 2), dtype=np.float64)


def gamma_matrices() -> np.ndarray:
    """complex [5][4][4]: gamma_x, gamma_y, gamma_z, gamma_t, gamma_5."""
    out = np.empty((5, 4, 4, 2), dtype=np.float64)
    lib().orc_get_gamma(_p(out))
    return out.view(np.complex128)[..., 0]


def sigma_matrices() -> np.ndarray:
    """complex [6][4][4]: sigma_munu for planes (01,02,03,12,13,23)."""
    out = np.empty((6, 4, 4, 2), dtype=np.float64)
    lib().orc_get_sigma(_p(out))
    return out.view(np.complex128)[..., 0]


def hop(psi, U, dims, tb=-1, dagger=False, parity_mask=2) -> np.ndarray:
    """(H psi)(x) of the north_star formula on the full lattice (or one parity)."""
    psi = _f64(psi); U = _f64(U)
    out = _spinor_like(dims)
    lib().orc_hop(_p(out), _p(psi), _p(U), _dims(dims), C.c_int(tb), C.c_int(int(dagger)),
                  C.c_int(parity_mask))
    return out


def hop_sites(psi, U, dims, sites, tb=-1, dagger=False) -> np.ndarray:
    """(H psi) at lexicographic sites ``sites`` only -> [n][4][3][2]."""
    psi = _f64(psi); U = _f64(U)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((len(sites), 4, 3, 2), dtype=np.float64)
    lib().orc_hop_sites(_p(out), _p(psi), _p(U), _dims(dims), C.c_int(tb), C.c_int(int(dagger)),
                        _p(sites), C.c_long(len(sites)))
    return out


def field_strength(U, dims) -> np.ndarray:
    """Fhat_munu(x), float64 [T][Z][Y][X][6][3][3][2], planes (01,02,03,12,13,23)."""
    U = _f64(U)
    X, Y, Z, T = (int(d) for d in dims)
    F = np.empty((T, Z, Y, X, 6, 3, 3, 2), dtype=np.float64)
    lib().orc_field_strength(_p(F), _p(U), _dims(dims))
    return F


def field_strength_sites(U, dims, sites) -> np.ndarray:
    U = _f64(U)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    F = np.empty((len(sites), 6, 3, 3, 2), dtype=np.float64)
    lib().orc_field_strength_sites(_p(F), _p(U), _dims(dims), _p(sites), C.c_long(len(sites)))
    return F


def clover_matrix(F, dims, coeff, add_unit=True) -> np.ndarray:
    """A(x) = 1 + coeff * sum_{mu<nu} i sigma_munu (x) Fhat_munu(x), float64
    [T][Z][Y][X][12][12][2], index = spin*3 + colour.  ``F`` may also be a
    [n][6][3][3][2] list of sites (then dims = (n,1,1,1))."""
    F = _f64(F)
    n = F.size // (6 * 9 * 2)
    A = np.empty(F.shape[:-4] + (12, 12, 2), dtype=np.float64)
    lib().orc_clover_matrix(_p(A), _p(F), _dims((n, 1, 1, 1)), C.c_double(coeff),
                            C.c_int(int(add_unit)))
    return A


def invert_12(A) -> np.ndarray:
    A = _f64(A)
    n = A.size // (144 * 2)
    Ainv = np.empty_like(A)
    bad = lib().orc_invert_12(_p(Ainv), _p(A), C.c_long(n))
    if bad:
        raise np.linalg.LinAlgError(f"{bad} singular clover blocks")
    return Ainv


def site_matrix_apply(M, psi, dims, parity_mask=2) -> np.ndarray:
    psi = _f64(psi)
    out = _spinor_like(dims)
    lib().orc_site_matrix_apply(_p(out), None if M is None else _p(_f64(M)), _p(psi), _dims(dims),
                                C.c_int(parity_mask))
    return out


def apply_M(psi, U, dims, kappa, A=None, Ainv=None, tb=-1, mode=2, dagger=False) -> np.ndarray:
    """mode 2: (A - kappa H) psi on the full lattice (A = 1 if None).
    mode p in {0,1}: even-odd Schur operator on parity p (psi must vanish on 1-p)."""
    psi = _f64(psi); U = _f64(U)
    out = _spinor_like(dims)
    rc = lib().orc_apply_M(_p(out), _p(psi), _p(U), None if A is None else _p(_f64(A)),
                           None if Ainv is None else _p(_f64(Ainv)), _dims(dims), C.c_double(kappa),
                           C.c_int(tb), C.c_int(mode), C.c_int(int(dagger)))
    if rc:
        raise MemoryError
    return out


def cg(b, U, dims, kappa, tol, maxiter, A=None, Ainv=None, tb=-1, mode=2):
    """CG on M^dag M x = b (reading O6). Returns (x, stats dict)."""
    b = _f64(b); U = _f64(U)
    x = _spinor_like(dims)
    st = np.zeros(8, dtype=np.float64)
    rc = lib().orc_cg(_p(x), _p(b), _p(U), None if A is None else _p(_f64(A)),
                      None if Ainv is None else _p(_f64(Ainv)), _dims(dims), C.c_double(kappa),
                      C.c_int(tb), C.c_int(mode), C.c_double(tol), C.c_int(maxiter), _p(st))
    if rc:
        raise MemoryError
    return x, dict(iters=int(st[0]), r_iter=st[1], r_true=st[2], converged=bool(st[3]),
                   breakdown=bool(st[4]))


def q16_codes(v):
    """(int16 codes [n][24], fp32 norms [n]) of the 16-bit spinor format (reading H1)."""
    v = np.ascontiguousarray(v, dtype=np.float32).reshape(-1, 24)
    codes = np.empty(v.shape, dtype=np.int16)
    norms = np.empty(len(v), dtype=np.float32)
    lib().orc_q16_codes(_p(v), _p(codes), _p(norms), C.c_long(len(v)))
    return codes, norms


def q16_spinor(v):
    """Spinor stored in 16 bits and read back (fp32 array, same shape)."""
    out = np.array(v, dtype=np.float32, order="C")
    lib().orc_q16_spinor(_p(out), C.c_long(out.size // 24))
    return out


def q16_links(U):
    out = np.array(U, dtype=np.float32, order="C")
    lib().orc_q16_links(_p(out), C.c_long(out.size // 18))
    return out


def q16_clover(A):
    out = np.array(A, dtype=np.float32, order="C")
    lib().orc_q16_clover(_p(out), C.c_long(out.size // 288))
    return out


def apply_M_q16(psi_q, Uq, dims, kappa, Aq=None, Ainvq=None, tb=-1, mode=2, dagger=False, store_out=False):
    """M (or M^dag) with 16-bit storage of links, clover and the even-odd intermediate; psi_q,
    Uq, Aq, Ainvq are stored-and-read-back fp32 fields (q16_*).  Returns fp32."""
    psi_q = np.ascontiguousarray(psi_q, dtype=np.float32)
    out = np.empty_like(psi_q)
    rc = lib().orc_apply_M_q16(_p(out), _p(psi_q), _p(np.ascontiguousarray(Uq, dtype=np.float32)),
                               None if Aq is None else _p(np.ascontiguousarray(Aq, dtype=np.float32)),
                               None if Ainvq is None else _p(np.ascontiguousarray(Ainvq, dtype=np.float32)),
                               _dims(dims), C.c_double(kappa), C.c_int(tb), C.c_int(mode), C.c_int(int(dagger)),
                               C.c_int(int(store_out)))
    if rc:
        raise MemoryError
    return out


def apply_N_q16(p, Uq, dims, kappa, Aq=None, Ainvq=None, tb=-1, mode=2):
    """q = M^dag store(M store(p)) with every streamed field in 16 bits; q in fp32."""
    p = np.ascontiguousarray(p, dtype=np.float32)
    out = np.empty_like(p)
    rc = lib().orc_apply_N_q16(_p(out), _p(p), _p(np.ascontiguousarray(Uq, dtype=np.float32)),
                               None if Aq is None else _p(np.ascontiguousarray(Aq, dtype=np.float32)),
                               None if Ainvq is None else _p(np.ascontiguousarray(Ainvq, dtype=np.float32)),
                               _dims(dims), C.c_double(kappa), C.c_int(tb), C.c_int(mode))
    if rc:
        raise MemoryError
    return out


def cg_mixed(b, U, dims, kappa, tol, maxiter, A=None, Ainv=None, tb=-1, mode=2, delta=0.1, half=False):
    """Reliable-update fp32/fp64 CG (reading O7).  The fp32 operator uses the
    fp64 fields rounded to fp32 (reading S15); with half=True the inner operator streams
    16-bit fields (reading H1): links, clover and spinors stored in 16 bits."""
    b = _f64(b); U = _f64(U)
    Ulo = np.ascontiguousarray(U, dtype=np.float32)
    Alo = None if A is None else np.ascontiguousarray(A, dtype=np.float32)
    Ailo = None if Ainv is None else np.ascontiguousarray(Ainv, dtype=np.float32)
    if half:
        Ulo = q16_links(Ulo)
        Alo = None if Alo is None else q16_clover(Alo)
        Ailo = None if Ailo is None else q16_clover(Ailo)
    y = _spinor_like(dims)
    st = np.zeros(8, dtype=np.float64)
    upd = np.zeros(256, dtype=np.int32)
    rc = lib().orc_cg_mixed(_p(y), _p(b), _p(U), None if A is None else _p(_f64(A)),
                            None if Ainv is None else _p(_f64(Ainv)), _p(Ulo),
                            None if Alo is None else _p(Alo), None if Ailo is None else _p(Ailo),
                            _dims(dims), C.c_double(kappa), C.c_int(tb), C.c_int(mode),
                            C.c_double(tol), C.c_int(maxiter), C.c_double(delta), C.c_int(int(half)), _p(st),
                            _p(upd), C.c_int(len(upd)))
    if rc:
        raise MemoryError
    return y, dict(iters=int(st[0]), r_iter=st[1], r_true=st[2], converged=bool(st[3]),
                   breakdown=bool(st[4]), reliable_updates=int(st[5]),
                   update_at=[int(k) for k in upd[:min(int(st[5]), len(upd))]])


def cg_multishift(b, U, dims, kappa, shifts, tol, maxiter, A=None, Ainv=None, tb=-1, mode=2):
    """Multi-shift CG: (M^dag M + shifts[i]) x_i = b with one N apply per iteration
    (SURVEY.md 8(f).3).  shifts ascending, >= 0.  Returns ([x_i], stats dict)."""
    b = _f64(b); U = _f64(U)
    sh = np.ascontiguousarray(shifts, dtype=np.float64)
    ns = len(sh)
    X, Y, Z, T = (int(d) for d in dims)
    x = np.empty((ns, T, Z, Y, X, 4, 3, 2), dtype=np.float64)
    st = np.zeros(8, dtype=np.float64)
    rt = np.zeros(ns, dtype=np.float64)
    rc = lib().orc_cg_multishift(_p(x), _p(b), _p(U), None if A is None else _p(_f64(A)),
                                 None if Ainv is None else _p(_f64(Ainv)), _dims(dims), C.c_double(kappa),
                                 C.c_int(tb), C.c_int(mode), _p(sh), C.c_int(ns), C.c_double(tol),
                                 C.c_int(maxiter), _p(st), _p(rt))
    if rc:
        raise MemoryError
    return [x[i] for i in range(ns)], dict(iters=int(st[0]), r_iter=st[1], converged=bool(st[3]),
                                           breakdown=bool(st[4]), r_true=rt.copy())


def apply_HW(psi, U, dims, kappa, tb=-1) -> np.ndarray:
    """H_W psi = gamma5 (1 - kappa H) psi."""
    psi = _f64(psi); U = _f64(U)
    out = _spinor_like(dims)
    lib().orc_apply_HW(_p(out), _p(psi), _p(U), _dims(dims), C.c_double(kappa), C.c_int(tb))
    return out


def cheb(v, U, dims, kappa, coeff, scale, tb=-1) -> np.ndarray:
    """y = sum_k coeff[k] T_k(H_W/scale) v by the forward recurrence (reading O8)."""
    v = _f64(v); U = _f64(U)
    coeff = np.ascontiguousarray(coeff, dtype=np.float64)
    y = _spinor_like(dims)
    rc = lib().orc_cheb(_p(y), _p(v), _p(U), _dims(dims), C.c_double(kappa), C.c_int(tb), _p(coeff),
                        C.c_int(len(coeff) - 1), C.c_double(scale))
    if rc:
        raise MemoryError
    return y


# ---- even-odd helpers written from the definitions (reading O5) -------------
def parity_mask_array(dims) -> np.ndarray:
    """[T][Z][Y][X] array of (x+y+z+t) & 1."""
    X, Y, Z, T = (int(d) for d in dims)
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    return (x + y + z + t) & 1


def eo_prepare_source(b, U, dims, kappa, Ainv, tb=-1, p=0):
    """bhat_p = b_p + kappa H_{p,pbar} A^{-1}_{pbar,pbar} b_pbar (zero on pbar)."""
    par = parity_mask_array(dims)
    b = _f64(b)
    b_pb = b * (par == 1 - p)[..., None, None, None]
    t = site_matrix_apply(Ainv, b_pb, dims, 1 - p)
    t = hop(t, U, dims, tb, False, p)
    return b * (par == p)[..., None, None, None] + kappa * t


def eo_reconstruct(x_p, b, U, dims, kappa, Ainv, tb=-1, p=0):
    """x_pbar = A^{-1}_{pbar,pbar} (b_pbar + kappa H_{pbar,p} x_p); returns the full x."""
    par = parity_mask_array(dims)
    b = _f64(b)
    t = hop(x_p, U, dims, tb, False, 1 - p)
    t = b * (par == 1 - p)[..., None, None, None] + kappa * t
    x_pb = site_matrix_apply(Ainv, t, dims, 1 - p)
    return _f64(x_p) + x_pb
