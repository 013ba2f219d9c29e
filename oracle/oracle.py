"""numpy/ctypes front end of oracle/cola_oracle.c -- TEST INFRASTRUCTURE, not the product.

Argument marshalling only; all arithmetic is in the C file.  Arrays are numpy complex128 in the
canonical layouts of SURVEY.md §8(c) O1:  U[t][z][y][x][mu][3][3], psi[t][z][y][x][4][3],
A[t][z][y][x][12][12].  `dims` = (Lx, Ly, Lz, Lt); `bc` = (+1|-1) per direction.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cola_oracle.c")
_LIB = os.path.join(_HERE, "libcola_oracle.so")

__all__ = [
    "build", "gamma", "sigma", "hop", "dslash_parity", "field_strength", "clover", "clover_inverse",
    "block_apply", "M", "schur", "eo_prepare", "eo_reconstruct", "apply_sites", "cgnr", "cgnr_mixed", "bicgstab", "lowest_modes",
    "dense_inverse", "num_threads", "parity_mask",
]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP on the site loops)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call([
            "gcc", "-O2", "-fopenmp", "-fcx-limited-range", "-shared", "-fPIC",
            "-o", _LIB, _SRC, "-lm",
        ])
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_clover_inverse.restype = ctypes.c_int
        _lib.oracle_dense_inverse.restype = ctypes.c_int
        _lib.oracle_cgnr.restype = ctypes.c_int
        _lib.oracle_cgnr_mixed.restype = ctypes.c_int
        _lib.oracle_bicgstab.restype = ctypes.c_int
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _c(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.complex128)


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _i4(v):
    return (ctypes.c_int * 4)(*[int(x) for x in v])


def _shape(dims):
    lx, ly, lz, lt = dims
    return (lt, lz, ly, lx)


def _vol(dims):
    lx, ly, lz, lt = dims
    return lx * ly * lz * lt


def num_threads() -> int:
    return int(_L().oracle_num_threads())


def gamma() -> np.ndarray:
    out = np.zeros((5, 4, 4), dtype=np.complex128)
    _L().oracle_gamma(_p(out))
    return out


def sigma() -> np.ndarray:
    out = np.zeros((4, 4, 4, 4), dtype=np.complex128)
    _L().oracle_sigma(_p(out))
    return out


def parity_mask(dims) -> np.ndarray:
    """[t][z][y][x] array of (x+y+z+t) mod 2 (index bookkeeping for tests)."""
    lx, ly, lz, lt = dims
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    return (x + y + z + t) & 1


def hop(dims, bc, U, psi) -> np.ndarray:
    U, psi = _c(U), _c(psi)
    out = np.empty_like(psi)
    _L().oracle_hop(_i4(dims), _i4(bc), _p(U), _p(psi), _p(out))
    return out


def dslash_parity(dims, bc, U, out_parity: int, psi) -> np.ndarray:
    U, psi = _c(U), _c(psi)
    out = np.empty_like(psi)
    _L().oracle_dslash_parity(_i4(dims), _i4(bc), _p(U), ctypes.c_int(out_parity), _p(psi), _p(out))
    return out


def field_strength(dims, U, trace_sub: bool = True) -> np.ndarray:
    U = _c(U)
    out = np.empty(_shape(dims) + (6, 3, 3), dtype=np.complex128)
    _L().oracle_field_strength(_i4(dims), _p(U), ctypes.c_int(int(trace_sub)), _p(out))
    return out


def clover(dims, U, kappa: float, csw: float, trace_sub: bool = True) -> np.ndarray:
    U = _c(U)
    out = np.empty(_shape(dims) + (12, 12), dtype=np.complex128)
    _L().oracle_clover(_i4(dims), _p(U), ctypes.c_double(kappa), ctypes.c_double(csw),
                       ctypes.c_int(int(trace_sub)), _p(out))
    return out


def clover_inverse(A) -> np.ndarray:
    A = _c(A)
    out = np.empty_like(A)
    n_sites = A.size // 144
    bad = _L().oracle_clover_inverse(ctypes.c_long(n_sites), _p(A), _p(out))
    if bad:
        raise ArithmeticError(f"{bad} singular clover blocks")
    return out


def dense_inverse(a) -> np.ndarray:
    a = _c(a)
    n = a.shape[0]
    out = np.empty_like(a)
    if _L().oracle_dense_inverse(ctypes.c_int(n), _p(a), _p(out)):
        raise ArithmeticError("singular matrix")
    return out


def block_apply(B, psi) -> np.ndarray:
    B, psi = _c(B), _c(psi)
    out = np.empty_like(psi)
    _L().oracle_block_apply(ctypes.c_long(psi.size // 12), _p(B), _p(psi), _p(out))
    return out


def M(dims, bc, U, A, kappa: float, psi, dagger: bool = False) -> np.ndarray:
    U, A, psi = _c(U), _c(A), _c(psi)
    out = np.empty_like(psi)
    _L().oracle_M(_i4(dims), _i4(bc), _p(U), _p(A), ctypes.c_double(kappa), ctypes.c_int(int(dagger)),
                  _p(psi), _p(out))
    return out


def schur(dims, bc, U, A, Ainv, kappa: float, x, dagger: bool = False) -> np.ndarray:
    U, A, Ainv, x = _c(U), _c(A), _c(Ainv), _c(x)
    out = np.empty_like(x)
    _L().oracle_schur(_i4(dims), _i4(bc), _p(U), _p(A), _p(Ainv), ctypes.c_double(kappa),
                      ctypes.c_int(int(dagger)), _p(x), _p(out))
    return out


def eo_prepare(dims, bc, U, Ainv, kappa: float, b) -> np.ndarray:
    U, Ainv, b = _c(U), _c(Ainv), _c(b)
    out = np.empty_like(b)
    _L().oracle_eo_prepare(_i4(dims), _i4(bc), _p(U), _p(Ainv), ctypes.c_double(kappa), _p(b), _p(out))
    return out


def eo_reconstruct(dims, bc, U, Ainv, kappa: float, b, x_even) -> np.ndarray:
    U, Ainv, b = _c(U), _c(Ainv), _c(b)
    x = _c(x_even).copy()
    _L().oracle_eo_reconstruct(_i4(dims), _i4(bc), _p(U), _p(Ainv), ctypes.c_double(kappa), _p(b), _p(x))
    return x


_WHICH = {"D": 0, "M": 1, "Mdag": 2, "S": 3, "Sdag": 4}


def apply_sites(dims, bc, U, kappa: float, csw: float, which: str, psi, sites, trace_sub: bool = True) -> np.ndarray:
    """(K psi)(x) at the lexicographic site indices `sites`; K in D, M, Mdag, S, Sdag (SURVEY O-L)."""
    U, psi = _c(U), _c(psi)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((sites.size, 4, 3), dtype=np.complex128)
    _L().oracle_apply_sites(_i4(dims), _i4(bc), _p(U), ctypes.c_double(kappa), ctypes.c_double(csw),
                            ctypes.c_int(int(trace_sub)), ctypes.c_int(_WHICH[which]), _p(psi),
                            ctypes.c_long(sites.size), sites.ctypes.data_as(ctypes.c_void_p), _p(out))
    return out


def cgnr(dims, bc, U, A, Ainv, kappa: float, b, even_odd: bool, tol: float = 1e-10, max_iter: int = 20000):
    """CGLS-form CGNR.  Returns dict(x, iters, converged, true_residual, history)."""
    U, A, b = _c(U), _c(A), _c(b)
    Ainv = _c(Ainv) if Ainv is not None else A
    x = np.zeros_like(b)
    iters = ctypes.c_int(0)
    true_res = ctypes.c_double(0.0)
    hist = np.zeros(max_iter, dtype=np.float64)
    st = _L().oracle_cgnr(_i4(dims), _i4(bc), _p(U), _p(A), _p(Ainv), ctypes.c_double(kappa),
                          ctypes.c_int(int(even_odd)), _p(b), _p(x), ctypes.c_double(tol),
                          ctypes.c_int(max_iter), ctypes.byref(iters), hist.ctypes.data_as(ctypes.c_void_p),
                          ctypes.byref(true_res))
    return dict(x=x, iters=iters.value, converged=(st == 0), true_residual=true_res.value,
                history=hist[: iters.value].copy())


def cgnr_mixed(dims, bc, U, A, Ainv, kappa: float, b, even_odd: bool, tol: float = 1e-10,
               delta: float = 0.1, max_iter: int = 20000):
    """Reliable-update mixed-precision CGLS model."""
    U, A, b = _c(U), _c(A), _c(b)
    Ainv = _c(Ainv) if Ainv is not None else A
    x = np.zeros_like(b)
    iters = ctypes.c_int(0)
    updates = ctypes.c_int(0)
    true_res = ctypes.c_double(0.0)
    hist = np.zeros(max_iter, dtype=np.float64)
    max_updates = 256
    upd = np.zeros(max_updates, dtype=np.int32)
    st = _L().oracle_cgnr_mixed(_i4(dims), _i4(bc), _p(U), _p(A), _p(Ainv), ctypes.c_double(kappa),
                                ctypes.c_int(int(even_odd)), _p(b), _p(x), ctypes.c_double(tol),
                                ctypes.c_double(delta), ctypes.c_int(max_iter), ctypes.byref(iters),
                                ctypes.byref(updates), ctypes.byref(true_res),
                                hist.ctypes.data_as(ctypes.c_void_p), upd.ctypes.data_as(ctypes.c_void_p),
                                ctypes.c_int(max_updates))
    return dict(x=x, iters=iters.value, updates=updates.value, converged=(st == 0),
                true_residual=true_res.value, history=hist[: iters.value].copy(),
                update_iters=[int(v) for v in upd[: min(updates.value, max_updates)]])


def bicgstab(dims, bc, U, A, Ainv, kappa: float, b, even_odd: bool, tol: float = 1e-10, max_iter: int = 20000):
    """BiCGStab in van der Vorst's order on M or on the Schur system.
    Returns dict(x, iters, converged, breakdown, true_residual, history); one iteration = two operator applications."""
    U, A, b = _c(U), _c(A), _c(b)
    Ainv = _c(Ainv) if Ainv is not None else A
    x = np.zeros_like(b)
    iters = ctypes.c_int(0)
    true_res = ctypes.c_double(0.0)
    hist = np.zeros(max_iter, dtype=np.float64)
    st = _L().oracle_bicgstab(_i4(dims), _i4(bc), _p(U), _p(A), _p(Ainv), ctypes.c_double(kappa),
                              ctypes.c_int(int(even_odd)), _p(b), _p(x), ctypes.c_double(tol),
                              ctypes.c_int(max_iter), ctypes.byref(iters), hist.ctypes.data_as(ctypes.c_void_p),
                              ctypes.byref(true_res))
    return dict(x=x, iters=iters.value, converged=(st == 0), breakdown=(st == 2), true_residual=true_res.value,
                history=hist[: iters.value].copy())


def lowest_modes(dims, bc, U, A, Ainv, kappa: float, k: int, dense_limit: int = 1600, tol: float = 1e-13):
    """The k smallest eigenvalues (ascending) and orthonormal eigenvectors of H = S^+ S on the even sites
    (the low modes the paper's "eigenmode solver" delivers, ref [1] P:65).

    It is the plain definition: for up to `dense_limit` even-site degrees of freedom the matrix of S is written out
    column by column with oracle.schur, H = S^+ S is formed and numpy's Hermitian eigen-solver is called; above that
    the library routine is scipy's ARPACK driver on a LinearOperator that applies oracle.schur twice.
    Returns (evals[k], evecs[k] + full-lattice spinor shape, zero on odd sites)."""
    shape = _shape(dims) + (4, 3)
    mask_e = np.broadcast_to((parity_mask(dims) == 0)[..., None, None], shape)
    idx = np.flatnonzero(mask_e.ravel())
    n = idx.size

    def S(xe, dagger=False):
        full = np.zeros(int(np.prod(shape)), dtype=np.complex128)
        full[idx] = xe
        return schur(dims, bc, U, A, Ainv, kappa, full.reshape(shape), dagger=dagger).ravel()[idx]

    if n <= dense_limit:
        Sd = np.empty((n, n), dtype=np.complex128)
        e = np.zeros(n, dtype=np.complex128)
        for j in range(n):
            e[j] = 1.0
            Sd[:, j] = S(e)
            e[j] = 0.0
        w, v = np.linalg.eigh(Sd.conj().T @ Sd)
        w, v = w[:k], v[:, :k]
    else:
        from scipy.sparse.linalg import LinearOperator, eigsh

        op = LinearOperator((n, n), matvec=lambda x: S(S(x), dagger=True), dtype=np.complex128)
        w, v = eigsh(op, k=k, which="SA", tol=tol, ncv=max(4 * k, 40), maxiter=20000)
        order = np.argsort(w)
        w, v = w[order], v[:, order]
    vecs = np.zeros((k, int(np.prod(shape))), dtype=np.complex128)
    vecs[:, idx] = v.T
    return w, vecs.reshape((k,) + shape)
