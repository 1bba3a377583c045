"""ctypes loader for the CPU oracle (oracle/gs_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may
import this package.  It imports nothing from paper_2502_02460_b200 and shares no code with the
CUDA path.  Each wrapper converts its inputs to column-major (Fortran-order) numpy arrays, calls the
plain-C routine, and returns new arrays; see gs_oracle.c for the passages each routine follows
(PAPER.md:61-67).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gs_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp, no -ffast-math, no BLAS."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        i64, p = ctypes.c_int64, ctypes.c_void_p
        for t in "dz":
            getattr(lib, f"orc_cholesky_{t}").argtypes = [i64, p]
            getattr(lib, f"orc_cholesky_{t}").restype = i64
            getattr(lib, f"orc_invert_upper_{t}").argtypes = [i64, p, p]
            getattr(lib, f"orc_invert_upper_{t}").restype = i64
            getattr(lib, f"orc_to_standard_{t}").argtypes = [i64, p, p, p, p]
            getattr(lib, f"orc_to_standard_{t}").restype = None
            getattr(lib, f"orc_backtransform_{t}").argtypes = [i64, i64, p, p, p]
            getattr(lib, f"orc_backtransform_{t}").restype = None
            getattr(lib, f"orc_jacobi_{t}").argtypes = [i64, p, p, p]
            getattr(lib, f"orc_jacobi_{t}").restype = i64
            getattr(lib, f"orc_density_{t}").argtypes = [i64, i64, p, p, p]
            getattr(lib, f"orc_density_{t}").restype = None
            for nm in ("hn", "nn"):
                getattr(lib, f"orc_matmul_{nm}_{t}").argtypes = [i64, i64, i64, p, p, p]
                getattr(lib, f"orc_matmul_{nm}_{t}").restype = None
            getattr(lib, f"orc_inertia_{t}").argtypes = [i64, p, ctypes.c_double]
            getattr(lib, f"orc_inertia_{t}").restype = i64
        lib.orc_sturm_count.argtypes = [i64, p, p, ctypes.c_double]
        lib.orc_sturm_count.restype = i64
        lib.orc_tridiag_eigenvalue.argtypes = [i64, p, p, i64]
        lib.orc_tridiag_eigenvalue.restype = ctypes.c_double
        lib.orc_tridiag_eigenvalues.argtypes = [i64, p, p, i64, p]
        lib.orc_tridiag_eigenvalues.restype = None
        lib.orc_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().orc_num_threads())


def _f(a, dtype=None) -> np.ndarray:
    a = np.asarray(a)
    if dtype is None:
        dtype = np.complex128 if np.iscomplexobj(a) else np.float64
    return np.array(a, dtype=dtype, order="F", copy=True)


def _sfx(a: np.ndarray) -> str:
    return "z" if a.dtype == np.complex128 else "d"


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


class NotPositiveDefinite(Exception):
    def __init__(self, info: int):
        super().__init__(f"pivot {info} is not positive")
        self.info = info


def cholesky(S) -> np.ndarray:
    """O1: S = U^H U, returns U (upper, zeros below).  Raises NotPositiveDefinite(info)."""
    U = _f(S)
    N = U.shape[0]
    assert U.shape == (N, N)
    info = getattr(_load(), f"orc_cholesky_{_sfx(U)}")(N, _ptr(U))
    if info != 0:
        raise NotPositiveDefinite(int(info))
    return U


def invert_upper(U) -> np.ndarray:
    """O2: V = U^-1 by back substitution (reads the upper triangle of U only)."""
    U = _f(U)
    N = U.shape[0]
    V = np.zeros_like(U, order="F")
    info = getattr(_load(), f"orc_invert_upper_{_sfx(U)}")(N, _ptr(U), _ptr(V))
    if info != 0:
        raise ZeroDivisionError(f"U({info},{info}) == 0")
    return V


def to_standard(H, V) -> np.ndarray:
    """O3: H~ = V^H H V, FULL matrix (both triangles computed independently)."""
    H = _f(H)
    V = _f(V, H.dtype)
    N = H.shape[0]
    W = np.zeros_like(H, order="F")
    Ht = np.zeros_like(H, order="F")
    getattr(_load(), f"orc_to_standard_{_sfx(H)}")(N, _ptr(H), _ptr(V), _ptr(W), _ptr(Ht))
    return Ht


def backtransform(V, Ct) -> np.ndarray:
    """O4: C = V C~ (no conjugation), C~ is N x nev."""
    V = _f(V)
    Ct = _f(Ct, V.dtype)
    if np.iscomplexobj(Ct) and not np.iscomplexobj(V):
        V = _f(V, np.complex128)
    N, nev = Ct.shape
    C = np.zeros_like(Ct, order="F")
    if nev > 0:
        getattr(_load(), f"orc_backtransform_{_sfx(V)}")(N, nev, _ptr(V), _ptr(Ct), _ptr(C))
    return C


def density_matrix(C, f) -> np.ndarray:
    """O7: P_ij = sum_l f_l conj(C_il) C_jl, FULL matrix."""
    C = _f(C)
    N, nev = C.shape
    f = np.ascontiguousarray(np.asarray(f, dtype=np.float64))
    assert f.shape == (nev,)
    P = np.zeros((N, N), dtype=C.dtype, order="F")
    getattr(_load(), f"orc_density_{_sfx(C)}")(N, nev, _ptr(C), f.ctypes.data_as(ctypes.c_void_p), _ptr(P))
    return P


def jacobi(A):
    """O5: cyclic Jacobi, full Hermitian A -> (eps ascending, Q with eigenvectors as columns, sweeps)."""
    A = _f(A)
    N = A.shape[0]
    eps = np.zeros(N, dtype=np.float64)
    Q = np.zeros_like(A, order="F")
    sweeps = getattr(_load(), f"orc_jacobi_{_sfx(A)}")(N, _ptr(A), _ptr(eps), _ptr(Q))
    if sweeps < 0:
        raise RuntimeError("Jacobi did not converge in 60 sweeps")
    return eps, Q, int(sweeps)


def _tri(d, e):
    d = np.ascontiguousarray(np.asarray(d, dtype=np.float64))
    e = np.ascontiguousarray(np.asarray(e, dtype=np.float64))
    n = d.shape[0]
    assert d.ndim == 1 and e.shape == (max(n - 1, 0),)
    if e.size == 0:
        e = np.zeros(1)
    return n, d, e


def sturm_count(d, e, x: float) -> int:
    """O8: number of eigenvalues of tridiag(e, d, e) that are < x."""
    n, d, e = _tri(d, e)
    return int(_load().orc_sturm_count(n, _ptr(d), _ptr(e), float(x)))


def tridiag_eigenvalues(d, e, nev=None) -> np.ndarray:
    """O9: the lowest nev eigenvalues (ascending) of tridiag(e, d, e) by Sturm bisection."""
    n, d, e = _tri(d, e)
    nev = n if nev is None else int(nev)
    out = np.zeros(nev, dtype=np.float64)
    if nev > 0:
        _load().orc_tridiag_eigenvalues(n, _ptr(d), _ptr(e), nev, _ptr(out))
    return out


def inertia_count(A, sigma: float) -> int:
    """O10: number of eigenvalues of the Hermitian matrix A (upper triangle read) that are < sigma, by LDL^H
    without pivoting.  Raises ZeroDivisionError if a pivot is exactly zero."""
    A = _f(A)
    N = A.shape[0]
    r = int(getattr(_load(), f"orc_inertia_{_sfx(A)}")(N, _ptr(A), float(sigma)))
    if r < 0:
        raise ZeroDivisionError("zero pivot in LDL^H: choose another sigma")
    return r


def _common(A, B):
    A, B = np.asarray(A), np.asarray(B)
    dt = np.complex128 if (np.iscomplexobj(A) or np.iscomplexobj(B)) else np.float64
    return _f(A, dt), _f(B, dt)


def matmul_hn(A, B) -> np.ndarray:
    """O11: C = A^H B by the plain triple loop (A: K x M, B: K x N)."""
    A, B = _common(A, B)
    K, Mm = A.shape
    K2, Nn = B.shape
    assert K == K2
    C = np.zeros((Mm, Nn), dtype=A.dtype, order="F")
    if Mm and Nn:
        getattr(_load(), f"orc_matmul_hn_{_sfx(A)}")(Mm, Nn, K, _ptr(A), _ptr(B), _ptr(C))
    return C


def matmul_nn(A, B) -> np.ndarray:
    """O11: C = A B by the plain triple loop (A: M x K, B: K x N)."""
    A, B = _common(A, B)
    Mm, K = A.shape
    K2, Nn = B.shape
    assert K == K2
    C = np.zeros((Mm, Nn), dtype=A.dtype, order="F")
    if Mm and Nn:
        getattr(_load(), f"orc_matmul_nn_{_sfx(A)}")(Mm, Nn, K, _ptr(A), _ptr(B), _ptr(C))
    return C


def truncated_eigh(H, S, delta: float, nev=None):
    """The route for an ill-conditioned S, step by step: eigenvectors D_i of the overlap matrix
    (Jacobi), omit every D_i with sigma_i < delta, transform the eigenproblem to that basis (scaled so that it is
    orthonormal in the S inner product: X = D_kept Sigma_kept^-1/2), solve the standard problem there (Jacobi),
    transform back.  Returns dict(sigma (all, ascending), kept, X (N x kept), Hr, eps, y, C)."""
    H, S = _f(H), _f(S)
    sigma, D, _ = jacobi(S)
    keep = sigma >= delta
    m = int(keep.sum())
    X = np.asfortranarray(D[:, keep] / np.sqrt(sigma[keep])[None, :])
    Hr = matmul_hn(X, matmul_nn(H, X))
    Hr = 0.5 * (Hr + Hr.conj().T)
    eps, y, _ = jacobi(Hr)
    nev = m if nev is None else min(int(nev), m)
    y = np.asfortranarray(y[:, :nev])
    return {"sigma": sigma, "kept": m, "X": X, "Hr": Hr, "eps": eps[:nev], "y": y, "C": matmul_nn(X, y)}


def hermitian_from_upper(Ht_upper) -> np.ndarray:
    """Mirror the upper triangle (incl. diagonal) into a full Hermitian matrix."""
    A = np.asarray(Ht_upper)
    up = np.triu(A, 1)
    d = np.diag(np.diag(A).real if np.iscomplexobj(A) else np.diag(A))
    return up + up.conj().T + d


def generalized_eigh(H, S, nev=None):
    """O6: the whole path of PAPER.md:61-67 on the CPU: returns dict with U, V, Ht (full), eps
    (lowest nev, ascending -- reading Q7), Ct, C."""
    U = cholesky(S)
    V = invert_upper(U)
    Ht = to_standard(H, V)
    eps, Q, sweeps = jacobi(hermitian_from_upper(Ht))
    N = U.shape[0]
    nev = N if nev is None else nev
    Ct = np.asfortranarray(Q[:, :nev])
    C = backtransform(V, Ct)
    return {"U": U, "V": V, "Ht": Ht, "eps": eps[:nev], "Ct": Ct, "C": C, "sweeps": sweeps}
