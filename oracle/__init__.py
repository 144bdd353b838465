"""CPU FP64 oracle for the GP prediction pipeline of arxiv/paper_2602_19683.

TEST INFRASTRUCTURE ONLY.  Importers allowed: ``tests/``, ``__graft_entry__.smoke()``
and the ``cpu_baseline`` / ``--impl reference`` legs of ``bench.py``.  The product
path (``paper_2602_19683_b200``) never imports this package and this package never
imports the product.

The arithmetic lives in ``gp_oracle.c`` (plain C, IEEE double, no BLAS, no tiling);
this module only compiles it with gcc, loads it with ctypes and marshals numpy arrays.
Every function cites the PAPER.md passage it follows in ``gp_oracle.c``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gp_oracle.c")
_LIB = os.path.join(_HERE, "libgp_oracle.so")

# Plain build: -O2, no fast-math, no FMA contraction, so every sum is exactly the
# index-order sum written in the source.
_CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math"]


def build(force: bool = False) -> str:
    """Compile gp_oracle.c -> libgp_oracle.so (idempotent). Returns the library path."""
    stale = force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if stale:
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.run(["gcc", *_CFLAGS, "-o", tmp, _SRC, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        i64 = ctypes.c_int64
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_set_num_threads.argtypes = [ctypes.c_int]
        lib.oracle_assemble.argtypes = [dp, i64, dp, i64, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                        ctypes.c_double, ctypes.c_int, ctypes.c_int, dp]
        lib.oracle_cholesky.argtypes = [dp, i64, dp]
        lib.oracle_cholesky.restype = i64
        lib.oracle_forward_subst.argtypes = [dp, i64, dp, dp]
        lib.oracle_backward_subst.argtypes = [dp, i64, dp, dp]
        lib.oracle_matvec.argtypes = [dp, i64, i64, dp, dp]
        lib.oracle_forward_subst_cols.argtypes = [dp, i64, dp, i64, dp]
        lib.oracle_posterior_cov.argtypes = [dp, i64, i64, dp, dp]
        lib.oracle_backward_subst_cols.argtypes = [dp, i64, dp, i64, dp]
        lib.oracle_posterior_var.argtypes = [dp, i64, i64, dp, dp]
        lib.oracle_log_marginal_likelihood.argtypes = [dp, i64, dp, dp]
        lib.oracle_log_marginal_likelihood.restype = ctypes.c_double
        _lib = lib
    return _lib


def _c(a: np.ndarray, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


@dataclass(frozen=True)
class Hyper:
    """ell = lengthscale, v = vertical lengthscale, noise = sigma^2.
    ell_squared selects the denominator 2*ell^2 instead of the printed 2*ell (reading A1)."""
    lengthscale: float = 1.0
    vertical: float = 1.0
    noise: float = 0.1
    ell_squared: bool = False


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(t: int) -> None:
    _load().oracle_set_num_threads(int(t))


def assemble(A: np.ndarray, B: np.ndarray, h: Hyper, add_noise_diag: bool) -> np.ndarray:
    """Eq. 1: the na x nb matrix of kernel evaluations k(A_i, B_j).
    add_noise_diag=True only for the training matrix K = K_{X,X} (reading A2)."""
    A = _c(A)
    B = _c(B)
    assert A.ndim == 2 and B.ndim == 2 and A.shape[1] == B.shape[1]
    K = np.empty((A.shape[0], B.shape[0]), dtype=np.float64)
    _load().oracle_assemble(_p(A), A.shape[0], _p(B), B.shape[0], A.shape[1], float(h.lengthscale),
                            float(h.vertical), float(h.noise), int(bool(h.ell_squared)),
                            int(bool(add_noise_diag)), _p(K))
    return K


def cholesky(K: np.ndarray) -> np.ndarray:
    """K = L L^T, unblocked; raises on a non-positive pivot."""
    K = _c(K)
    n = K.shape[0]
    assert K.shape == (n, n)
    L = np.zeros((n, n), dtype=np.float64)
    info = _load().oracle_cholesky(_p(K), n, _p(L))
    if info != 0:
        raise np.linalg.LinAlgError(f"oracle_cholesky: non-positive pivot at column {info} (1-based)")
    return L


def forward_subst(L: np.ndarray, b: np.ndarray) -> np.ndarray:
    """L x = b."""
    L = _c(L)
    n = L.shape[0]
    b = _c(b, (n,))
    x = np.empty(n, dtype=np.float64)
    _load().oracle_forward_subst(_p(L), n, _p(b), _p(x))
    return x


def backward_subst(L: np.ndarray, b: np.ndarray) -> np.ndarray:
    """L^T x = b."""
    L = _c(L)
    n = L.shape[0]
    b = _c(b, (n,))
    x = np.empty(n, dtype=np.float64)
    _load().oracle_backward_subst(_p(L), n, _p(b), _p(x))
    return x


def matvec(M: np.ndarray, x: np.ndarray) -> np.ndarray:
    """M x with index-order dot products (y^ = K_{X^,X} alpha)."""
    M = _c(M)
    x = _c(x, (M.shape[1],))
    y = np.empty(M.shape[0], dtype=np.float64)
    _load().oracle_matvec(_p(M), M.shape[0], M.shape[1], _p(x), _p(y))
    return y


def forward_subst_cols(L: np.ndarray, B: np.ndarray) -> np.ndarray:
    """L V = B column by column; B and V are n x m."""
    L = _c(L)
    n = L.shape[0]
    B = _c(B)
    assert B.shape[0] == n
    V = np.empty_like(B)
    _load().oracle_forward_subst_cols(_p(L), n, _p(B), B.shape[1], _p(V))
    return V


def backward_subst_cols(L: np.ndarray, B: np.ndarray) -> np.ndarray:
    """L^T X = B column by column (PAPER.md:72 recurrence per column); B and X are n x m."""
    L = _c(L)
    n = L.shape[0]
    B = _c(B)
    assert B.shape[0] == n
    X = np.empty_like(B)
    _load().oracle_backward_subst_cols(_p(L), n, _p(B), B.shape[1], _p(X))
    return X


def posterior_cov(V: np.ndarray, Kss: np.ndarray) -> np.ndarray:
    """Sigma = K_{X^,X^} - V^T V."""
    V = _c(V)
    n, m = V.shape
    Kss = _c(Kss, (m, m))
    S = np.empty((m, m), dtype=np.float64)
    _load().oracle_posterior_cov(_p(V), n, m, _p(Kss), _p(S))
    return S


def posterior_var(V: np.ndarray, kss_diag: np.ndarray) -> np.ndarray:
    """diag(Sigma): var_a = k(x^_a, x^_a) - sum_i V_ia^2."""
    V = _c(V)
    n, m = V.shape
    kss_diag = _c(kss_diag, (m,))
    var = np.empty(m, dtype=np.float64)
    _load().oracle_posterior_var(_p(V), n, m, _p(kss_diag), _p(var))
    return var


def log_marginal_likelihood(L: np.ndarray, y: np.ndarray, alpha: np.ndarray) -> float:
    """log p(y) = -1/2 y^T alpha - sum_i log L_ii - n/2 log(2 pi)."""
    L = _c(L)
    n = L.shape[0]
    return float(_load().oracle_log_marginal_likelihood(_p(L), n, _p(_c(y, (n,))), _p(_c(alpha, (n,)))))


@dataclass
class Prediction:
    K: np.ndarray | None
    L: np.ndarray
    beta: np.ndarray
    alpha: np.ndarray
    mean: np.ndarray | None = None
    V: np.ndarray | None = None
    Sigma: np.ndarray | None = None
    var: np.ndarray | None = None


def fit(X: np.ndarray, y: np.ndarray, h: Hyper, keep_K: bool = True) -> Prediction:
    """Steps a1-a8: assemble K (noise on the diagonal), L, beta, alpha."""
    K = assemble(X, X, h, add_noise_diag=True)
    L = cholesky(K)
    beta = forward_subst(L, y)
    alpha = backward_subst(L, beta)
    return Prediction(K=K if keep_K else None, L=L, beta=beta, alpha=alpha)


def predict(X: np.ndarray, y: np.ndarray, Xs: np.ndarray, h: Hyper, full_cov: bool = True,
            fitted: Prediction | None = None, variance: bool = False) -> Prediction:
    """The whole pipeline of PAPER.md section 4.1 in the paper's order:
    K, L, beta, alpha, K_{X^,X}, mean, V, W, Sigma."""
    p = fitted if fitted is not None else fit(X, y, h)
    Kxs = assemble(Xs, X, h, add_noise_diag=False)          # m x n, noise-free (A2, A5)
    p.mean = matvec(Kxs, p.alpha)                           # Eq. 2
    if full_cov:
        p.V = forward_subst_cols(p.L, np.ascontiguousarray(Kxs.T))   # L V = K_{X,X^}
        Kss = assemble(Xs, Xs, h, add_noise_diag=False)     # prior test covariance, noise-free
        p.Sigma = posterior_cov(p.V, Kss)                   # Eq. 3
    if variance:                                            # "predict with uncertainty": the diagonal only
        if p.V is None:
            p.V = forward_subst_cols(p.L, np.ascontiguousarray(Kxs.T))
        p.var = posterior_var(p.V, np.full(Xs.shape[0], h.vertical))   # k(x,x) = v exp(0), noise-free (A2)
    return p
