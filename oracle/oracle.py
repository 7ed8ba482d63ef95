"""ctypes front end of the CPU oracle (oracle/ovl_oracle.c) + dense helpers.

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the cpu_baseline /
--impl reference legs of bench.py.  Never imported by the product package, and imports nothing from it.

All arrays are numpy complex128 in the canonical layout of DESIGN.md "Boundary":
links (V,4,3,3), spinors (V,4,3), eigenvectors (nev,V,4,3); dims = (Lx,Ly,Lz,Lt).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ovl_oracle.c")
_LIB = os.path.join(_HERE, "libovl_oracle.so")
_lib = None

_c = ctypes
_pd = _c.POINTER(_c.c_double)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C99 + OpenMP). Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = _c.CDLL(_LIB)
        _lib.orc_cheb_scalar.restype = _c.c_double
        _lib.orc_cheb_scalar.argtypes = [_c.c_int, _c.c_void_p, _c.c_double]
        _lib.orc_cg.restype = _c.c_int
        _lib.orc_cg_chiral.restype = _c.c_int
        _lib.orc_num_threads.restype = _c.c_int
    return _lib


def num_threads() -> int:
    return int(_load().orc_num_threads())


def _dims(dims):
    return (_c.c_int * 4)(*[int(d) for d in dims])


def _vol(dims):
    return int(np.prod([int(d) for d in dims]))


def _in(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _p(a):
    return a.ctypes.data_as(_c.c_void_p)


def _alpha(alpha):
    return np.ascontiguousarray(alpha, dtype=np.float64)


def gamma(mu: int) -> np.ndarray:
    out = np.zeros((4, 4), dtype=np.complex128)
    _load().orc_gamma(_c.c_int(mu), _p(out))
    return out


def dw(dims, U, psi):
    """D_W psi, eq. 2.2."""
    v = _vol(dims)
    U = _in(U, (v, 4, 3, 3)); psi = _in(psi, (v, 4, 3))
    out = np.empty_like(psi)
    _load().orc_dw(_dims(dims), _p(U), _p(psi), _p(out))
    return out


def khat(dims, U, psi, m_w=1.5, lambda_max=6.5):
    """K^ psi = gamma5 (D_W - m_w) psi / lambda_max."""
    v = _vol(dims)
    U = _in(U, (v, 4, 3, 3)); psi = _in(psi, (v, 4, 3))
    out = np.empty_like(psi)
    _load().orc_khat(_dims(dims), _p(U), _c.c_double(m_w), _c.c_double(lambda_max), _p(psi), _p(out))
    return out


def cheb(dims, U, alpha, psi, m_w=1.5, lambda_max=6.5, clenshaw=False):
    """sum_m alpha_m T_m(K^) psi (first sum of eq. 2.3)."""
    v = _vol(dims)
    U = _in(U, (v, 4, 3, 3)); psi = _in(psi, (v, 4, 3)); alpha = _alpha(alpha)
    out = np.empty_like(psi)
    fn = _load().orc_clenshaw if clenshaw else _load().orc_cheb
    fn(_dims(dims), _p(U), _c.c_double(m_w), _c.c_double(lambda_max), _c.c_int(len(alpha) - 1), _p(alpha),
       _p(psi), _p(out))
    return out


def cheb_scalar(alpha, x: float) -> float:
    alpha = _alpha(alpha)
    return float(_load().orc_cheb_scalar(_c.c_int(len(alpha) - 1), _p(alpha), _c.c_double(x)))


def _defl(dims, phi, lam):
    if phi is None or len(lam) == 0:
        return 0, np.zeros(1, dtype=np.complex128), np.zeros(1, dtype=np.float64)
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    phi = _in(phi, (len(lam), _vol(dims), 4, 3))
    return len(lam), phi, lam


def sign(dims, U, alpha, psi, phi=None, lam=(), m_w=1.5, lambda_max=6.5):
    """Deflated Chebyshev sign(K) psi, eq. 2.3."""
    v = _vol(dims)
    U = _in(U, (v, 4, 3, 3)); psi = _in(psi, (v, 4, 3)); alpha = _alpha(alpha)
    nev, phi, lam = _defl(dims, phi, lam)
    out = np.empty_like(psi)
    _load().orc_sign(_dims(dims), _p(U), _c.c_double(m_w), _c.c_double(lambda_max), _c.c_int(len(alpha) - 1),
                     _p(alpha), _c.c_int(nev), _p(phi), _p(lam), _p(psi), _p(out))
    return out


def overlap(dims, U, alpha, mu, psi, phi=None, lam=(), dagger=False, m_w=1.5, lambda_max=6.5):
    """D[mu] psi (eq. 2.1) or D[mu]^dag psi."""
    v = _vol(dims)
    U = _in(U, (v, 4, 3, 3)); psi = _in(psi, (v, 4, 3)); alpha = _alpha(alpha)
    nev, phi, lam = _defl(dims, phi, lam)
    out = np.empty_like(psi)
    _load().orc_overlap(_dims(dims), _p(U), _c.c_double(m_w), _c.c_double(lambda_max), _c.c_int(len(alpha) - 1),
                        _p(alpha), _c.c_int(nev), _p(phi), _p(lam), _c.c_double(mu), _c.c_int(int(dagger)),
                        _p(psi), _p(out))
    return out


def cg(dims, U, alpha, mu, b, tol, maxiter, phi=None, lam=(), m_w=1.5, lambda_max=6.5):
    """CG on D^dag D x = b, x0 = 0. Returns (x, iterations, true relative residual)."""
    v = _vol(dims)
    U = _in(U, (v, 4, 3, 3)); b = _in(b, (v, 4, 3)); alpha = _alpha(alpha)
    nev, phi, lam = _defl(dims, phi, lam)
    x = np.empty_like(b)
    rel = _c.c_double(0.0)
    it = _load().orc_cg(_dims(dims), _p(U), _c.c_double(m_w), _c.c_double(lambda_max), _c.c_int(len(alpha) - 1),
                        _p(alpha), _c.c_int(nev), _p(phi), _p(lam), _c.c_double(mu), _p(b), _p(x),
                        _c.c_double(tol), _c.c_int(maxiter), _c.byref(rel))
    return x, int(it), float(rel.value)


def chiral_op(dims, U, alpha, mu, chirality, v, phi=None, lam=(), m_w=1.5, lambda_max=6.5):
    """A_c v = 1/2 (1+mu^2) P_c v + c/2 (1-mu^2) P_c sign(K) P_c v  (reading R23)."""
    vv = _vol(dims)
    U = _in(U, (vv, 4, 3, 3)); v = _in(v, (vv, 4, 3)); alpha = _alpha(alpha)
    nev, phi, lam = _defl(dims, phi, lam)
    out = np.empty_like(v)
    _load().orc_chiral_op(_dims(dims), _p(U), _c.c_double(m_w), _c.c_double(lambda_max), _c.c_int(len(alpha) - 1),
                          _p(alpha), _c.c_int(nev), _p(phi), _p(lam), _c.c_double(mu), _c.c_int(int(chirality)),
                          _p(v), _p(out))
    return out


def cg_chiral(dims, U, alpha, mu, chirality, b, tol, maxiter, phi=None, lam=(), m_w=1.5, lambda_max=6.5):
    """CG on A_c x = P_c b in the chirality sector. Returns (x, iterations, true relative residual)."""
    v = _vol(dims)
    U = _in(U, (v, 4, 3, 3)); b = _in(b, (v, 4, 3)); alpha = _alpha(alpha)
    nev, phi, lam = _defl(dims, phi, lam)
    x = np.empty_like(b)
    rel = _c.c_double(0.0)
    it = _load().orc_cg_chiral(_dims(dims), _p(U), _c.c_double(m_w), _c.c_double(lambda_max), _c.c_int(len(alpha) - 1),
                               _p(alpha), _c.c_int(nev), _p(phi), _p(lam), _c.c_double(mu), _c.c_int(int(chirality)),
                               _p(b), _p(x), _c.c_double(tol), _c.c_int(maxiter), _c.byref(rel))
    return x, int(it), float(rel.value)


# --------------------------------------------------------------------------------------
# dense helpers (tiny lattices only): the oracle's own operator as a matrix, exact sign
# --------------------------------------------------------------------------------------

def dense(apply, n: int) -> np.ndarray:
    """Matrix of a linear map given as a function on (V,4,3) spinors, column by column."""
    m = np.empty((n, n), dtype=np.complex128)
    e = np.zeros(n, dtype=np.complex128)
    for j in range(n):
        e[j] = 1.0
        m[:, j] = apply(e.reshape(n // 12, 4, 3)).reshape(n)
        e[j] = 0.0
    return m


def dense_k(dims, U, m_w=1.5):
    """K = gamma5 (D_W - m_w) as a dense 12V x 12V matrix (unscaled)."""
    n = 12 * _vol(dims)
    return dense(lambda p: khat(dims, U, p, m_w, 1.0), n)


def exact_sign_dense(K: np.ndarray):
    """sign(K) of a Hermitian matrix by eigendecomposition. Returns (sign matrix, eigenvalues, eigenvectors)."""
    lam, w = np.linalg.eigh(0.5 * (K + K.conj().T))
    return (w * np.sign(lam)) @ w.conj().T, lam, w


def lowest_eigenpairs(dims, U, nev: int, m_w=1.5, filter_degree: int = 0, tol: float = 1e-9, seed: int = 7):
    """The nev eigenpairs of K with smallest |lambda| ("oracle Lanczos"; reading R11):
    ARPACK on K^2 (shift-free, smallest algebraic) followed by a Rayleigh-Ritz of K in the found subspace.
    Returns (phi (nev,V,4,3), lambda (nev,), max residual ||K phi - lambda phi||)."""
    from scipy.sparse.linalg import LinearOperator, eigsh
    v = _vol(dims)
    n = 12 * v

    def k_apply(x):
        return khat(dims, U, x.reshape(v, 4, 3), m_w, 1.0).reshape(n)

    def k2(x):
        return k_apply(k_apply(np.asarray(x, dtype=np.complex128)))

    op = LinearOperator((n, n), matvec=k2, dtype=np.complex128)
    rng = np.random.Generator(np.random.PCG64(seed))
    v0 = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    extra = max(4, nev // 2)
    _, vecs = eigsh(op, k=nev + extra, which="SA", tol=tol, v0=v0, ncv=max(3 * (nev + extra), 40))
    q, _ = np.linalg.qr(vecs)
    kq = np.stack([k_apply(q[:, j]) for j in range(q.shape[1])], axis=1)
    h = q.conj().T @ kq
    lam, y = np.linalg.eigh(0.5 * (h + h.conj().T))
    order = np.argsort(np.abs(lam))[:nev]
    lam = lam[order]
    phi = q @ y[:, order]
    res = max(np.linalg.norm(k_apply(phi[:, j]) - lam[j] * phi[:, j]) for j in range(nev))
    return np.ascontiguousarray(phi.T.reshape(nev, v, 4, 3)), lam, float(res)
