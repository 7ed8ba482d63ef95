"""Seeded synthetic input generators (numpy only) shared by tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no Wilson stencil, no sign function,
no overlap operator): it only manufactures the *inputs* the hot path consumes --
gauge links, spinors, Chebyshev coefficient tables -- so that the CUDA path and the CPU
oracle can be fed identical arrays while sharing no code.

Stand-in statement: the paper measures on Luscher-Weisz / MILC asqtad ensembles
(Table 2) that are not available; seeded near-identity SU(3) links with
3 steps of stout smearing (plain isotropic stout, reading R16)
stand in for them, with the paper's two volumes 8^3x32 and 20^3x64.

Conventions: dims = (Lx, Ly, Lz, Lt); site index
s = x + Lx*(y + Ly*(z + Lz*t)); links U[s, mu, row, col] with mu in (x, y, z, t);
spinors psi[s, spin, colour]; everything complex128, C-contiguous.
"""
from __future__ import annotations

import numpy as np

SEED_BASE = 1510068970  # arXiv number + one digit; per-config seeds are SEED_BASE + k


def volume(dims) -> int:
    lx, ly, lz, lt = (int(d) for d in dims)
    return lx * ly * lz * lt


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(int(seed)))


def _complex_gaussian(rng: np.random.Generator, shape) -> np.ndarray:
    """(g1 + i g2)/sqrt(2), all real parts drawn first, then all imaginary parts (R15/R17)."""
    re = rng.standard_normal(shape)
    im = rng.standard_normal(shape)
    return (re + 1j * im) / np.sqrt(2.0)


def gaussian_spinor(dims, seed: int) -> np.ndarray:
    """Complex Gaussian spinor, 12 components per site, shape (V, 4, 3) complex128 (R17)."""
    return np.ascontiguousarray(_complex_gaussian(_rng(seed), (volume(dims), 4, 3)))


def unit_links(dims) -> np.ndarray:
    """Free field U = 1, shape (V, 4, 3, 3)."""
    u = np.zeros((volume(dims), 4, 3, 3), dtype=np.complex128)
    u[..., 0, 0] = u[..., 1, 1] = u[..., 2, 2] = 1.0
    return u


def _traceless_hermitian(rng: np.random.Generator, shape) -> np.ndarray:
    a = _complex_gaussian(rng, shape + (3, 3))
    h = 0.5 * (a + np.conj(np.swapaxes(a, -1, -2)))
    tr = np.trace(h, axis1=-2, axis2=-1).real / 3.0
    h[..., 0, 0] -= tr
    h[..., 1, 1] -= tr
    h[..., 2, 2] -= tr
    return h


def _exp_i_hermitian(h: np.ndarray, eps: float) -> np.ndarray:
    """exp(i*eps*H) through the Hermitian eigendecomposition: exactly unitary, det 1 for tr H = 0."""
    lam, w = np.linalg.eigh(h)
    ph = np.exp(1j * eps * lam)
    return np.einsum("...ij,...j,...kj->...ik", w, ph, np.conj(w))


def random_links(dims, eps: float, seed: int) -> np.ndarray:
    """U = exp(i*eps*H), H seeded Gaussian traceless Hermitian 3x3 per link (BASELINE.json configs, R15)."""
    h = _traceless_hermitian(_rng(seed), (volume(dims), 4))
    return np.ascontiguousarray(_exp_i_hermitian(h, eps))


def tiled_links(dims, block, eps: float, seed: int) -> np.ndarray:
    """random_links on a `block` sub-lattice, repeated periodically to fill `dims` (every extent of dims a multiple of
    the block's).  Still a valid SU(3) gauge field; used where generating V*4 independent matrices on the host would
    take minutes (the 48^3 x 96 volume of BASELINE config 4)."""
    reps = [d // b for d, b in zip(dims, block)]
    assert all(r * b == d for r, b, d in zip(reps, block, dims)), "dims must be multiples of block"
    u = _lat(random_links(block, eps, seed), block)                       # (bt, bz, by, bx, 4, 3, 3)
    u = np.tile(u, (reps[3], reps[2], reps[1], reps[0], 1, 1, 1))
    return np.ascontiguousarray(u.reshape(volume(dims), 4, 3, 3))


def random_su3_field(dims, seed: int, eps: float = 2.0) -> np.ndarray:
    """One SU(3) matrix g(x) per site, far from identity; shape (V, 3, 3). For gauge transformations."""
    h = _traceless_hermitian(_rng(seed), (volume(dims),))
    return np.ascontiguousarray(_exp_i_hermitian(h, eps))


def _lat(a: np.ndarray, dims) -> np.ndarray:
    lx, ly, lz, lt = dims
    return a.reshape((lt, lz, ly, lx) + a.shape[1:])


_AXIS = {0: 3, 1: 2, 2: 1, 3: 0}  # direction mu -> numpy axis of the (Lt, Lz, Ly, Lx, ...) view


def shift(field: np.ndarray, dims, mu: int, step: int) -> np.ndarray:
    """Return f'(x) = f(x + step*mu_hat), periodic. `field` has leading axis V."""
    f = _lat(field, dims)
    return np.roll(f, -step, axis=_AXIS[mu]).reshape(field.shape)


def pure_gauge_links(dims, seed: int):
    """U_mu(x) = g(x) g(x+mu)^dagger with random g: plaquette exactly 1. Returns (U, g)."""
    g = random_su3_field(dims, seed)
    u = np.empty((volume(dims), 4, 3, 3), dtype=np.complex128)
    for mu in range(4):
        gp = shift(g, dims, mu, +1)
        u[:, mu] = g @ np.conj(np.swapaxes(gp, -1, -2))
    return u, g


def gauge_transform_links(u: np.ndarray, g: np.ndarray, dims) -> np.ndarray:
    """U^g_mu(x) = g(x) U_mu(x) g(x+mu)^dagger."""
    out = np.empty_like(u)
    for mu in range(4):
        gp = shift(g, dims, mu, +1)
        out[:, mu] = g @ u[:, mu] @ np.conj(np.swapaxes(gp, -1, -2))
    return out


def _dag(m: np.ndarray) -> np.ndarray:
    return np.conj(np.swapaxes(m, -1, -2))


def plaquette(u: np.ndarray, dims) -> float:
    """Average of Re tr U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag / 3 over sites and the 6 planes."""
    tot = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            p = u[:, mu] @ shift(u[:, nu], dims, mu, 1) @ _dag(shift(u[:, mu], dims, nu, 1)) @ _dag(u[:, nu])
            tot += np.trace(p, axis1=-2, axis2=-1).real.mean() / 3.0
    return tot / 6.0


def stout_smear(u: np.ndarray, dims, rho: float = 0.1, steps: int = 3) -> np.ndarray:
    """Plain isotropic 4-D stout smearing (Morningstar-Peardon, PAPER.md:60 / ref [6]; reading R16):
    C_mu = rho * sum_{nu != mu} (two staples), Omega = C_mu U_mu^dag,
    Q = (i/2)(Omega^dag - Omega) - (i/6) tr(Omega^dag - Omega), U' = exp(iQ) U. Periodic links."""
    u = u.copy()
    for _ in range(steps):
        new = np.empty_like(u)
        for mu in range(4):
            c = np.zeros_like(u[:, mu])
            for nu in range(4):
                if nu == mu:
                    continue
                u_nu = u[:, nu]
                # upper staple: U_nu(x) U_mu(x+nu) U_nu(x+mu)^dag
                c += u_nu @ shift(u[:, mu], dims, nu, 1) @ _dag(shift(u_nu, dims, mu, 1))
                # lower staple: U_nu(x-nu)^dag U_mu(x-nu) U_nu(x-nu+mu)
                low = _dag(u_nu) @ u[:, mu] @ shift(u_nu, dims, mu, 1)
                c += shift(low, dims, nu, -1)
            omega = rho * c @ _dag(u[:, mu])
            d = _dag(omega) - omega
            tr = np.trace(d, axis1=-2, axis2=-1)
            q = 0.5j * d
            for k in range(3):
                q[:, k, k] -= (1j / 6.0) * tr
            q = 0.5 * (q + _dag(q))  # remove rounding-level anti-Hermitian part
            new[:, mu] = _exp_i_hermitian(q, 1.0) @ u[:, mu]
        u = new
    return np.ascontiguousarray(u)


def config_links(dims, eps: float, seed: int, stout_steps: int = 0, rho: float = 0.1) -> np.ndarray:
    u = random_links(dims, eps, seed)
    if stout_steps:
        u = stout_smear(u, dims, rho, stout_steps)
    return u


# --------------------------------------------------------------------------------------
# Chebyshev coefficient table alpha_m (input data of the hot path, reading R6)
# --------------------------------------------------------------------------------------

def chebyshev_sign_coeffs(degree: int, eps: float) -> np.ndarray:
    """alpha[0..degree] with sum_m alpha_m T_m(x) ~ sign(x) on eps <= |x| <= 1.

    Recipe (R6): n = floor((degree-1)/2); c_k = Chebyshev coefficients of y^(-1/2) on
    y in [eps^2, 1] in the variable z = (2y - 1 - eps^2)/(1 - eps^2) (Gauss-Chebyshev
    quadrature); the odd polynomial p(x) = x * sum_k c_k T_k(z(x^2)) of degree 2n+1 is
    re-expanded exactly in T_m(x) by a discrete Chebyshev transform; even m are set to 0.
    """
    degree = int(degree)
    if degree < 1 or not (0.0 < eps < 1.0):
        raise ValueError("degree >= 1 and 0 < eps < 1 required")
    n = (degree - 1) // 2
    # inner expansion of y^(-1/2)
    nq = 8 * (n + 1)
    th = np.pi * (np.arange(nq) + 0.5) / nq
    z = np.cos(th)
    y = 0.5 * ((1.0 - eps * eps) * z + 1.0 + eps * eps)
    f = 1.0 / np.sqrt(y)
    k = np.arange(n + 1)
    c = (2.0 / nq) * (np.cos(np.outer(k, th)) @ f)
    c[0] *= 0.5
    # outer re-expansion in T_m(x), exact for a polynomial of degree 2n+1 with nx > 2n+1 nodes
    nx = 2 * (degree + 2)
    tx = np.pi * (np.arange(nx) + 0.5) / nx
    x = np.cos(tx)
    zx = (2.0 * x * x - 1.0 - eps * eps) / (1.0 - eps * eps)
    p = x * np.polynomial.chebyshev.chebval(zx, c)
    m = np.arange(degree + 1)
    alpha = (2.0 / nx) * (np.cos(np.outer(m, tx)) @ p)
    alpha[0] *= 0.5
    alpha[0::2] = 0.0
    return np.ascontiguousarray(alpha)


def chebyshev_eval(alpha: np.ndarray, x: np.ndarray) -> np.ndarray:
    """sum_m alpha_m T_m(x) through numpy's own Chebyshev evaluator (for checking tables only)."""
    return np.polynomial.chebyshev.chebval(np.asarray(x, dtype=np.float64), np.asarray(alpha))


def orthonormal_vectors(dims, nvec: int, seed: int) -> np.ndarray:
    """nvec orthonormal complex vectors of length 12V, shape (nvec, V, 4, 3): a generic deflation-shaped
    input (QR of a Gaussian block). NOT eigenvectors -- eq. 2.3 is a well-defined linear map for any
    (phi_i, lambda_i) (reading R10), which is all parity and timing need."""
    v = volume(dims)
    a = _complex_gaussian(_rng(seed), (12 * v, nvec))
    q, _ = np.linalg.qr(a)
    return np.ascontiguousarray(q.T.reshape(nvec, v, 4, 3))


def phase_vectors(dims, nvec: int, seed: int) -> np.ndarray:
    """nvec exactly orthonormal vectors in O(12V) work each, for deflation-shaped inputs at volumes where a QR of a
    (12V x nvec) Gaussian block is too expensive: phi_i[e] = exp(i (theta_e + 2 pi i e / n)) / sqrt(n), theta seeded
    uniform phases, e the flat (site, spin, colour) index, n = 12V.  <phi_i, phi_j> = (1/n) sum_e exp(2 pi i (j-i) e/n)
    = delta_ij.  NOT eigenvectors (reading R10).  Shape (nvec, V, 4, 3)."""
    n = 12 * volume(dims)
    theta = _rng(seed).uniform(0.0, 2.0 * np.pi, n)
    e = np.arange(n, dtype=np.float64)
    out = np.empty((nvec, n), dtype=np.complex128)
    for i in range(nvec):
        ang = theta + (2.0 * np.pi * i / n) * e
        out[i] = (np.cos(ang) + 1j * np.sin(ang)) / np.sqrt(n)
    return out.reshape(nvec, volume(dims), 4, 3)


# --------------------------------------------------------------------------------------
# The BASELINE.json configurations as concrete seeded inputs; bench.py times exactly these
# arrays and tests/test_gpu_configs.py holds the CUDA path against the oracle on them.
# --------------------------------------------------------------------------------------

WORKLOADS = {
    # name: dims, link eps, stout steps, mu, degree, nev, eps of the polynomial (lower spectral edge / lambda_max)
    "cfg3": dict(dims=(20, 20, 20, 64), link_eps=0.25, stout=3, mu=0.01, degree=400, nev=50, poly_eps=0.95 * 0.5 / 6.5, k=3,
                 desc="BASELINE config 3: 20^3x64, U=exp(0.25iH)+3 stout rho=0.1, mu=0.01, degree 400, 50 deflation vectors"),
    "cfg1": dict(dims=(8, 8, 8, 32), link_eps=0.3, stout=3, mu=0.01, degree=200, nev=20, poly_eps=0.95 * 0.505 / 6.5, k=1,
                 desc="BASELINE config 1: 8^3x32, U=exp(0.3iH)+3 stout rho=0.1, mu=0.01, degree 200, 20 deflation vectors"),
    "tiny": dict(dims=(4, 4, 4, 8), link_eps=0.3, stout=1, mu=0.01, degree=40, nev=4, poly_eps=0.09, k=9,
                 desc="4^3x8 smoke-sized workload (not a benchmark)"),
}
CFG2_MU, CFG2_TOL, CFG2_SEED_OFF = 0.05, 1e-8, 7  # BASELINE config 2 = the cfg1 lattice, CG on D^dag D x = b


def workload(name: str) -> dict:
    return dict(WORKLOADS[name], name=name)


def workload_inputs(w: dict, seed_off: int = 0, need_phi: bool = True):
    """(U, psi, alpha, phi, lambda) of a workload: smeared seeded links, Gaussian right-hand side (seed_off selects
    another one on the same links), the Chebyshev table, and nev exactly orthonormal deflation-shaped vectors with
    prescribed eigenvalues of both signs near the lower spectral edge (reading R10: eq. 2.3 is a linear map for any
    (phi_i, lambda_i); true eigenpairs at these volumes exist in closed form on pure-gauge links only, tests/closed_forms.py)."""
    dims, k = w["dims"], w.get("k", 7)
    U = config_links(dims, w["link_eps"], SEED_BASE + k, stout_steps=w["stout"])
    psi = gaussian_spinor(dims, SEED_BASE + 100 + k + 1000 * seed_off)
    alpha = chebyshev_sign_coeffs(w["degree"], w["poly_eps"])
    nev = w["nev"]
    phi = phase_vectors(dims, nev, SEED_BASE + 200 + k) if (nev and need_phi) else None
    lam = 0.5 * np.where(np.arange(nev) % 2 == 0, 1.0, -1.0) * (1.0 + 0.002 * np.arange(nev))
    return U, psi, alpha, phi, lam
