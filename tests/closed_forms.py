"""Closed forms the oracle is pinned against (numpy; independent of oracle/ovl_oracle.c and of the CUDA path).

Everything here follows from eq. 2.2 by Fourier analysis, not by re-running the stencil:
on U = 1 (or a pure gauge) plane waves diagonalise D_W.
"""
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden_gammas():
    """The four gamma matrices of tests/golden/gamma_basis.txt (R2)."""
    blocks, cur = [], []
    with open(os.path.join(GOLDEN, "gamma_basis.txt")) as f:
        for line in f:
            line = line.strip()
            if line.startswith("#"):
                continue
            if not line:
                if cur:
                    blocks.append(cur)
                    cur = []
                continue
            cur.append([complex(*map(float, tok.split(","))) for tok in line.split()])
    if cur:
        blocks.append(cur)
    g = np.array(blocks, dtype=np.complex128)
    assert g.shape == (4, 4, 4)
    return g


def momenta(dims):
    """p_mu grids: periodic x,y,z (2 pi n / L), antiperiodic t (2 pi (n + 1/2) / Lt). Returns 4 arrays broadcast
    to the (Lt, Lz, Ly, Lx) lattice view."""
    lx, ly, lz, lt = dims
    px = 2 * np.pi * np.arange(lx) / lx
    py = 2 * np.pi * np.arange(ly) / ly
    pz = 2 * np.pi * np.arange(lz) / lz
    pt = 2 * np.pi * (np.arange(lt) + 0.5) / lt
    return (px[None, None, None, :], py[None, None, :, None], pz[None, :, None, None], pt[:, None, None, None])


def plane_wave(dims, n, u):
    """psi(x) = u exp(i p.x), p from integer mode numbers n (t component is n_t + 1/2). Shape (V,4,3)."""
    lx, ly, lz, lt = dims
    p = [2 * np.pi * n[0] / lx, 2 * np.pi * n[1] / ly, 2 * np.pi * n[2] / lz, 2 * np.pi * (n[3] + 0.5) / lt]
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    ph = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t)).reshape(-1)
    return ph[:, None, None] * u[None, :, :], p


def dw_symbol(p, gammas, mass=0.0):
    """4x4 spin matrix (4 - mass - sum cos p_mu) + i sum gamma_mu sin p_mu: D_W - mass on a plane wave."""
    m = (4.0 - mass - sum(np.cos(pm) for pm in p)) * np.eye(4, dtype=np.complex128)
    for mu in range(4):
        m = m + 1j * np.sin(p[mu]) * gammas[mu]
    return m


def free_sign_fft(dims, psi, gammas, m_w=1.5, g=None):
    """Exact sign(K) psi on a pure gauge U_mu(x) = g(x) g(x+mu)^dag (g = None: U = 1), any volume:
    sign(K) = g F^-1 [ gamma5 ((4 - m_w - sum cos p) + i sum gamma_mu sin p) / omega(p) ] F g^dag."""
    lx, ly, lz, lt = dims
    v = lx * ly * lz * lt
    f = psi.reshape(v, 4, 3)
    if g is not None:
        f = np.einsum("xba,xsb->xsa", np.conj(g), f)  # g^dag psi
    f = f.reshape(lt, lz, ly, lx, 4, 3)
    tw = np.exp(-1j * np.pi * np.arange(lt) / lt)[:, None, None, None, None, None]
    ft = np.fft.fftn(f * tw, axes=(0, 1, 2, 3))
    px, py, pz, pt = momenta(dims)
    a = 4.0 - m_w - (np.cos(px) + np.cos(py) + np.cos(pz) + np.cos(pt))
    s = [np.sin(px) + 0 * a, np.sin(py) + 0 * a, np.sin(pz) + 0 * a, np.sin(pt) + 0 * a]
    omega = np.sqrt(a * a + sum(si * si for si in s))
    g5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(np.complex128)
    sym = a[..., None, None] * np.eye(4)[None, None, None, None]
    for mu in range(4):
        sym = sym + 1j * s[mu][..., None, None] * gammas[mu][None, None, None, None]
    sym = np.einsum("ab,...bc->...ac", g5, sym) / omega[..., None, None]
    out = np.einsum("...ab,...bc->...ac", sym, ft)
    out = np.fft.ifftn(out, axes=(0, 1, 2, 3)) * np.conj(tw)
    out = out.reshape(v, 4, 3)
    if g is not None:
        out = np.einsum("xab,xsb->xsa", g, out)
    return out, omega


def lowest_pure_gauge_eigenpairs(dims, g, gammas, nev, m_w=1.5):
    """Exact eigenpairs of K = gamma5 (D_W - m_w) on the pure gauge U_mu(x) = g(x) g(x+mu)^dag (g = None: U = 1), the
    `nev` of smallest |lambda| (ties cut in a fixed order, R11): K[U^g] = g K[1] g^dag site by site, and on
    U = 1 the plane wave exp(i p.x) u e_c is an eigenvector whenever u is an eigenvector of the Hermitian 4x4 symbol
    gamma5 ((4 - m_w - sum cos p) + i sum gamma_mu sin p), eigenvalues +-omega(p), each twice, times 3 colours.
    Returns (phi of shape (nev, V, 4, 3), orthonormal; lambda of shape (nev,))."""
    lx, ly, lz, lt = dims
    v = lx * ly * lz * lt
    px, py, pz, pt = momenta(dims)
    a = 4.0 - m_w - (np.cos(px) + np.cos(py) + np.cos(pz) + np.cos(pt))
    om = np.sqrt(a * a + np.sin(px) ** 2 + np.sin(py) ** 2 + np.sin(pz) ** 2 + np.sin(pt) ** 2 + 0 * a).reshape(-1)
    order = np.argsort(om, kind="stable")
    g5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(np.complex128)
    gm = np.eye(3, dtype=np.complex128)[None].repeat(v, 0) if g is None else g
    phis, lams = [], []
    for flat in order:
        nt, rem = divmod(int(flat), lz * ly * lx)
        nz, rem = divmod(rem, ly * lx)
        ny, nx = divmod(rem, lx)
        wave, p = plane_wave(dims, (nx, ny, nz, nt), np.ones((1, 1)))
        ph = wave[:, 0, 0] / np.sqrt(v)
        lam, vec = np.linalg.eigh(g5 @ dw_symbol(p, gammas, m_w))
        for j in np.argsort(np.abs(lam), kind="stable"):
            for c in range(3):
                phis.append(ph[:, None, None] * vec[:, j][None, :, None] * gm[:, None, :, c])
                lams.append(lam[j])
                if len(phis) == nev:
                    return np.ascontiguousarray(np.stack(phis)), np.array(lams)
    raise ValueError("nev exceeds 12 V")
