"""Pins of the CPU oracle (oracle/ovl_oracle.c) against what the paper and the mathematics fix.

No GPU here.  Each test is chosen so that a plausible mistake in the oracle -- a dropped term, a wrong sign or
index, a transposed link, a wrong boundary phase -- fails at least one of them.
"""
import numpy as np
import pytest

from paper_1510_06897_b200 import inputs
from tests.closed_forms import dw_symbol, free_sign_fft, golden_gammas, lowest_pure_gauge_eigenpairs, plane_wave
from tests.conftest import rel_err

G5 = np.array([1.0, 1.0, -1.0, -1.0])


def g5(psi):
    return psi * G5[None, :, None]


def vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


# ---------------------------------------------------------------- gamma basis (R2)

def test_gamma_basis_matches_golden_and_clifford(orc):
    gold = golden_gammas()
    gam = np.array([orc.gamma(mu) for mu in range(4)])
    assert np.array_equal(gam, gold)
    for mu in range(4):
        assert np.array_equal(gam[mu], gam[mu].conj().T)
        for nu in range(4):
            anti = gam[mu] @ gam[nu] + gam[nu] @ gam[mu]
            assert np.allclose(anti, 2.0 * (mu == nu) * np.eye(4), atol=0)
    assert np.array_equal(gam[0] @ gam[1] @ gam[2] @ gam[3], np.diag(G5).astype(complex))


# ---------------------------------------------------------------- D_W (eq. 2.2)

@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 10), (2, 2, 2, 2), (6, 4, 2, 8), (3, 5, 4, 6), (5, 3, 7, 3)])
def test_dw_free_field_plane_waves(orc, dims):
    """U = 1: D_W u e^{ipx} = [(4 - sum cos p) + i sum gamma sin p] u e^{ipx}; antiperiodic t -> p_t half-integer."""
    gam = golden_gammas()
    U = inputs.unit_links(dims)
    rng = np.random.default_rng(11)
    for trial in range(6):
        n = [int(rng.integers(0, d)) for d in dims]
        u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        psi, p = plane_wave(dims, n, u)
        want = np.einsum("ab,xbc->xac", dw_symbol(p, gam), psi)
        got = orc.dw(dims, U, psi)
        assert rel_err(got, want) < 1e-13, (dims, n)


def test_dw_free_spectrum_dense(orc):
    """Dense 2^4 and 4x2x2x4 free operators: eigenvalues (4 - sum cos p) +- i sqrt(sum sin^2 p), each x6."""
    for dims in [(2, 2, 2, 2), (4, 2, 2, 4)]:
        U = inputs.unit_links(dims)
        n = 12 * inputs.volume(dims)
        D = orc.dense(lambda p: orc.dw(dims, U, p), n)
        ev = np.linalg.eigvals(D)
        want = []
        lx, ly, lz, lt = dims
        for a in range(lx):
            for b in range(ly):
                for c in range(lz):
                    for d in range(lt):
                        p = [2 * np.pi * a / lx, 2 * np.pi * b / ly, 2 * np.pi * c / lz, 2 * np.pi * (d + .5) / lt]
                        re = 4 - sum(np.cos(p))
                        im = np.sqrt(sum(np.sin(q) ** 2 for q in p))
                        want += [re + 1j * im] * 6 + [re - 1j * im] * 6
        want = np.array(want)
        key = lambda zz: np.lexsort((np.round(zz.imag, 8), np.round(zz.real, 8)))
        assert np.allclose(ev[key(ev)], want[key(want)], atol=1e-9)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 10), (5, 3, 7, 3)])
def test_dw_gamma5_hermiticity(orc, dims):
    """<chi, gamma5 D_W gamma5 psi> = <D_W chi, psi> on rough random links."""
    U = inputs.random_links(dims, 0.9, 5)
    psi = inputs.gaussian_spinor(dims, 6)
    chi = inputs.gaussian_spinor(dims, 7)
    lhs = vdot(chi, g5(orc.dw(dims, U, g5(psi))))
    rhs = vdot(orc.dw(dims, U, chi), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 10), (5, 3, 7, 3)])
def test_dw_gauge_covariance(orc, dims):
    """D_W[U^g](g psi) = g D_W[U] psi, U^g_mu(x) = g(x) U_mu(x) g(x+mu)^dag: every link path vs a closed form."""
    U = inputs.random_links(dims, 0.7, 21)
    g = inputs.random_su3_field(dims, 22)
    psi = inputs.gaussian_spinor(dims, 23)
    Ug = inputs.gauge_transform_links(U, g, dims)
    gpsi = np.einsum("xab,xsb->xsa", g, psi)
    lhs = orc.dw(dims, Ug, gpsi)
    rhs = np.einsum("xab,xsb->xsa", g, orc.dw(dims, U, psi))
    assert rel_err(lhs, rhs) < 1e-13


def test_dw_pure_gauge_plane_wave(orc):
    """U_mu(x) = g(x) g(x+mu)^dag: g u e^{ipx} is an eigen-plane-wave with the free symbol (transposed-link trap:
    a U <-> U^dag or row <-> column slip breaks this while keeping gamma5-hermiticity)."""
    dims = (4, 6, 4, 8)
    gam = golden_gammas()
    U, g = inputs.pure_gauge_links(dims, 31)
    rng = np.random.default_rng(3)
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    pw, p = plane_wave(dims, [1, 5, 2, 3], u)
    psi = np.einsum("xab,xsb->xsa", g, pw)
    want = np.einsum("xab,xsb->xsa", g, np.einsum("ab,xbc->xac", dw_symbol(p, gam), pw))
    assert rel_err(orc.dw(dims, U, psi), want) < 1e-13


def test_k_hermitian_and_norm_bound(dense44):
    K = dense44["K"]
    assert np.abs(K - K.conj().T).max() < 1e-14
    lam = dense44["lam"]
    assert np.abs(lam).max() <= 6.5 + 1e-12  # ||K|| <= |4 - m_w| + 4 (R5)
    assert np.abs(lam).min() > 0.3
    # +- pairing is not exact on rough links, but both signs must be there
    assert (lam > 0).sum() > 1000 and (lam < 0).sum() > 1000


def test_khat_is_gamma5_dw_shifted_scaled(orc):
    dims = (4, 4, 6, 4)
    U = inputs.random_links(dims, 0.3, 1)
    psi = inputs.gaussian_spinor(dims, 2)
    want = g5(orc.dw(dims, U, psi) - 1.5 * psi) / 6.5
    assert rel_err(orc.khat(dims, U, psi, 1.5, 6.5), want) < 1e-15


# ---------------------------------------------------------------- Chebyshev table (R6) and evaluation (eq. 2.3)

@pytest.mark.parametrize("N,eps,bound", [(101, 0.09, 6e-5), (200, 0.077, 1e-7), (400, 0.077, 5e-13), (21, 0.3, 2e-3)])
def test_chebyshev_table_approximates_sign(N, eps, bound):
    alpha = inputs.chebyshev_sign_coeffs(N, eps)
    assert alpha.shape == (N + 1,)
    assert np.all(alpha[0::2] == 0.0)
    x = np.concatenate([np.linspace(eps, 1, 4001), -np.linspace(eps, 1, 4001)])
    err = np.abs(inputs.chebyshev_eval(alpha, x) - np.sign(x)).max()
    assert err < bound
    assert np.abs(alpha).sum() < 6.0


def test_cheb_scalar_matches_numpy_chebval(orc):
    alpha = inputs.chebyshev_sign_coeffs(101, 0.09)
    for x in [-0.93, -0.2, 0.0931, 0.5, 1.0]:
        assert abs(orc.cheb_scalar(alpha, x) - inputs.chebyshev_eval(alpha, x)) < 1e-13


def test_cheb_matches_spectral_polynomial_dense(orc, dense44):
    """sum alpha_m T_m(K^) psi == W p(Lambda^) W^dag psi with the dense eigendecomposition (transposition/recurrence
    index slips show up at O(1))."""
    d = dense44
    alpha = inputs.chebyshev_sign_coeffs(101, 0.09)
    psi = inputs.gaussian_spinor(d["dims"], inputs.SEED_BASE + 100)
    pl = inputs.chebyshev_eval(alpha, d["lam"] / 6.5)
    want = (d["W"] * pl) @ (d["W"].conj().T @ psi.ravel())
    got = orc.cheb(d["dims"], d["U"], alpha, psi)
    assert rel_err(got.ravel(), want) < 1e-12
    got_c = orc.cheb(d["dims"], d["U"], alpha, psi, clenshaw=True)
    assert rel_err(got_c, got) < 1e-14


def test_cheb_low_degree_by_hand(orc):
    """N = 3 with arbitrary (also even) coefficients: a0 psi + a1 K psi + a2 (2K^2 - 1) psi + a3 (4K^3 - 3K) psi."""
    dims = (4, 4, 4, 4)
    U = inputs.random_links(dims, 0.5, 9)
    psi = inputs.gaussian_spinor(dims, 10)
    a = np.array([0.3, -1.1, 0.7, 0.45])
    k1 = orc.khat(dims, U, psi)
    k2 = orc.khat(dims, U, k1)
    k3 = orc.khat(dims, U, k2)
    want = a[0] * psi + a[1] * k1 + a[2] * (2 * k2 - psi) + a[3] * (4 * k3 - 3 * k1)
    assert rel_err(orc.cheb(dims, U, a, psi), want) < 1e-14
    assert rel_err(orc.cheb(dims, U, a, psi, clenshaw=True), want) < 1e-14


def test_sign_within_polynomial_error_of_exact_dense(orc, dense44):
    """Config 0 Tier B: ||p(K^) psi - sign(K) psi|| <= max_i |p(lam_i) - sign lam_i| ||psi||."""
    d = dense44
    eps = 0.95 * np.abs(d["lam"]).min() / 6.5
    alpha = inputs.chebyshev_sign_coeffs(101, eps)
    psi = inputs.gaussian_spinor(d["dims"], inputs.SEED_BASE + 100)
    delta = np.abs(inputs.chebyshev_eval(alpha, d["lam"] / 6.5) - np.sign(d["lam"])).max()
    assert delta < 1e-4
    got = orc.sign(d["dims"], d["U"], alpha, psi).ravel()
    exact = d["S"] @ psi.ravel()
    err = np.linalg.norm(got - exact) / np.linalg.norm(psi)
    assert err <= delta * (1 + 1e-9) + 1e-13
    assert err > 1e-9  # an approximation, not a copy of the exact answer


def test_sign_exact_on_pure_gauge_fft(orc):
    """Any-volume Tier B: pure gauge links, sign(K) psi in closed form by FFT."""
    dims = (4, 6, 4, 8)
    gam = golden_gammas()
    U, g = inputs.pure_gauge_links(dims, 41)
    psi = inputs.gaussian_spinor(dims, 42)
    exact, omega = free_sign_fft(dims, psi, gam, 1.5, g)
    eps = 0.95 * omega.min() / 6.5
    alpha = inputs.chebyshev_sign_coeffs(151, eps)
    got = orc.sign(dims, U, alpha, psi)
    x = omega.ravel() / 6.5
    delta = np.abs(inputs.chebyshev_eval(alpha, x) - 1.0).max()
    assert delta < 1e-5
    assert np.linalg.norm(got - exact) / np.linalg.norm(psi) <= delta * (1 + 1e-9) + 1e-13


def test_sign_squared_is_one(orc):
    dims = (4, 4, 4, 8)
    U = inputs.config_links(dims, 0.3, 77, stout_steps=3)
    psi = inputs.gaussian_spinor(dims, 78)
    alpha = inputs.chebyshev_sign_coeffs(201, 0.077)
    s2 = orc.sign(dims, U, alpha, orc.sign(dims, U, alpha, psi))
    assert rel_err(s2, psi) < 5e-7


# ---------------------------------------------------------------- deflation (second sum of eq. 2.3)

def test_deflation_with_exact_eigenpairs_dense(orc, dense44):
    """With exact eigenpairs the deflated map is W diag(sign lam_i [i deflated], p(lam_i) [otherwise]) W^dag.
    Coarse polynomial (N = 15) so that the deflation term is O(1), not O(1e-5)."""
    d = dense44
    nev = 20
    order = np.argsort(np.abs(d["lam"]))
    idx = order[:nev]
    lam_d = d["lam"][idx]
    phi = np.ascontiguousarray(d["W"][:, idx].T).reshape(nev, -1, 4, 3)
    alpha = inputs.chebyshev_sign_coeffs(15, 0.2)
    psi = inputs.gaussian_spinor(d["dims"], 55)
    diag = inputs.chebyshev_eval(alpha, d["lam"] / 6.5)
    assert np.abs(diag[idx] - np.sign(lam_d)).min() > 1e-3
    diag[idx] = np.sign(lam_d)
    want = (d["W"] * diag) @ (d["W"].conj().T @ psi.ravel())
    got = orc.sign(d["dims"], d["U"], alpha, psi, phi, lam_d)
    assert rel_err(got.ravel(), want) < 1e-12
    # and deflation tightens the distance to the exact sign function
    exact = d["S"] @ psi.ravel()
    e_defl = np.linalg.norm(got.ravel() - exact)
    e_plain = np.linalg.norm(orc.sign(d["dims"], d["U"], alpha, psi).ravel() - exact)
    assert e_defl < e_plain


def test_lowest_eigenpairs_match_dense(orc, dense44):
    d = dense44
    phi, lam, res = orc.lowest_eigenpairs(d["dims"], d["U"], 6)
    assert res < 1e-6
    want = d["lam"][np.argsort(np.abs(d["lam"]))[:6]]
    assert np.allclose(np.sort(np.abs(lam)), np.sort(np.abs(want)), atol=1e-7)


# ---------------------------------------------------------------- overlap operator (eq. 2.1)

def test_overlap_dense_properties(orc, dense44):
    d = dense44
    dims, U = d["dims"], d["U"]
    n = d["K"].shape[0]
    eps = 0.95 * np.abs(d["lam"]).min() / 6.5
    alpha = inputs.chebyshev_sign_coeffs(401, eps)  # delta ~ 1e-13: "exact" polynomial
    psi = inputs.gaussian_spinor(dims, 61)
    G5m = np.tile(np.repeat(G5, 3), n // 12)
    for mu in (0.0, 0.1):
        Dex = 0.5 * ((1 + mu) * np.eye(n) + (1 - mu) * (G5m[:, None] * d["S"]))
        got = orc.overlap(dims, U, alpha, mu, psi)
        assert rel_err(got.ravel(), Dex @ psi.ravel()) < 1e-11
        got_d = orc.overlap(dims, U, alpha, mu, psi, dagger=True)
        assert rel_err(got_d.ravel(), Dex.conj().T @ psi.ravel()) < 1e-11
        # D^dag = gamma5 D gamma5
        assert rel_err(got_d, g5(orc.overlap(dims, U, alpha, mu, g5(psi)))) < 1e-13
    # spectrum of the exact D[mu] on the circle centre (1+mu)/2 radius (1-mu)/2
    mu = 0.1
    ev = np.linalg.eigvals(0.5 * ((1 + mu) * np.eye(n) + (1 - mu) * (G5m[:, None] * d["S"])))
    assert np.abs(np.abs(ev - (1 + mu) / 2) - (1 - mu) / 2).max() < 1e-10
    # mu = 1: D = 1
    assert rel_err(orc.overlap(dims, U, alpha, 1.0, psi), psi) < 1e-15


def test_ginsparg_wilson(orc):
    """{gamma5, D} = 2 D gamma5 D at mu = 0, up to the polynomial error: residual = 1/2 gamma5 (1 - s^2) psi."""
    dims = (4, 4, 4, 8)
    U = inputs.config_links(dims, 0.3, 77, stout_steps=3)
    psi = inputs.gaussian_spinor(dims, 79)
    for N, bound in [(101, 2e-3), (201, 5e-7), (401, 1e-12)]:
        alpha = inputs.chebyshev_sign_coeffs(N, 0.077)
        D = lambda v: orc.overlap(dims, U, alpha, 0.0, v)
        lhs = g5(D(psi)) + D(g5(psi))
        rhs = 2 * D(g5(D(psi)))
        assert np.linalg.norm(lhs - rhs) / np.linalg.norm(psi) < bound


# ---------------------------------------------------------------- CG on D^dag D

def test_cg_against_dense_solve(orc, dense44):
    d = dense44
    dims, U = d["dims"], d["U"]
    n = d["K"].shape[0]
    mu = 0.05
    alpha = inputs.chebyshev_sign_coeffs(101, 0.95 * np.abs(d["lam"]).min() / 6.5)
    # the operator CG actually inverts: D built from the SAME polynomial, densely
    pl = inputs.chebyshev_eval(alpha, d["lam"] / 6.5)
    Sp = (d["W"] * pl) @ d["W"].conj().T
    G5m = np.tile(np.repeat(G5, 3), n // 12)
    Dm = 0.5 * ((1 + mu) * np.eye(n) + (1 - mu) * (G5m[:, None] * Sp))
    A = Dm.conj().T @ Dm
    b = inputs.gaussian_spinor(dims, 91)
    xs = np.linalg.solve(A, b.ravel())
    x, it, rel = orc.cg(dims, U, alpha, mu, b, 1e-10, 500)
    assert 5 < it < 500
    assert rel < 1.5e-10
    assert np.linalg.norm(x.ravel() - xs) / np.linalg.norm(xs) < 1e-7
    assert np.vdot(x.ravel(), A @ x.ravel()).real > 0
    # A-norm of the error decreases monotonically with the iteration count
    errs = []
    for k in (2, 4, 8, 16):
        xk, itk, _ = orc.cg(dims, U, alpha, mu, b, 0.0, k)
        assert itk == k
        e = xk.ravel() - xs
        errs.append(np.vdot(e, A @ e).real)
    assert all(e1 > e2 for e1, e2 in zip(errs, errs[1:]))


# ---------------------------------------------------------------- chiral-sector D^dag D (reading R23)

def test_chiral_sector_operator_dense(orc, dense44):
    """orc_chiral_op against the plain definition: P_c D^dag D P_c with D = 1/2 (1 + mu + (1 - mu) gamma5 S) built densely
    from the EXACT sign matrix S of the eigendecomposition (S^2 = 1).  With a delta ~ 1e-13 polynomial the two agree to
    1e-11: pins the constants 1/2 (1 + mu^2), c/2 (1 - mu^2), both chiralities and the projections; D^dag D commutes
    with gamma5."""
    d = dense44
    dims, U = d["dims"], d["U"]
    n = d["K"].shape[0]
    alpha = inputs.chebyshev_sign_coeffs(401, 0.95 * np.abs(d["lam"]).min() / 6.5)
    G5m = np.tile(np.repeat(G5, 3), n // 12)
    v = inputs.gaussian_spinor(dims, 67)  # NOT chiral: the routine projects
    for mu in (0.0, 0.05, 0.3):
        Dex = 0.5 * ((1 + mu) * np.eye(n) + (1 - mu) * (G5m[:, None] * d["S"]))
        A = Dex.conj().T @ Dex
        assert np.abs(A * G5m[None, :] - G5m[:, None] * A).max() < 1e-12      # [D^dag D, gamma5] = 0 for the exact sign
        for c in (+1, -1):
            Pc = 0.5 * (1 + c * G5m)
            want = Pc * (A @ (Pc * v.ravel()))
            got = orc.chiral_op(dims, U, alpha, mu, c, v)
            assert rel_err(got.ravel(), want) < 1e-11
            assert np.abs((1 - Pc) * got.ravel()).max() == 0.0                 # stays in the sector exactly
            # and against the oracle's own two-apply D^dag D on a chiral vector
            pv = (Pc * v.ravel()).reshape(v.shape)
            two = orc.overlap(dims, U, alpha, mu, orc.overlap(dims, U, alpha, mu, pv), dagger=True)
            assert rel_err(got, two) < 1e-11


def test_chiral_sector_error_term(orc, dense44):
    """With a POOR polynomial (delta = max |p(lambda^) - sign| over the dense spectrum) the sector operator differs from
    P_c D^dag D P_c (the oracle's two applies, same polynomial) by exactly 1/4 (1 - mu)^2 P_c (s^2 - 1) P_c: norm <=
    1/4 (1 - mu)^2 (2 delta + delta^2) ||v||, and it is not accidentally zero."""
    d = dense44
    dims, U = d["dims"], d["U"]
    n = d["K"].shape[0]
    alpha = inputs.chebyshev_sign_coeffs(41, 0.95 * np.abs(d["lam"]).min() / 6.5)
    delta = np.abs(inputs.chebyshev_eval(alpha, d["lam"] / 6.5) - np.sign(d["lam"])).max()
    assert 1e-4 < delta < 0.5
    G5m = np.tile(np.repeat(G5, 3), n // 12)
    mu = 0.1
    for c in (+1, -1):
        Pc = 0.5 * (1 + c * G5m)
        pv = (Pc * inputs.gaussian_spinor(dims, 68).ravel()).reshape(-1, 4, 3)
        two = orc.overlap(dims, U, alpha, mu, orc.overlap(dims, U, alpha, mu, pv), dagger=True)
        got = orc.chiral_op(dims, U, alpha, mu, c, pv)
        diff = np.linalg.norm(Pc * two.ravel() - got.ravel()) / np.linalg.norm(pv.ravel())
        assert 1e-8 < diff <= 0.25 * (1 - mu) ** 2 * (2 * delta + delta * delta) * 1.0000001
        # the predicted form of the difference, through the oracle's own sign function
        s2 = orc.sign(dims, U, alpha, orc.sign(dims, U, alpha, pv))
        pred = 0.25 * (1 - mu) ** 2 * (Pc * (s2.ravel() - pv.ravel()))
        assert rel_err(Pc * two.ravel() - got.ravel(), pred) < 1e-9


def test_cg_chiral_against_dense_solve(orc, dense44):
    """orc_cg_chiral vs numpy's dense solve of the sector system built from the SAME polynomial (so the comparison is
    limited by the CG tolerance only), and vs the full D^dag D solve on a chiral source (limited by kappa * delta)."""
    d = dense44
    dims, U = d["dims"], d["U"]
    n = d["K"].shape[0]
    mu = 0.05
    alpha = inputs.chebyshev_sign_coeffs(101, 0.95 * np.abs(d["lam"]).min() / 6.5)
    pl = inputs.chebyshev_eval(alpha, d["lam"] / 6.5)
    Sp = (d["W"] * pl) @ d["W"].conj().T
    G5m = np.tile(np.repeat(G5, 3), n // 12)
    b = inputs.gaussian_spinor(dims, 92)
    for c in (+1, -1):
        Pc = 0.5 * (1 + c * G5m)
        idx = np.nonzero(Pc)[0]
        Ac = 0.5 * (1 + mu * mu) * np.eye(len(idx)) + 0.5 * c * (1 - mu * mu) * Sp[np.ix_(idx, idx)]
        xs = np.zeros(n, complex)
        xs[idx] = np.linalg.solve(Ac, b.ravel()[idx])
        x, it, rel = orc.cg_chiral(dims, U, alpha, mu, c, b, 1e-10, 500)
        assert 5 < it < 500 and rel < 1.5e-10
        assert np.abs((1 - Pc) * x.ravel()).max() == 0.0
        assert np.linalg.norm(x.ravel() - xs) / np.linalg.norm(xs) < 1e-7
        # the full operator on the chiral source: same solution up to the polynomial's s^2 - 1 (delta ~ 3e-5 here)
        xf, _, _ = orc.cg(dims, U, alpha, mu, (Pc * b.ravel()).reshape(b.shape), 1e-10, 500)
        assert np.linalg.norm(xf.ravel() - x.ravel()) / np.linalg.norm(x.ravel()) < 1e-2
        # fixed iteration count honoured; zero sector source -> zero iterations
        xk, itk, _ = orc.cg_chiral(dims, U, alpha, mu, c, b, 0.0, 7)
        assert itk == 7
        x0, it0, rel0 = orc.cg_chiral(dims, U, alpha, mu, c, ((1 - Pc) * b.ravel()).reshape(b.shape), 1e-10, 50)
        assert it0 == 0 and rel0 == 0.0 and not x0.any()


# ---------------------------------------------------------------- input generators

def test_links_unitary_and_smearing_raises_plaquette():
    dims = (4, 4, 4, 6)
    U = inputs.random_links(dims, 0.3, 3)
    I = np.eye(3)
    assert np.abs(U @ np.conj(np.swapaxes(U, -1, -2)) - I).max() < 1e-13
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-13
    p0 = inputs.plaquette(U, dims)
    assert 0.74 < p0 < 0.83
    prev, Us = p0, U
    for _ in range(3):
        Us = inputs.stout_smear(Us, dims, 0.1, 1)
        p = inputs.plaquette(Us, dims)
        assert p > prev
        prev = p
    assert prev > 0.99
    assert np.abs(Us @ np.conj(np.swapaxes(Us, -1, -2)) - I).max() < 1e-12
    assert np.abs(np.linalg.det(Us) - 1).max() < 1e-12
    # smearing is gauge covariant
    g = inputs.random_su3_field(dims, 4)
    a = inputs.stout_smear(inputs.gauge_transform_links(U, g, dims), dims, 0.1, 1)
    b = inputs.gauge_transform_links(inputs.stout_smear(U, dims, 0.1, 1), g, dims)
    assert np.abs(a - b).max() < 1e-12
    Upg, _ = inputs.pure_gauge_links(dims, 8)
    assert abs(inputs.plaquette(Upg, dims) - 1) < 1e-13


def test_deflation_with_closed_form_eigenpairs_pure_gauge(orc):
    """eq. 2.3 with TRUE eigenpairs at a volume with no dense matrix: on a pure gauge the lowest eigenpairs of K are
    gauge-rotated plane waves (tests/closed_forms.py).  (i) the oracle's K reproduces them; (ii) with them deflated,
    sign(K) phi_i = sign(lambda_i) phi_i to rounding even with a deliberately poor polynomial, while without deflation
    the error is the polynomial's |1 - p(lambda^_i)|; (iii) on a random psi the deflated sum is within the polynomial's
    error on the REST of the spectrum of the FFT closed form."""
    dims, nev = (4, 4, 6, 8), 24
    U, g = inputs.pure_gauge_links(dims, 51)
    G = golden_gammas()
    phi, lam = lowest_pure_gauge_eigenpairs(dims, g, G, nev)
    for i in (0, 7, 23):
        assert np.linalg.norm(orc.khat(dims, U, phi[i], 1.5, 6.5) * 6.5 - lam[i] * phi[i]) < 1e-13
    alpha = inputs.chebyshev_sign_coeffs(11, 0.3)          # poor on purpose: |lambda^| ~ 0.09 < eps = 0.3
    perr = np.abs(inputs.chebyshev_eval(alpha, np.abs(lam) / 6.5) - 1.0)
    assert perr.min() > 0.05
    for i in (0, 11, 23):
        with_defl = orc.sign(dims, U, alpha, phi[i], phi, lam)
        without = orc.sign(dims, U, alpha, phi[i])
        assert np.linalg.norm(with_defl - np.sign(lam[i]) * phi[i]) < 1e-13
        assert abs(np.linalg.norm(without - np.sign(lam[i]) * phi[i]) - perr[i]) < 1e-10
    psi = inputs.gaussian_spinor(dims, 52)
    exact, omega = free_sign_fft(dims, psi, G, 1.5, g)
    rest = np.sort(omega.ravel())[nev // 12:]              # |lambda| of the modes that are not deflated (12 per momentum)
    alpha = inputs.chebyshev_sign_coeffs(81, 0.95 * rest.min() / 6.5)
    delta = np.abs(inputs.chebyshev_eval(alpha, rest / 6.5) - 1.0).max()
    got = orc.sign(dims, U, alpha, psi, phi, lam)
    assert np.linalg.norm(got - exact) <= 1.05 * delta * np.linalg.norm(psi) + 1e-12
