"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by element on the same
seeded inputs.  Tolerances are BASELINE.json north_star's: 1e-12 (fp64 D_W), 1e-10 (fp64 sign / overlap /
fixed-iteration CG), 1e-5 (fp32), relative L2 over the whole field."""
import numpy as np
import pytest

from paper_1510_06897_b200 import inputs
from tests.conftest import rel_err

pytestmark = pytest.mark.gpu

TOL_DW, TOL_OVL, TOL_F32 = 1e-12, 1e-10, 1e-5
G5 = np.array([1.0, 1.0, -1.0, -1.0])


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def api(torch):
    from paper_1510_06897_b200 import api, binding
    binding.load_library()  # fail loudly if the CUDA extension is missing
    return api


def dev(torch, a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t.to(dtype) if dtype is not None else t


def host(t):
    return t.detach().cpu().numpy()


def rough_alpha(n, seed=5):
    """A generic (not sign-like) table with non-zero even AND odd entries: exercises every accumulate branch."""
    rng = np.random.default_rng(seed)
    a = rng.standard_normal(n + 1) / (1 + np.arange(n + 1))
    if n >= 5:
        a[4] = 0.0
    return a


# even, extent-2, non-cubic, ragged tiles (V % 128 != 0) and odd extents (the forward and backward wrap of an odd direction differ)
DW_DIMS = [(4, 4, 4, 4), (2, 2, 2, 2), (4, 6, 8, 10), (6, 4, 2, 8), (8, 8, 8, 8), (10, 6, 4, 12), (8, 8, 8, 32), (3, 5, 4, 6), (5, 3, 7, 3)]


@pytest.mark.parametrize("dims", DW_DIMS)
@pytest.mark.parametrize("recon", [18, 12])
def test_dw_fp64(torch, api, orc, dims, recon):
    U = inputs.random_links(dims, 0.7, 100 + sum(dims))
    psi = inputs.gaussian_spinor(dims, 200 + sum(dims))
    want = orc.dw(dims, U, psi)
    with api.Overlap(dims, dev(torch, U), "f64", recon) as op:
        got = host(op.dw(dev(torch, psi)))
    assert rel_err(got, want) < TOL_DW
    assert np.abs(got - want).max() < 1e-12 * np.abs(want).max() * 10


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 10), (8, 8, 8, 32), (5, 3, 7, 3)])
@pytest.mark.parametrize("recon", [18, 12])
def test_dw_fp32(torch, api, orc, dims, recon):
    U = inputs.random_links(dims, 0.7, 31)
    psi = inputs.gaussian_spinor(dims, 32)
    want = orc.dw(dims, U, psi)
    with api.Overlap(dims, dev(torch, U), "f32", recon) as op:
        got = host(op.dw(dev(torch, psi, torch.complex64)))
    assert got.dtype == np.complex64
    assert rel_err(got.astype(np.complex128), want) < TOL_F32


def test_khat_fp64(torch, api, orc):
    dims = (4, 6, 8, 10)
    U = inputs.random_links(dims, 0.3, 1)
    psi = inputs.gaussian_spinor(dims, 2)
    with api.Overlap(dims, dev(torch, U), m_w=1.4, lambda_max=6.1) as op:
        got = host(op.khat(dev(torch, psi)))
    assert rel_err(got, orc.khat(dims, U, psi, 1.4, 6.1)) < TOL_DW


RECS = ["clenshaw", "forward"]  # both evaluation orders of the polynomial sum (ovl_set_recurrence)


@pytest.mark.parametrize("dims,N", [((4, 4, 4, 4), 1), ((4, 4, 4, 4), 2), ((4, 4, 4, 4), 3), ((4, 4, 4, 4), 4), ((4, 4, 4, 4), 5),
                                    ((4, 6, 8, 10), 24), ((6, 4, 2, 8), 37)])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("rec", RECS)
def test_sign_generic_coefficients(torch, api, orc, dims, N, recon, rec):
    """Every order accumulates (even and odd alpha non-zero, one zero in the middle): recurrence indexing, including
    the short tables N = 1..5 where the Clenshaw start-up launches (b_{N-1}, b_{N-2}) and the final one overlap."""
    U = inputs.random_links(dims, 0.5, 9)
    psi = inputs.gaussian_spinor(dims, 10)
    alpha = rough_alpha(N)
    want = orc.sign(dims, U, alpha, psi)
    with api.Overlap(dims, dev(torch, U), "f64", recon) as op:
        op.set_recurrence(rec)
        assert op.set_chebyshev(alpha) == N
        got = host(op.sign(dev(torch, psi)))
    assert rel_err(got, want) < TOL_OVL


@pytest.mark.parametrize("rec", RECS)
@pytest.mark.parametrize("zeros", [(0,), (0, 2), (1, 3), (0, 1, 2, 3, 4, 5), (5, 7), (6, 8)])
def test_sign_with_vanishing_coefficients(torch, api, orc, rec, zeros):
    """Tables with zeros in the places the recurrences special-case: alpha_0 (no psi term in the last Clenshaw launch),
    alpha_{N-1} and alpha_{N-2} - alpha_N (start-up launches), runs of zeros (orders that skip the psi / acc stream)."""
    dims, N = (4, 4, 4, 6), 8
    U = inputs.random_links(dims, 0.5, 19)
    psi = inputs.gaussian_spinor(dims, 20)
    alpha = rough_alpha(N, seed=11)
    for z in zeros:
        alpha[z] = 0.0
    if zeros == (6, 8):
        alpha[6], alpha[8] = 0.25, 0.25  # alpha_{N-2} - alpha_N = 0
    want = orc.sign(dims, U, alpha, psi)
    with api.Overlap(dims, dev(torch, U)) as op:
        op.set_recurrence(rec)
        op.set_chebyshev(alpha)
        got = host(op.sign(dev(torch, psi)))
    assert rel_err(got, want) < TOL_OVL


@pytest.mark.parametrize("rec", RECS)
def test_trailing_zero_coefficients_are_skipped(torch, api, orc, rec):
    dims = (4, 4, 4, 4)
    U = inputs.random_links(dims, 0.5, 9)
    psi = inputs.gaussian_spinor(dims, 10)
    alpha = np.concatenate([rough_alpha(9), np.zeros(5)])
    with api.Overlap(dims, dev(torch, U)) as op:
        op.set_recurrence(rec)
        assert op.set_chebyshev(alpha) == 9  # reading R7
        got = host(op.sign(dev(torch, psi)))
    assert rel_err(got, orc.sign(dims, U, alpha, psi)) < TOL_OVL


def test_config0_overlap_4x4(torch, api, orc, dense44):
    """BASELINE config 0: 4^4, U = exp(0.3 i H), D_W and D[0.1] with degree 101, no deflation; Tier A vs the oracle
    and Tier B vs the dense exact sign function (error bounded by the polynomial's error on the spectrum)."""
    d = dense44
    dims, U = d["dims"], d["U"]
    psi = inputs.gaussian_spinor(dims, inputs.SEED_BASE + 100)
    eps = 0.95 * np.abs(d["lam"]).min() / 6.5
    alpha = inputs.chebyshev_sign_coeffs(101, eps)
    with api.Overlap(dims, dev(torch, U)) as op:
        assert op.set_chebyshev(alpha) == 101
        p = dev(torch, psi)
        assert rel_err(host(op.dw(p)), orc.dw(dims, U, psi)) < TOL_DW
        got = host(op.overlap(p, 0.1))
        got_d = host(op.overlap(p, 0.1, dagger=True))
        s = host(op.sign(p))
    assert rel_err(got, orc.overlap(dims, U, alpha, 0.1, psi)) < TOL_OVL
    assert rel_err(got_d, orc.overlap(dims, U, alpha, 0.1, psi, dagger=True)) < TOL_OVL
    delta = np.abs(inputs.chebyshev_eval(alpha, d["lam"] / 6.5) - np.sign(d["lam"])).max()
    exact = d["S"] @ psi.ravel()
    assert np.linalg.norm(s.ravel() - exact) / np.linalg.norm(psi) <= delta * (1 + 1e-6) + 1e-12
    n = d["K"].shape[0]
    g5m = np.tile(np.repeat(G5, 3), n // 12)
    dex = 0.5 * (1.1 * psi.ravel() + 0.9 * g5m * exact)
    assert np.linalg.norm(got.ravel() - dex) / np.linalg.norm(dex) < 2 * delta


@pytest.mark.parametrize("prec,tol", [("f64", TOL_OVL), ("f32", TOL_F32)])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("rec", RECS)
def test_deflated_sign_and_overlap(torch, api, orc, prec, tol, recon, rec):
    """eq. 2.3 complete, with generic orthonormal vectors and 'eigenvalues' of both signs (reading R10: a well-defined
    linear map for any (phi_i, lambda_i)); coarse polynomial so the deflation term is O(1)."""
    dims = (4, 6, 8, 10)
    nev = 7
    U = inputs.config_links(dims, 0.3, 3, stout_steps=1)
    psi = inputs.gaussian_spinor(dims, 4)
    phi = inputs.orthonormal_vectors(dims, nev, 5)
    lam = np.array([0.31, -0.33, 0.35, -0.4, 0.42, 0.5, -0.55])
    alpha = inputs.chebyshev_sign_coeffs(31, 0.2)
    want_s = orc.sign(dims, U, alpha, psi, phi, lam)
    plain = orc.sign(dims, U, alpha, psi)
    assert rel_err(want_s, plain) > 1e-3  # deflation does something here
    cd = torch.complex128 if prec == "f64" else torch.complex64
    with api.Overlap(dims, dev(torch, U), prec, recon) as op:
        op.set_recurrence(rec)
        op.set_chebyshev(alpha)
        op.set_deflation(dev(torch, phi), lam)
        p = dev(torch, psi, cd)
        assert rel_err(host(op.sign(p)), want_s) < tol
        for mu, dag in [(0.01, False), (0.05, True)]:
            want = orc.overlap(dims, U, alpha, mu, psi, phi, lam, dagger=dag)
            assert rel_err(host(op.overlap(p, mu, dagger=dag)), want) < tol
        op.set_deflation(None, [])  # switch deflation off again
        assert rel_err(host(op.sign(p)), plain) < tol


@pytest.mark.parametrize("rec", RECS)
def test_config1_shape_8x8x8x32_degree200_nev20(torch, api, orc, rec):
    """BASELINE config 1 shape: 8^3 x 32, smeared links, mu = 0.01, degree 200, 20 deflation vectors (generic
    orthonormal stand-ins for the Lanczos vectors, DESIGN.md input recipe); several tiles + ragged last block."""
    dims = (8, 8, 8, 32)
    U = inputs.config_links(dims, 0.3, inputs.SEED_BASE + 1, stout_steps=3)
    psi = inputs.gaussian_spinor(dims, inputs.SEED_BASE + 101)
    phi = inputs.orthonormal_vectors(dims, 20, inputs.SEED_BASE + 201)
    lam = 0.505 * np.where(np.arange(20) % 2 == 0, 1.0, -1.0) * (1 + 0.001 * np.arange(20))
    alpha = inputs.chebyshev_sign_coeffs(200, 0.95 * 0.505 / 6.5)
    want = orc.overlap(dims, U, alpha, 0.01, psi, phi, lam)
    with api.Overlap(dims, dev(torch, U)) as op:
        op.set_recurrence(rec)
        assert op.set_chebyshev(alpha) == 199  # degree 200 table, alpha_200 = 0 (reading R7)
        p = dev(torch, psi)
        s2 = host(op.sign(op.sign(p)))  # before the stand-in vectors are set: the polynomial alone
        op.set_deflation(dev(torch, phi), lam)
        got = host(op.overlap(p, 0.01))
    assert rel_err(got, want) < TOL_OVL
    # sign^2 = 1 up to the polynomial error: ||s^2 psi - psi|| <= (2 delta + delta^2) ||psi|| (SURVEY §8(c) pins), delta =
    # max |p - 1| on [eps, 1]; the stand-in vectors are not eigenvectors, so the bound is checked without them
    delta = np.abs(inputs.chebyshev_eval(alpha, np.linspace(0.95 * 0.505 / 6.5, 1.0, 20001)) - 1.0).max()
    assert rel_err(s2, psi) <= 2 * delta + delta * delta + 1e-12


def test_cg_fixed_iterations_and_to_tolerance(torch, api, orc, dense44):
    d = dense44
    dims, U = d["dims"], d["U"]
    mu = 0.05
    alpha = inputs.chebyshev_sign_coeffs(101, 0.95 * np.abs(d["lam"]).min() / 6.5)
    b = inputs.gaussian_spinor(dims, 91)
    with api.Overlap(dims, dev(torch, U)) as op:
        op.set_chebyshev(alpha)
        bd = dev(torch, b)
        # (iii) of reading R14: fixed iteration count, no stopping test
        xk, itk, _, ok = op.cg(bd, mu, tol=0.0, maxiter=10)
        want_k, it_o, _ = orc.cg(dims, U, alpha, mu, b, 0.0, 10)
        assert itk == it_o == 10 and ok
        assert rel_err(host(xk), want_k) < TOL_OVL
        # (i) + (ii): to tolerance
        x, it, rel, ok = op.cg(bd, mu, tol=1e-8, maxiter=500)
        xo, ito, relo = orc.cg(dims, U, alpha, mu, b, 1e-8, 500)
        assert ok and abs(it - ito) <= 2
        assert rel < 1.05e-8 and relo < 1.05e-8
        assert rel_err(host(x), xo) < 1e-5
        # not converged -> OVL_ENOTCONV surfaced as ok = False, x = last iterate
        x3, it3, rel3, ok3 = op.cg(bd, mu, tol=1e-8, maxiter=3)
        assert it3 == 3 and not ok3 and rel3 > 1e-8
        want3, _, _ = orc.cg(dims, U, alpha, mu, b, 1e-8, 3)
        assert rel_err(host(x3), want3) < TOL_OVL


def test_cg_with_deflation_8x8x8x8(torch, api, orc):
    dims = (8, 8, 8, 8)
    U = inputs.config_links(dims, 0.3, 13, stout_steps=2)
    b = inputs.gaussian_spinor(dims, 14)
    phi = inputs.orthonormal_vectors(dims, 5, 15)
    lam = np.array([0.5, -0.51, 0.52, -0.53, 0.54])
    alpha = inputs.chebyshev_sign_coeffs(61, 0.075)
    with api.Overlap(dims, dev(torch, U)) as op:
        op.set_chebyshev(alpha)
        op.set_deflation(dev(torch, phi), lam)
        x, it, rel, ok = op.cg(dev(torch, b), 0.2, tol=0.0, maxiter=6)
    want, _, relo = orc.cg(dims, U, alpha, 0.2, b, 0.0, 6, phi, lam)
    assert rel_err(host(x), want) < TOL_OVL
    assert abs(rel - relo) < 1e-9


def test_host_pointers_and_native_fields(torch, api, orc):
    """numpy (host) in/out through the C-ABI staging path; native import/export is an exact round trip."""
    dims = (4, 6, 8, 10)
    U = inputs.random_links(dims, 0.4, 51)
    psi = inputs.gaussian_spinor(dims, 52)
    alpha = rough_alpha(12)
    with api.Overlap(dims, U) as op:  # host links
        op.set_chebyshev(alpha)
        got = op.overlap(psi, 0.1)  # host spinor in, host spinor out
        assert isinstance(got, np.ndarray)
        assert rel_err(got, orc.overlap(dims, U, alpha, 0.1, psi)) < TOL_OVL
        nat = op.to_native(dev(torch, psi))
        back = host(op.from_native(nat))
        assert np.array_equal(back, psi)
        nat_out = op.native_empty()
        op.dw_native(nat, nat_out)
        assert rel_err(host(op.from_native(nat_out)), orc.dw(dims, U, psi)) < TOL_DW
        op.overlap_native(nat, nat_out, 0.1)
        assert np.array_equal(host(op.from_native(nat_out)), got)
        phi = inputs.orthonormal_vectors(dims, 3, 53)
        lam = [0.4, -0.5, 0.6]
        op.set_deflation(phi, lam)  # host eigenvectors
        assert rel_err(op.sign(psi), orc.sign(dims, U, alpha, psi, phi, lam)) < TOL_OVL


@pytest.mark.parametrize("rec", RECS)
def test_graph_replay_equals_direct_launches(torch, api, orc, rec):
    """On a real (non-default) stream the polynomial loop is replayed from a CUDA graph; results must be bit-identical
    to direct launches, also after the table, the kernel parameters or the source buffer change (graph invalidation)."""
    dims = (4, 6, 8, 10)
    U = inputs.random_links(dims, 0.4, 41)
    psi = inputs.gaussian_spinor(dims, 42)
    chi = inputs.gaussian_spinor(dims, 43)
    a1, a2 = rough_alpha(17, seed=3), rough_alpha(12, seed=4)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        with api.Overlap(dims, dev(torch, U), stream=side) as op:
            op.set_recurrence(rec)
            res = {}
            for graphs in (True, False):
                op.set_graphs(graphs)
                out = []
                op.set_chebyshev(a1)
                p, q = dev(torch, psi), dev(torch, chi)
                out.append(host(op.sign(p)))
                out.append(host(op.sign(p)))      # replay
                out.append(host(op.sign(q)))
                op.set_chebyshev(a2)              # new table -> new launch sequence
                out.append(host(op.sign(p)))
                B_ = __import__("paper_1510_06897_b200.binding", fromlist=["x"])
                B_.ovl_set_kernel(op.ctx, 1.4, 6.2)
                out.append(host(op.sign(p)))
                B_.ovl_set_kernel(op.ctx, 1.5, 6.5)
                nat_in, nat_out = op.to_native(p), op.native_empty()
                op.overlap_native(nat_in, nat_out, 0.03)
                out.append(host(op.from_native(nat_out)))
                res[graphs] = out
            side.synchronize()
    for g, d in zip(res[True], res[False]):
        assert np.array_equal(g, d)
    assert rel_err(res[True][0], orc.sign(dims, U, a1, psi)) < TOL_OVL
    assert rel_err(res[True][3], orc.sign(dims, U, a2, psi)) < TOL_OVL
    assert rel_err(res[True][4], orc.sign(dims, U, a2, psi, m_w=1.4, lambda_max=6.2)) < TOL_OVL


@pytest.mark.parametrize("prec,tol", [("f64", TOL_OVL), ("f32", TOL_F32)])
@pytest.mark.parametrize("rec", RECS)
@pytest.mark.parametrize("nrhs,dagger", [(1, False), (3, False), (5, True), (12, False)])
def test_multi_rhs_overlap(torch, api, orc, prec, tol, rec, nrhs, dagger):
    """ovl_overlap_multi: every right-hand side against the oracle, and bit-identical to the
    single-right-hand-side call (same arithmetic per site; only the CTA -> (tile, rhs) map differs)."""
    dims = (4, 6, 8, 10)   # 1920 sites = 15 tiles of 128
    nev = 4
    U = inputs.config_links(dims, 0.3, 51, stout_steps=1)
    phi = inputs.orthonormal_vectors(dims, nev, 52)
    lam = np.array([0.31, -0.33, 0.35, -0.4])
    alpha = inputs.chebyshev_sign_coeffs(21, 0.2)
    psis = np.stack([inputs.gaussian_spinor(dims, 60 + r) for r in range(nrhs)])
    cd = torch.complex128 if prec == "f64" else torch.complex64
    with api.Overlap(dims, dev(torch, U), prec) as op:
        op.set_recurrence(rec)
        op.set_chebyshev(alpha)
        op.set_deflation(dev(torch, phi), lam)
        p = dev(torch, psis, cd)
        got = op.overlap_multi(p, 0.02, dagger=dagger)
        singles = torch.stack([op.overlap(p[r].contiguous(), 0.02, dagger=dagger) for r in range(nrhs)])
        assert torch.equal(got, singles)
        again = op.overlap_multi(p, 0.02, dagger=dagger)       # workspace already grown, graph replay on side streams
        assert torch.equal(got, again)
    got = host(got)
    for r in range(nrhs):
        want = orc.overlap(dims, U, alpha, 0.02, psis[r], phi, lam, dagger=dagger)
        assert rel_err(got[r].astype(np.complex128), want) < tol, r


def test_cg_multi_lockstep(torch, api, orc):
    """ovl_cg_multi: 3 systems with very different right-hand sides (one is a constant vector that converges at a
    different iteration and must be frozen).  Each solution is bit-identical to the single-system ovl_cg, iteration
    counts agree, true residuals <= tol; a fixed-iteration run matches the oracle CG at 1e-10."""
    dims = (4, 4, 4, 8)
    U = inputs.config_links(dims, 0.3, 77, stout_steps=1)
    alpha = inputs.chebyshev_sign_coeffs(41, 0.09)
    phi = inputs.orthonormal_vectors(dims, 3, 78)
    lam = np.array([0.45, -0.47, 0.5])
    b = np.stack([inputs.gaussian_spinor(dims, 79), 1e-3 * inputs.gaussian_spinor(dims, 80), inputs.gaussian_spinor(dims, 81)])
    b[2] = b[2] * 0 + 1.0          # constant vector: a different (smaller) Krylov space
    mu = 0.2
    with api.Overlap(dims, dev(torch, U)) as op:
        op.set_chebyshev(alpha)
        op.set_deflation(dev(torch, phi), lam)
        bd = dev(torch, b)
        x, its, rels, ok = op.cg_multi(bd, mu, tol=1e-9, maxiter=500)
        assert ok and len(its) == 3
        for r in range(3):
            xs, it1, rel1, ok1 = op.cg(bd[r].contiguous(), mu, tol=1e-9, maxiter=500)
            assert ok1 and it1 == its[r]
            assert torch.equal(xs, x[r])
            assert rels[r] <= 1.05e-9 and abs(rels[r] - rel1) <= 1e-12
        assert len(set(its)) > 1       # they did not all stop together: freezing was exercised
        x5, its5, _, _ = op.cg_multi(bd, mu, tol=0.0, maxiter=5)
        assert its5 == [5, 5, 5]
        xnc, itn, reln, okn = op.cg_multi(bd, mu, tol=1e-9, maxiter=3)
        assert not okn and itn == [3, 3, 3]
    x5 = host(x5)
    for r in range(3):
        xo, _, _ = orc.cg(dims, U, alpha, mu, b[r], 0.0, 5, phi, lam)
        assert rel_err(x5[r], xo) < TOL_OVL


def test_cg_mixed_precision(torch, api, orc):
    """ovl_cg_mixed: fp32 inner solves, fp64 outer residuals.  Reaches a true fp64 residual of 1e-11 -- far below what the
    fp32 path alone can represent -- and agrees with the oracle's fp64 CG solution (R14: both are solutions to their
    tolerance; kappa * tol bounds the difference).  Also with a lower-degree ("relaxed") inner polynomial."""
    from paper_1510_06897_b200 import binding as B
    dims = (4, 4, 4, 8)
    U = inputs.config_links(dims, 0.3, 177, stout_steps=1)
    alpha = inputs.chebyshev_sign_coeffs(61, 0.09)
    alpha_lo = inputs.chebyshev_sign_coeffs(31, 0.09)
    phi = inputs.orthonormal_vectors(dims, 3, 178)
    lam = np.array([0.45, -0.47, 0.5])
    b = inputs.gaussian_spinor(dims, 179)
    mu = 0.2
    xo, ito, relo = orc.cg(dims, U, alpha, mu, b, 1e-11, 500, phi, lam)
    with api.Overlap(dims, dev(torch, U), "f64") as op, api.Overlap(dims, dev(torch, U), "f32") as op32:
        for o in (op, op32):
            o.set_chebyshev(alpha)
            o.set_deflation(dev(torch, phi), lam)
        bd = dev(torch, b)
        x, no, ni, rel, ok = op.cg_mixed(op32, bd, mu, tol=1e-11, inner_tol=1e-4)
        assert ok and rel <= 1e-11 and 2 <= no <= 6 and ni >= ito // 2
        assert rel_err(host(x), xo) < 1e-8
        # the residual reported is the true one: recompute it through the public fp64 operator
        ax = op.overlap(op.overlap(x, mu), mu, dagger=True)
        assert abs(float(torch.linalg.norm(bd - ax) / torch.linalg.norm(bd)) - rel) < 1e-13
        # relaxed inner sign function: lower-degree table in the fp32 context only
        op32.set_chebyshev(alpha_lo)
        x2, no2, ni2, rel2, ok2 = op.cg_mixed(op32, bd, mu, tol=1e-9, inner_tol=1e-3, max_outer=60)
        assert ok2 and rel2 <= 1e-9 and rel_err(host(x2), xo) < 1e-6
        # not converged within the outer budget -> OVL_ENOTCONV, best iterate returned
        x3, no3, _, rel3, ok3 = op.cg_mixed(op32, bd, mu, tol=1e-12, inner_tol=1e-1, max_outer=1)
        assert not ok3 and no3 == 1 and rel3 < 1.0
        # argument checks: wrong precisions, different lattices
        out = torch.empty_like(bd)
        with pytest.raises(B.OvlError):
            B.ovl_cg_mixed(op32.ctx, op.ctx, mu, bd, out, 1e-8, 1e-4, 5, 100)
        with api.Overlap((4, 4, 4, 4), inputs.random_links((4, 4, 4, 4), 0.3, 1), "f32") as other:
            other.set_chebyshev(alpha)
            with pytest.raises(B.OvlError):
                B.ovl_cg_mixed(op.ctx, other.ctx, mu, bd, out, 1e-8, 1e-4, 5, 100)


def test_eigensolver_4x4_against_dense_spectrum(torch, api, orc, dense44):
    """ovl_lowest_eigenpairs on the config-0 lattice: eigenvalues against the dense spectrum of the
    oracle's K (both signs), residuals recomputed with the ORACLE's K, orthonormality, and the pairs used as a
    deflation space: sign(K) phi_i = sign(lambda_i) phi_i even with a poor polynomial."""
    d = dense44
    dims, U = d["dims"], d["U"]
    nev = 12
    ev = d["lam"][np.argsort(np.abs(d["lam"]))][:nev]
    with api.Overlap(dims, dev(torch, U)) as op:
        phi, lam, res, cyc, ok = op.lowest_eigenpairs(nev, tol=1e-9, filter_degree=40)
        assert ok and cyc > 0 and res.max() <= 1e-9
        assert np.abs(np.sort(lam) - np.sort(ev)).max() < 1e-10
        assert (lam > 0).any() and (lam < 0).any()
        ph = host(phi)
        gram = np.einsum("ixsc,jxsc->ij", ph.conj(), ph)
        assert np.abs(gram - np.eye(nev)).max() < 1e-10
        for i in (0, 5, nev - 1):
            r = orc.khat(dims, U, ph[i], 1.5, 6.5) * 6.5 - lam[i] * ph[i]
            assert np.linalg.norm(r) < 5e-9 and abs(np.linalg.norm(r) - res[i]) < 1e-9
        op.set_chebyshev(inputs.chebyshev_sign_coeffs(11, 0.3))
        op.set_deflation(phi, lam)
        for i in (0, nev - 1):
            s = host(op.sign(phi[i].contiguous()))
            assert rel_err(s, np.sign(lam[i]) * ph[i]) < 1e-8


def test_eigensolver_config1_lattice(torch, api, orc):
    """The deflation space of BASELINE config 1 computed on the GPU: 8^3 x 32, 20 pairs.  (i) pure gauge: |lambda| equals
    the closed-form lowest level (24-fold, tests/closed_forms.py); (ii) the smeared config-1 links: residuals checked
    with the oracle's K, both signs present, nearly degenerate +-pairs resolved."""
    from tests.closed_forms import free_sign_fft, golden_gammas
    dims, nev = (8, 8, 8, 32), 20
    U, g = inputs.pure_gauge_links(dims, inputs.SEED_BASE + 31)
    _, omega = free_sign_fft(dims, inputs.gaussian_spinor(dims, 1), golden_gammas(), 1.5, g)
    with api.Overlap(dims, dev(torch, U)) as op:
        phi, lam, res, cyc, ok = op.lowest_eigenpairs(nev, tol=1e-8, filter_degree=200, block=40)
    assert ok and np.abs(np.abs(lam) - omega.min()).max() < 1e-9
    U = inputs.config_links(dims, 0.3, inputs.SEED_BASE + 1, stout_steps=3)
    with api.Overlap(dims, dev(torch, U)) as op:
        phi, lam, res, cyc, ok = op.lowest_eigenpairs(nev, tol=1e-8, filter_degree=200, block=40)
        ph = host(phi)
    assert ok and res.max() <= 1e-8 and (lam > 0).any() and (lam < 0).any()
    assert 0.45 < np.abs(lam).min() and np.abs(lam).max() < 0.56 and np.all(np.diff(np.abs(lam)) >= -1e-12)
    for i in (0, 9, 19):
        r = orc.khat(dims, U, ph[i], 1.5, 6.5) * 6.5 - lam[i] * ph[i]
        assert np.linalg.norm(r) < 5e-8
    gram = np.einsum("ixsc,jxsc->ij", ph.conj(), ph)
    assert np.abs(gram - np.eye(nev)).max() < 1e-9


def test_eigensolver_mixed_precision(torch, api, orc, dense44):
    """ovl_lowest_eigenpairs_mixed: the Chebyshev filter on the fp32 kernels of a sibling context while the block is far
    from the tolerance, everything else in fp64.  (i) 4^4: eigenvalues against the dense spectrum of the oracle's K at the
    same 1e-10 as the all-fp64 solver, residuals <= tol; (ii) the smeared config-1 links (8^3 x 32, 20 pairs, block 40):
    residuals recomputed with the ORACLE's K, eigenvalues equal to the all-fp64 solver's, at least one filter cycle really
    ran in fp32 (the first cycles from a random start need the rescaled recurrence: T_d ~ 1e100 there); (iii) argument
    checks."""
    from paper_1510_06897_b200 import binding as B
    d = dense44
    dims, U = d["dims"], d["U"]
    nev = 12
    ev = d["lam"][np.argsort(np.abs(d["lam"]))][:nev]
    with api.Overlap(dims, dev(torch, U)) as op, api.Overlap(dims, dev(torch, U), "f32") as op32:
        phi, lam, res, cyc, c32, ok = op.lowest_eigenpairs_mixed(op32, nev, tol=1e-9, filter_degree=40)
        assert ok and c32 >= 1 and cyc > c32 and res.max() <= 1e-9
        assert np.abs(np.sort(lam) - np.sort(ev)).max() < 1e-10
        ph = host(phi)
        gram = np.einsum("ixsc,jxsc->ij", ph.conj(), ph)
        assert np.abs(gram - np.eye(nev)).max() < 1e-10
        out = torch.empty((2, 256, 4, 3), dtype=torch.complex128, device="cuda")
        for a, b in ((op32, op), (op, op)):
            with pytest.raises(B.OvlError) as e:
                B.ovl_lowest_eigenpairs_mixed(a.ctx, b.ctx, 2, 1e-6, 5, 20, 0, out)
            assert e.value.code == B.OVL_EINVAL
    dims, nev = (8, 8, 8, 32), 20
    U = inputs.config_links(dims, 0.3, inputs.SEED_BASE + 1, stout_steps=3)
    with api.Overlap(dims, dev(torch, U)) as op, api.Overlap(dims, dev(torch, U), "f32") as op32:
        phi, lam, res, cyc, c32, ok = op.lowest_eigenpairs_mixed(op32, nev, tol=1e-8, filter_degree=200, block=40)
        ph = host(phi)
        _, lam64, _, cyc64, ok64 = op.lowest_eigenpairs(nev, tol=1e-8, filter_degree=200, block=40)
    assert ok and ok64 and c32 >= 2 and res.max() <= 1e-8
    assert np.abs(np.sort(lam) - np.sort(lam64)).max() < 1e-9
    for i in (0, 9, 19):
        r = orc.khat(dims, U, ph[i], 1.5, 6.5) * 6.5 - lam[i] * ph[i]
        assert np.linalg.norm(r) < 5e-8
    gram = np.einsum("ixsc,jxsc->ij", ph.conj(), ph)
    assert np.abs(gram - np.eye(nev)).max() < 1e-9


def test_eigensolver_argument_checks(torch, api):
    from paper_1510_06897_b200 import binding as B
    dims = (4, 4, 4, 4)
    U = inputs.random_links(dims, 0.3, 3)
    with api.Overlap(dims, U, "f32") as op32:
        phi = torch.empty((2, 256, 4, 3), dtype=torch.complex128, device="cuda")
        with pytest.raises(B.OvlError) as e:
            B.ovl_lowest_eigenpairs(op32.ctx, 2, 1e-6, 5, 20, 0, phi)
        assert e.value.code == B.OVL_EINVAL
    with api.Overlap(dims, U) as op:
        phi, lam, res, cyc, ok = op.lowest_eigenpairs(4, tol=1e-14, max_cycles=1, filter_degree=5)
        assert not ok and cyc == 1 and np.isfinite(lam).all()      # OVL_ENOTCONV, best Ritz pairs returned
        out = np.empty((3, 256, 4, 3), dtype=np.complex128)         # host output buffer
        rc, lam, res, cyc = B.ovl_lowest_eigenpairs(op.ctx, 3, 1e-8, 60, 40, 0, out)
        assert rc == B.OVL_OK and abs(np.vdot(out[0], out[0]) - 1) < 1e-10


def test_multi_rhs_host_pointers_and_errors(torch, api, orc):
    from paper_1510_06897_b200 import binding as B
    dims = (4, 4, 4, 6)
    U = inputs.random_links(dims, 0.4, 71)
    alpha = rough_alpha(9, seed=2)
    psis = np.stack([inputs.gaussian_spinor(dims, 80 + r) for r in range(2)])
    with api.Overlap(dims, U) as op:            # host links
        with pytest.raises(B.OvlError) as e:
            op.overlap_multi(psis, 0.1)          # no polynomial yet
        assert e.value.code == B.OVL_ESTATE
        op.set_chebyshev(alpha)
        got = op.overlap_multi(psis, 0.1)        # numpy in, numpy out: staged by the library
        for r in range(2):
            assert rel_err(got[r], orc.overlap(dims, U, alpha, 0.1, psis[r])) < TOL_OVL
        out = np.empty_like(psis)
        for bad in (0, B.OVL_MAX_RHS + 1):
            rc = B.load_library().ovl_overlap_multi(op.ctx, bad, 0.1, 0, B._ptr(psis), B._ptr(out))
            assert rc == B.OVL_EINVAL


@pytest.mark.parametrize("prec,tol", [("f64", TOL_OVL), ("f32", TOL_F32)])
def test_config1_true_eigenpairs_pure_gauge_8x8x8x32(torch, api, orc, prec, tol):
    """BASELINE config 1 with TRUE eigenpairs: 8^3 x 32, degree 200, the 20 lowest-|lambda| eigenpairs of K in closed form
    on a pure gauge (gauge-rotated plane waves, tests/closed_forms.py; pinned against the oracle's K in the CPU suite).
    Tier A against the oracle, Tier B against the FFT closed form, and sign(K) phi_i = sign(lambda_i) phi_i."""
    from tests.closed_forms import free_sign_fft, golden_gammas, lowest_pure_gauge_eigenpairs
    dims, nev = (8, 8, 8, 32), 20
    U, g = inputs.pure_gauge_links(dims, inputs.SEED_BASE + 31)
    G = golden_gammas()
    phi, lam = lowest_pure_gauge_eigenpairs(dims, g, G, nev)
    psi = inputs.gaussian_spinor(dims, inputs.SEED_BASE + 131)
    exact, omega = free_sign_fft(dims, psi, G, 1.5, g)
    alpha = inputs.chebyshev_sign_coeffs(200, 0.95 * omega.min() / 6.5)
    delta = np.abs(inputs.chebyshev_eval(alpha, omega.ravel() / 6.5) - 1.0).max()
    want = orc.overlap(dims, U, alpha, 0.01, psi, phi, lam)
    with api.Overlap(dims, dev(torch, U), prec) as op:
        assert op.set_chebyshev(alpha) == 199
        op.set_deflation(dev(torch, phi), lam)
        p = dev(torch, psi, op.cdtype)
        got = host(op.overlap(p, 0.01)).astype(np.complex128)
        s = host(op.sign(p)).astype(np.complex128)
        e7 = host(op.sign(dev(torch, phi[7], op.cdtype))).astype(np.complex128)
    assert rel_err(got, want) < tol                                       # Tier A
    assert rel_err(s, exact) < max(2 * delta, tol)                        # Tier B (delta ~ 5e-8 at N = 200)
    assert rel_err(e7, np.sign(lam[7]) * phi[7]) < (1e-12 if prec == "f64" else tol)


def test_bit_identical_run_to_run(torch, api):
    dims = (6, 6, 6, 10)
    U = dev(torch, inputs.random_links(dims, 0.4, 61))
    psi = dev(torch, inputs.gaussian_spinor(dims, 62))
    phi = dev(torch, inputs.orthonormal_vectors(dims, 4, 63))
    alpha = inputs.chebyshev_sign_coeffs(41, 0.1)
    outs = []
    for _ in range(2):
        with api.Overlap(dims, U) as op:
            op.set_chebyshev(alpha)
            op.set_deflation(phi, [0.3, -0.3, 0.4, -0.4])
            y = op.overlap(psi, 0.03)
            x, it, rel, _ = op.cg(psi, 0.3, tol=1e-6, maxiter=50)
            outs.append((host(y), host(x), it, rel))
    assert np.array_equal(outs[0][0], outs[1][0])
    assert np.array_equal(outs[0][1], outs[1][1])
    assert outs[0][2:] == outs[1][2:]


def test_error_statuses(torch, api):
    from paper_1510_06897_b200 import binding as B
    dims = (4, 4, 4, 4)
    U = dev(torch, inputs.unit_links(dims))
    psi = dev(torch, inputs.gaussian_spinor(dims, 1))
    with pytest.raises(B.OvlError) as e:
        api.Overlap((4, 4, 1, 4), U)
    assert e.value.code == B.OVL_EINVAL
    with api.Overlap(dims, U) as op:
        with pytest.raises(B.OvlError) as e:
            op.sign(psi)  # no polynomial yet
        assert e.value.code == B.OVL_ESTATE and "chebyshev" in str(e.value)
        with pytest.raises(B.OvlError) as e:
            B.ovl_dw(op.ctx, psi, psi)  # aliasing
        assert e.value.code == B.OVL_EINVAL
        with pytest.raises(B.OvlError) as e:
            op.set_chebyshev([0.0, float("nan")])
        assert e.value.code == B.OVL_EINVAL
        op.set_chebyshev([0.0, 1.0])
        with pytest.raises(B.OvlError) as e:
            op.set_deflation(psi.reshape(1, -1, 4, 3), [0.0])  # reading R9
        assert e.value.code == B.OVL_EINVAL
        with pytest.raises(B.OvlError) as e:
            B.ovl_set_kernel(op.ctx, 1.5, -1.0)
        assert e.value.code == B.OVL_EINVAL
        assert op.launch_count() > 0


def test_deflation_exact_eigenpairs_4x4(torch, api, orc, dense44):
    """True eigenpairs (dense 4^4): the deflated GPU map equals W diag(sign lam_i [deflated] | p(lam_i)) W^dag psi and
    sits closer to the exact sign function than the undeflated one (coarse N = 15 polynomial)."""
    d = dense44
    nev = 20
    idx = np.argsort(np.abs(d["lam"]))[:nev]
    lam_d = d["lam"][idx]
    phi = np.ascontiguousarray(d["W"][:, idx].T).reshape(nev, -1, 4, 3)
    alpha = inputs.chebyshev_sign_coeffs(15, 0.2)
    psi = inputs.gaussian_spinor(d["dims"], 55)
    diag = inputs.chebyshev_eval(alpha, d["lam"] / 6.5)
    diag[idx] = np.sign(lam_d)
    want = (d["W"] * diag) @ (d["W"].conj().T @ psi.ravel())
    with api.Overlap(d["dims"], dev(torch, d["U"])) as op:
        op.set_chebyshev(alpha)
        p = dev(torch, psi)
        plain = host(op.sign(p)).ravel()
        op.set_deflation(dev(torch, phi), lam_d)
        got = host(op.sign(p)).ravel()
    assert rel_err(got, want) < 1e-11
    assert rel_err(got, orc.sign(d["dims"], d["U"], alpha, psi, phi, lam_d).ravel()) < TOL_OVL
    exact = d["S"] @ psi.ravel()
    assert np.linalg.norm(got - exact) < np.linalg.norm(plain - exact)


@pytest.mark.parametrize("rec", RECS)
def test_table_with_only_alpha0(torch, api, orc, rec):
    """alpha = [c0, 0]: no K^ term at all (reading R8: alpha_0 is honoured) -- sign() must return c0 psi, not NaN."""
    dims = (4, 4, 4, 4)
    U = inputs.random_links(dims, 0.5, 9)
    psi = inputs.gaussian_spinor(dims, 10)
    alpha = np.array([0.75, 0.0])
    with api.Overlap(dims, dev(torch, U)) as op:
        op.set_recurrence(rec)
        assert op.set_chebyshev(alpha) == 1
        got = host(op.sign(dev(torch, psi)))
    assert rel_err(got, orc.sign(dims, U, alpha, psi)) < TOL_OVL
    assert rel_err(got, 0.75 * psi) < 1e-14


def test_cg_multi_with_a_zero_right_hand_side(torch, api, orc):
    """One zero source among several: its solution is exactly 0 (no NaN from 0/0) and the others are untouched."""
    dims = (4, 4, 4, 8)
    U = inputs.config_links(dims, 0.3, 77, stout_steps=1)
    alpha = inputs.chebyshev_sign_coeffs(41, 0.09)
    b = np.stack([inputs.gaussian_spinor(dims, 79), np.zeros((int(np.prod(dims)), 4, 3), complex), inputs.gaussian_spinor(dims, 81)])
    with api.Overlap(dims, dev(torch, U)) as op:
        op.set_chebyshev(alpha)
        bd = dev(torch, b)
        x, its, rels, ok = op.cg_multi(bd, 0.2, tol=1e-9, maxiter=500)
        assert ok and its[1] == 0 and rels[1] == 0.0
        assert torch.count_nonzero(x[1]).item() == 0
        for r in (0, 2):
            xs, it1, _, ok1 = op.cg(bd[r].contiguous(), 0.2, tol=1e-9, maxiter=500)
            assert ok1 and it1 == its[r] and torch.equal(xs, x[r])
        x0, it0, rel0, ok0 = op.cg(bd[1].contiguous(), 0.2, tol=1e-9, maxiter=50)
        assert ok0 and it0 == 0 and torch.count_nonzero(x0).item() == 0


def test_eigensolver_not_converged_returns_consistent_ritz_pairs(torch, api, orc):
    """OVL_ENOTCONV path: with too few cycles the returned (phi_i, lambda_i, resid_i) must still belong together --
    ||K phi_i - lambda_i phi_i|| recomputed with the oracle's K equals the reported residual."""
    dims = (4, 4, 4, 8)
    U = inputs.config_links(dims, 0.3, 61, stout_steps=1)
    with api.Overlap(dims, dev(torch, U)) as op:
        for cycles, tol in [(1, 1e-13), (2, 1e-9), (3, 1e-11)]:
            phi, lam, res, cyc, ok = op.lowest_eigenpairs(4, tol=tol, max_cycles=cycles, filter_degree=6, block=6)
            ph = host(phi)
            for i in range(4):
                kp = 6.5 * orc.khat(dims, U, ph[i])
                r = np.linalg.norm((kp - lam[i] * ph[i]).ravel())
                assert abs(r - res[i]) <= 1e-9 + 1e-6 * res[i], (cycles, i, r, res[i], ok)
                assert abs(np.linalg.norm(ph[i].ravel()) - 1.0) < 1e-10


def test_caller_owned_workspace(torch, api, orc):
    """a context created inside a torch-owned workspace (ovl_create_ws) never allocates or frees device memory
    afterwards -- torch's allocator sees every byte -- and gives results bit-identical to the library-owned context.
    Exceeding a capacity the workspace was sized for is OVL_EINVAL, not a hidden allocation."""
    from paper_1510_06897_b200 import binding as B
    dims = (4, 4, 6, 8)
    U = inputs.config_links(dims, 0.3, 41, stout_steps=1)
    alpha = inputs.chebyshev_sign_coeffs(41, 0.09)
    phi = inputs.orthonormal_vectors(dims, 4, 43)
    lam = np.array([0.45, -0.47, 0.5, -0.52])
    psi = np.stack([inputs.gaussian_spinor(dims, 50 + r) for r in range(3)])
    Ud, phid, pd = dev(torch, U), dev(torch, phi), dev(torch, psi)
    need = B.ovl_workspace_bytes(dims, B.OVL_F64, B.OVL_RECON18, 4, 3, 12)
    assert need > 0
    ws = torch.empty(need + 512, dtype=torch.uint8, device="cuda")
    with api.Overlap(dims, Ud) as ref, api.Overlap(dims, Ud, workspace=dict(max_nev=4, max_rhs=3, eig_block=12, buffer=ws)) as op:
        for o in (ref, op):
            o.set_chebyshev(alpha)
            o.set_deflation(phid, lam)
        import gc
        gc.collect()
        torch.cuda.synchronize()
        outs = torch.empty_like(pd)
        x = torch.empty_like(pd)
        xs = torch.empty_like(pd[0])
        ev = torch.empty((4, int(np.prod(dims)), 4, 3), dtype=torch.complex128, device="cuda")
        # every kernel once on the library-owned context first: the driver loads a kernel's code on its first launch (CUDA
        # lazy loading) and takes device memory for it, which is not an allocation of the library
        ref.overlap_multi(pd, 0.05); ref.cg(pd[0], 0.2, tol=1e-9, maxiter=3); ref.cg_multi(pd, 0.2, tol=1e-9, maxiter=3)
        ref.overlap(psi[1], 0.05); ref.lowest_eigenpairs(4, tol=1e-8, max_cycles=60, filter_degree=40, block=12)
        alloc1 = torch.cuda.memory_allocated()
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        # every entry point that used to allocate lazily: multi-rhs, CG, multi-CG, host-pointer staging, the eigensolver
        B.ovl_overlap_multi(op.ctx, 3, 0.05, 0, pd, outs)
        B.ovl_cg(op.ctx, 0.2, pd[0], xs, 1e-9, 200)
        B.ovl_cg_multi(op.ctx, 3, 0.2, pd, x, 1e-9, 200)
        hy = op.overlap(psi[1], 0.05)                      # numpy in / out: staged through the workspace
        rc, lam_e, res_e, cyc = B.ovl_lowest_eigenpairs(op.ctx, 4, 1e-8, 60, 40, 12, ev)
        torch.cuda.synchronize()
        free2, _ = torch.cuda.mem_get_info()
        assert torch.cuda.memory_allocated() <= alloc1  # (torch may have released temporaries of earlier tests)
        assert free2 == free1, "the library allocated device memory behind torch's back"
        assert rc == B.OVL_OK
        # same results as the library-owned context, bit for bit
        assert torch.equal(outs, ref.overlap_multi(pd, 0.05))
        xr, itr, _, _ = ref.cg(pd[0], 0.2, tol=1e-9, maxiter=200)
        assert torch.equal(xs, xr)
        assert np.array_equal(hy, ref.overlap(psi[1], 0.05))
        pr, lr, _, _, okr = ref.lowest_eigenpairs(4, tol=1e-8, max_cycles=60, filter_degree=40, block=12)
        assert okr and np.array_equal(lam_e, lr) and torch.equal(ev, pr)
        # capacities are hard limits
        five = dev(torch, inputs.orthonormal_vectors(dims, 5, 44))
        with pytest.raises(B.OvlError) as e:
            op.set_deflation(five, np.array([0.4, -0.4, 0.5, -0.5, 0.6]))
        assert e.value.code == B.OVL_EINVAL
        four = torch.cat([pd, pd[:1]])
        with pytest.raises(B.OvlError) as e:
            op.overlap_multi(four, 0.05)
        assert e.value.code == B.OVL_EINVAL
        with pytest.raises(B.OvlError) as e:
            op.lowest_eigenpairs(4, block=16)
        assert e.value.code == B.OVL_EINVAL
        assert torch.equal(op.overlap(pd[0], 0.05), ref.overlap(pd[0], 0.05))  # still usable after the errors
    # a too small or misaligned workspace is refused
    with pytest.raises(B.OvlError):
        B.ovl_create_ws(dims, Ud, ws[: need - 256], max_nev=4, max_rhs=3, eig_block=12)
    with pytest.raises(B.OvlError):
        B.ovl_create_ws(dims, Ud, ws[8:], max_nev=4, max_rhs=3, eig_block=12)
    assert float(np.abs(host(outs)).max()) > 0


@pytest.mark.parametrize("chir", [+1, -1])
def test_cg_chiral_sector(torch, api, orc, chir):
    """ovl_cg_chiral (reading R23) against the oracle's chiral-sector CG: fixed iterations at 1e-10, to
    tolerance (R14's checks), solution confined to the sector, half the stencil launches of the full D^dag D solve, and
    agreement with the full solve on the projected source up to the polynomial's s^2 - 1."""
    dims = (4, 4, 6, 8)
    U = inputs.config_links(dims, 0.3, 21, stout_steps=2)
    alpha = inputs.chebyshev_sign_coeffs(161, 0.07)     # delta ~ 1e-6 on this spectrum
    phi = inputs.orthonormal_vectors(dims, 3, 23)
    lam = np.array([0.5, -0.51, 0.52])
    b = inputs.gaussian_spinor(dims, 24)
    mu = 0.1
    g5v = G5[None, :, None]
    with api.Overlap(dims, dev(torch, U)) as op:
        op.set_chebyshev(alpha)
        op.set_deflation(dev(torch, phi), lam)
        bd = dev(torch, b)
        xk, itk, _, okk = op.cg_chiral(bd, mu, chir, tol=0.0, maxiter=8)
        l0 = op.launch_count()
        x, it, rel, ok = op.cg_chiral(bd, mu, chir, tol=1e-9, maxiter=500)
        l1 = op.launch_count()
        pb = dev(torch, 0.5 * (1 + chir * g5v) * b)
        xf, itf, relf, okf = op.cg(pb, mu, tol=1e-9, maxiter=500)
        l2 = op.launch_count()
    wk, ito, _ = orc.cg_chiral(dims, U, alpha, mu, chir, b, 0.0, 8, phi, lam)
    assert itk == ito == 8 and okk
    assert rel_err(host(xk), wk) < TOL_OVL
    xo, ito, relo = orc.cg_chiral(dims, U, alpha, mu, chir, b, 1e-9, 500, phi, lam)
    assert ok and abs(it - ito) <= 2 and rel < 1.05e-9 and relo < 1.05e-9
    assert rel_err(host(x), xo) < 1e-6
    assert np.abs(0.5 * (1 - chir * g5v) * host(x)).max() == 0.0            # x = P_c x exactly
    # one sign application per iteration instead of two
    assert okf and abs(itf - it) <= 2
    per_it_chiral, per_it_full = (l1 - l0) / (it + 1), (l2 - l1) / (itf + 1)
    assert per_it_chiral < 0.55 * per_it_full
    assert rel_err(host(xf), host(x)) < 1e-3                                # kappa * 1/4 (1-mu)^2 * 2 delta


@pytest.mark.parametrize("chir", [+1, -1])
def test_cg_mixed_chiral(torch, api, orc, chir):
    """ovl_cg_mixed_chiral: the chiral-sector system A_c x = P_c b (R23) by defect correction with fp32 inner solves.  A true
    fp64 residual of 1e-11 -- below what fp32 can represent -- the oracle's chiral-sector CG solution, x = P_c x exactly, the
    reported residual recomputed through the public fp64 operator (A_c from one ovl_sign), and half the stencil launches of
    ovl_cg_mixed on the projected source."""
    from paper_1510_06897_b200 import binding as B
    dims = (4, 4, 4, 8)
    U = inputs.config_links(dims, 0.3, 177, stout_steps=1)
    alpha = inputs.chebyshev_sign_coeffs(61, 0.09)
    phi = inputs.orthonormal_vectors(dims, 3, 178)
    lam = np.array([0.45, -0.47, 0.5])
    b = inputs.gaussian_spinor(dims, 179)
    mu = 0.2
    g5v = G5[None, :, None]
    xo, ito, relo = orc.cg_chiral(dims, U, alpha, mu, chir, b, 1e-11, 500, phi, lam)
    with api.Overlap(dims, dev(torch, U), "f64") as op, api.Overlap(dims, dev(torch, U), "f32") as op32:
        for o in (op, op32):
            o.set_chebyshev(alpha)
            o.set_deflation(dev(torch, phi), lam)
        bd = dev(torch, b)
        l0 = op.launch_count() + op32.launch_count()
        x, no, ni, rel, ok = op.cg_mixed_chiral(op32, bd, mu, chir, tol=1e-11, inner_tol=1e-4)
        l1 = op.launch_count() + op32.launch_count()
        assert ok and rel <= 1e-11 and 2 <= no <= 6
        assert rel_err(host(x), xo) < 1e-8
        assert np.abs(0.5 * (1 - chir * g5v) * host(x)).max() == 0.0
        pc = dev(torch, 0.5 * (1 + chir * g5v) * np.ones_like(b))
        pb = pc * bd
        acx = 0.5 * (1 + mu * mu) * x + 0.5 * chir * (1 - mu * mu) * pc * op.sign(x)
        assert abs(float(torch.linalg.norm(pb - acx) / torch.linalg.norm(pb)) - rel) < 1e-13
        xf, nof, nif, relf, okf = op.cg_mixed(op32, pb, mu, tol=1e-11, inner_tol=1e-4)
        l2 = op.launch_count() + op32.launch_count()
        assert okf and (l1 - l0) / max(ni, 1) < 0.6 * (l2 - l1) / max(nif, 1)
        out = torch.empty_like(bd)
        with pytest.raises(B.OvlError) as e:
            B.ovl_cg_mixed_chiral(op.ctx, op32.ctx, mu, 0, bd, out, 1e-8, 1e-4, 5, 100)
        assert e.value.code == B.OVL_EINVAL
        with pytest.raises(B.OvlError):
            B.ovl_cg_mixed_chiral(op32.ctx, op.ctx, mu, chir, bd, out, 1e-8, 1e-4, 5, 100)


def test_cg_multi_chiral(torch, api, orc):
    """ovl_cg_multi_chiral: several chiral-sector systems in lockstep -- every solution bit-identical to the single-system
    ovl_cg_chiral, one of them against the oracle's chiral-sector CG, a source with P_c b = 0 among the others returns
    x = 0 after 0 iterations."""
    dims = (4, 4, 6, 8)
    U = inputs.config_links(dims, 0.3, 21, stout_steps=2)
    alpha = inputs.chebyshev_sign_coeffs(101, 0.07)
    phi = inputs.orthonormal_vectors(dims, 3, 23)
    lam = np.array([0.5, -0.51, 0.52])
    mu, chir = 0.1, -1
    bs = np.stack([inputs.gaussian_spinor(dims, 300 + r) for r in range(4)])
    bs[2] = 0.5 * (1 - chir * G5[None, :, None]) * bs[2]        # lives entirely in the other sector: P_c b = 0
    with api.Overlap(dims, dev(torch, U)) as op:
        op.set_chebyshev(alpha)
        op.set_deflation(dev(torch, phi), lam)
        bd = dev(torch, bs)
        x, it, rel, ok = op.cg_multi_chiral(bd, mu, chir, tol=1e-9, maxiter=500)
        singles = [op.cg_chiral(bd[r].contiguous(), mu, chir, tol=1e-9, maxiter=500) for r in range(4)]
    assert ok and it[2] == 0 and float(torch.abs(x[2]).max()) == 0.0
    for r in range(4):
        assert torch.equal(x[r], singles[r][0]) and it[r] == singles[r][1]
        if r != 2:
            assert rel[r] < 1.05e-9
    xo, ito, relo = orc.cg_chiral(dims, U, alpha, mu, chir, bs[1], 1e-9, 500, phi, lam)
    assert abs(it[1] - ito) <= 2 and rel_err(host(x[1]), xo) < 1e-6


def test_fused_variant_argument_checks(torch, api):
    from paper_1510_06897_b200 import binding as B
    dims = (5, 3, 7, 3)     # Lz, Lt odd: no brick decomposition
    with api.Overlap(dims, inputs.random_links(dims, 0.3, 5)) as op:
        with pytest.raises(B.OvlError) as e:
            op.set_fused_variant("brick")
        assert e.value.code == B.OVL_EINVAL
        with pytest.raises(B.OvlError) as e:
            op.set_fused_variant(7)
        assert e.value.code == B.OVL_EINVAL
        for v in ("plain", "bulk", "register"):
            op.set_fused_variant(v)
        p = dev(torch, inputs.gaussian_spinor(dims, 6))
        assert torch.isfinite(torch.view_as_real(op.dw(p))).all()


def test_workspace_contexts_mixed_precision_calls(torch, api):
    """The calls that pair an fp64 with an fp32 context (ovl_cg_mixed_chiral, ovl_lowest_eigenpairs_mixed) and the chiral
    lockstep solver, with BOTH contexts inside torch-owned workspaces: no device allocation behind torch's back, results
    bit-identical to library-owned contexts."""
    from paper_1510_06897_b200 import binding as B
    dims = (4, 4, 6, 8)
    U = inputs.config_links(dims, 0.3, 41, stout_steps=1)
    alpha = inputs.chebyshev_sign_coeffs(41, 0.09)
    phi = inputs.orthonormal_vectors(dims, 4, 43)
    lam = np.array([0.45, -0.47, 0.5, -0.52])
    psi = np.stack([inputs.gaussian_spinor(dims, 50 + r) for r in range(3)])
    Ud, phid, pd = dev(torch, U), dev(torch, phi), dev(torch, psi)
    caps = dict(max_nev=4, max_rhs=3, eig_block=12)
    with api.Overlap(dims, Ud) as r64, api.Overlap(dims, Ud, "f32") as r32, \
            api.Overlap(dims, Ud, workspace=dict(caps)) as w64, api.Overlap(dims, Ud, "f32", workspace=dict(caps)) as w32:
        for o in (r64, r32, w64, w32):
            o.set_chebyshev(alpha)
            o.set_deflation(phid, lam)
        x1, x2 = torch.empty_like(pd[0]), torch.empty_like(pd)
        ev = torch.empty((4, int(np.prod(dims)), 4, 3), dtype=torch.complex128, device="cuda")
        # reference results first: they also load every kernel's code (CUDA lazy loading takes device memory per kernel)
        y1, _, _, _, ok1 = r64.cg_mixed_chiral(r32, pd[0], 0.2, +1, tol=1e-10, inner_tol=1e-4, max_outer=10, max_inner=200)
        y2, _, _, ok2 = r64.cg_multi_chiral(pd, 0.2, -1, tol=1e-9, maxiter=200)
        pr, lr, _, _, _, ok3 = r64.lowest_eigenpairs_mixed(r32, 4, tol=1e-8, max_cycles=60, filter_degree=40, block=12)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        rc1, no, ni, rel = B.ovl_cg_mixed_chiral(w64.ctx, w32.ctx, 0.2, +1, pd[0], x1, 1e-10, 1e-4, 10, 200)
        rc2, its, rels = B.ovl_cg_multi_chiral(w64.ctx, 3, 0.2, -1, pd, x2, 1e-9, 200)
        rc3, lam_e, res_e, cyc, c32 = B.ovl_lowest_eigenpairs_mixed(w64.ctx, w32.ctx, 4, 1e-8, 60, 40, 12, ev)
        torch.cuda.synchronize()
        free2, _ = torch.cuda.mem_get_info()
        assert free2 == free1, "the library allocated device memory behind torch's back"
        assert rc1 == rc2 == rc3 == B.OVL_OK and rel <= 1e-10 and c32 >= 1
        assert ok1 and ok2 and ok3
        assert torch.equal(x1, y1) and torch.equal(x2, y2) and np.array_equal(lam_e, lr) and torch.equal(ev, pr)


def test_cg_chiral_argument_checks(torch, api):
    from paper_1510_06897_b200 import binding as B
    dims = (4, 4, 4, 4)
    U = inputs.random_links(dims, 0.3, 5)
    b = dev(torch, inputs.gaussian_spinor(dims, 6))
    with api.Overlap(dims, dev(torch, U)) as op:
        with pytest.raises(B.OvlError) as e:
            op.cg_chiral(b, 0.1, +1)
        assert e.value.code == B.OVL_ESTATE
        op.set_chebyshev(inputs.chebyshev_sign_coeffs(21, 0.1))
        with pytest.raises(B.OvlError) as e:
            op.cg_chiral(b, 0.1, 0)
        assert e.value.code == B.OVL_EINVAL
        z = torch.zeros_like(b)
        z[:, 2:] = b[:, 2:]                                                  # purely negative chirality
        x0, it0, rel0, ok0 = op.cg_chiral(z, 0.1, +1, tol=1e-9, maxiter=10)
        assert ok0 and it0 == 0 and rel0 == 0.0 and torch.count_nonzero(x0).item() == 0


@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
@pytest.mark.parametrize("dims", [(8, 8, 8, 32), (4, 4, 4, 6), (6, 6, 6, 8)])
def test_bulk_copy_variant_bit_identical(torch, api, orc, prec, recon, dims):
    """OVL_FUSED_BULK (persistent warps, the links landed in shared memory by cp.async.bulk + mbarrier) gives the same bits
    as the default register-landing kernel: D_W, K^, the deflated sign function (both eligible and fallback lattices:
    6^3 x 8 has Lx Ly Lz = 216, not a multiple of 32, and silently stays on the default kernel)."""
    U = inputs.config_links(dims, 0.4, 51, stout_steps=1)
    psi = inputs.gaussian_spinor(dims, 52)
    alpha = rough_alpha(24, seed=7)
    phi = inputs.orthonormal_vectors(dims, 2, 53)
    lam = np.array([0.5, -0.6])
    with api.Overlap(dims, dev(torch, U), prec, recon) as op:
        op.set_chebyshev(alpha)
        op.set_deflation(dev(torch, phi), lam)
        p = dev(torch, psi, op.cdtype)
        want = [op.dw(p), op.khat(p), op.sign(p), op.overlap(p, 0.1, dagger=True)]
        op.set_fused_variant("bulk")
        got = [op.dw(p), op.khat(p), op.sign(p), op.overlap(p, 0.1, dagger=True)]
        again = op.sign(p)
        op.set_fused_variant("register")
        back = op.sign(p)
    for g_, w_ in zip(got, want):
        assert torch.equal(g_, w_)
    assert torch.equal(again, want[2]) and torch.equal(back, want[2])
    tol = TOL_OVL if prec == "f64" else TOL_F32
    assert rel_err(host(got[2]).astype(np.complex128), orc.sign(dims, U, alpha, psi, phi, lam)) < tol


@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f64", 12), ("f32", 18), ("f32", 12)])
@pytest.mark.parametrize("dims", [(8, 8, 8, 32), (4, 6, 8, 10), (6, 4, 2, 8), (2, 2, 2, 2), (10, 6, 4, 12), (8, 8, 8, 8), (12, 12, 12, 24)])
def test_brick_order_bit_identical_to_plain_order(torch, api, orc, prec, recon, dims):
    """Brick order (k_wilson_fused_brick: a CTA takes a 2 x 2 stack in (z, t) of 32-site chunks; the default for
    2^15 <= V <= 2^17, forced here with OVL_FUSED_BRICK) against the plain tile order (OVL_FUSED_PLAIN) on the same lattice:
    D_W, K^, the deflated sign function in both recurrences and D^dag must agree bit for bit -- ragged chunks (V/2 not a
    multiple of 32 per time-slice pair), extent-2 directions, non-cubic shapes -- and the plain-order result is held
    against the oracle."""
    U = inputs.config_links(dims, 0.4, 61, stout_steps=1)
    psi = inputs.gaussian_spinor(dims, 62)
    alpha = rough_alpha(17, seed=9)
    phi = inputs.orthonormal_vectors(dims, 2, 63)
    lam = np.array([0.45, -0.55])

    def run(op, p):
        res = [op.dw(p), op.khat(p)]
        for rec in RECS:
            op.set_recurrence(rec)
            res += [op.sign(p), op.overlap(p, 0.1, dagger=True)]
        op.set_recurrence("clenshaw")
        return res

    with api.Overlap(dims, dev(torch, U), prec, recon) as op:
        op.set_chebyshev(alpha)
        op.set_deflation(dev(torch, phi), lam)
        p = dev(torch, psi, op.cdtype)
        default = op.sign(p)
        op.set_fused_variant("brick")
        brick = run(op, p)
        op.set_fused_variant("plain")
        plain = run(op, p)
        op.set_fused_variant("register")
        back = op.sign(p)
    for b_, p_ in zip(brick, plain):
        assert torch.equal(b_, p_)
    assert torch.equal(back, brick[2]) and torch.equal(default, brick[2])
    tol = TOL_OVL if prec == "f64" else TOL_F32
    assert rel_err(host(plain[0]).astype(np.complex128), orc.dw(dims, U, psi)) < (TOL_DW if prec == "f64" else TOL_F32)
    assert rel_err(host(plain[2]).astype(np.complex128), orc.sign(dims, U, alpha, psi, phi, lam)) < tol
