"""GPU parity at BASELINE.json's full size (20^3 x 64, the launch configuration bench.py times): the whole D_W field
and a low-degree deflated overlap apply against the oracle, and the degree-400 sign function against the FFT closed
form on a pure gauge (tests/closed_forms.py), in fp64 and fp32."""
import numpy as np
import pytest

from paper_1510_06897_b200 import inputs
from tests.closed_forms import free_sign_fft, golden_gammas, lowest_pure_gauge_eigenpairs
from tests.conftest import rel_err

pytestmark = pytest.mark.gpu
DIMS = (20, 20, 20, 64)


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def api(torch):
    from paper_1510_06897_b200 import api, binding
    binding.load_library()
    return api


@pytest.fixture(scope="module")
def rough(torch):
    U = inputs.random_links(DIMS, 0.25, inputs.SEED_BASE + 3)
    psi = inputs.gaussian_spinor(DIMS, inputs.SEED_BASE + 103)
    return U, psi


def dev(torch, a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t.to(dtype) if dtype is not None else t


@pytest.mark.parametrize("prec,recon,tol", [("f64", 18, 1e-12), ("f64", 12, 1e-12), ("f32", 18, 1e-5), ("f32", 12, 1e-5)])
def test_dw_full_field_20x20x20x64(torch, api, orc, rough, prec, recon, tol):
    U, psi = rough
    want = orc.dw(DIMS, U, psi)
    with api.Overlap(DIMS, dev(torch, U), prec, recon) as op:
        got = op.dw(dev(torch, psi, op.cdtype)).cpu().numpy().astype(np.complex128)
    assert rel_err(got, want) < tol
    # sampled sites, element by element (max norm), including both t boundaries
    v = want.shape[0]
    sites = np.concatenate([np.arange(0, 50), np.arange(v - 50, v), np.random.default_rng(1).integers(0, v, 500)])
    scale = np.abs(want).max()
    assert np.abs(got[sites] - want[sites]).max() < 20 * tol * scale


@pytest.mark.parametrize("rec", ["clenshaw", "forward"])
def test_low_degree_deflated_overlap_vs_oracle_full_size(torch, api, orc, rough, rec):
    """The fused Chebyshev step, deflation and assembly in the full-size launch configuration against the oracle
    (degree 9 keeps the oracle to seconds; every kernel variant of the degree-400 path is exercised)."""
    U, psi = rough
    phi = inputs.phase_vectors(DIMS, 3, inputs.SEED_BASE + 203)
    lam = np.array([0.5, -0.51, 0.52])
    alpha = inputs.chebyshev_sign_coeffs(9, 0.3)
    want = orc.overlap(DIMS, U, alpha, 0.01, psi, phi, lam)
    with api.Overlap(DIMS, dev(torch, U)) as op:
        op.set_recurrence(rec)
        op.set_chebyshev(alpha)
        op.set_deflation(dev(torch, phi), lam)
        got = op.overlap(dev(torch, psi), 0.01).cpu().numpy()
    assert rel_err(got, want) < 1e-10


@pytest.mark.parametrize("prec,tol", [("f64", 1e-12), ("f32", 1e-5)])
def test_dw_maximum_volume_48x48x48x96(torch, api, orc, prec, tol):
    """The largest volume of BASELINE config 4 (10.6 M sites; canonical links 6.1 GB, i.e. byte offsets beyond 2^32 and
    382 M-element planes): D_W over the whole field against the oracle.  Links are a 12^3 x 24 random block repeated
    periodically (inputs.tiled_links) so that the host can generate them in seconds; the spinor is fully random."""
    dims, block = (48, 48, 48, 96), (12, 12, 12, 24)
    U = inputs.tiled_links(dims, block, 0.3, inputs.SEED_BASE + 4)
    psi = inputs.gaussian_spinor(dims, inputs.SEED_BASE + 104)
    want = orc.dw(dims, U, psi)
    with api.Overlap(dims, U, prec, 18) as op:           # host links: staged by the library
        p = dev(torch, psi, op.cdtype)
        got = op.dw(p).cpu().numpy()
        del p
    err = rel_err(got.astype(np.complex128), want)
    assert err < tol, err
    v = want.shape[0]
    sites = np.concatenate([np.arange(0, 64), np.arange(v - 64, v), np.random.default_rng(2).integers(0, v, 2000)])
    assert np.abs(got[sites] - want[sites]).max() < 20 * tol * np.abs(want).max()


def test_multi_rhs_full_size_matches_single(torch, api, rough):
    """4 right-hand sides at 20^3 x 64 in the launch configuration bench.py times (grid = 4 x 4000 CTAs): bit-identical
    to four single applies (which the tests above pin to the oracle and to the FFT closed form)."""
    U, psi = rough
    alpha = inputs.chebyshev_sign_coeffs(12, 0.3)
    phi = inputs.phase_vectors(DIMS, 2, inputs.SEED_BASE + 204)
    lam = np.array([0.5, -0.51])
    with api.Overlap(DIMS, dev(torch, U)) as op:
        op.set_chebyshev(alpha)
        op.set_deflation(dev(torch, phi), lam)
        p0 = dev(torch, psi)
        ps = torch.stack([p0, p0.conj().contiguous(), (1j * p0), p0.flip(0).contiguous()])
        got = op.overlap_multi(ps, 0.01)
        for r in range(4):
            assert torch.equal(got[r], op.overlap(ps[r].contiguous(), 0.01)), r


@pytest.mark.parametrize("prec,tol,rec", [("f64", 1e-10, "clenshaw"), ("f64", 1e-10, "forward"), ("f32", 1e-5, "clenshaw"),
                                          ("f32", 1e-5, "forward")])
def test_degree400_sign_vs_fft_closed_form_full_size(torch, api, prec, tol, rec):
    """Pure gauge U_mu(x) = g(x) g(x+mu)^dag at 20^3 x 64: sign(K) psi is known in closed form at any volume. With the
    degree-400 table the polynomial error on the spectrum is < 1e-12, so GPU vs closed form tests the whole
    399-order recurrence in bench.py's configuration."""
    U, g = inputs.pure_gauge_links(DIMS, inputs.SEED_BASE + 33)
    psi = inputs.gaussian_spinor(DIMS, inputs.SEED_BASE + 133)
    exact, omega = free_sign_fft(DIMS, psi, golden_gammas(), 1.5, g)
    eps = 0.95 * omega.min() / 6.5
    alpha = inputs.chebyshev_sign_coeffs(400, eps)
    delta = np.abs(inputs.chebyshev_eval(alpha, omega.ravel() / 6.5) - 1.0).max()
    assert delta < 1e-11
    # on a side stream, as bench.py runs it: the 399 launches are replayed from a CUDA graph
    side = torch.cuda.Stream()
    with torch.cuda.stream(side), api.Overlap(DIMS, dev(torch, U), prec, stream=side) as op:
        op.set_recurrence(rec)
        assert op.set_chebyshev(alpha) == 399
        p = dev(torch, psi, op.cdtype)
        s = op.sign(p)
        got = s.cpu().numpy().astype(np.complex128)
        s2 = op.sign(s).cpu().numpy().astype(np.complex128)
        side.synchronize()
    assert rel_err(got, exact) < tol
    assert rel_err(s2, psi) < 2 * tol  # sign(K)^2 = 1


@pytest.mark.parametrize("prec,tol", [("f64", 1e-10), ("f32", 1e-5)])
def test_config3_true_eigenpairs_degree400_nev50_full_size(torch, api, prec, tol):
    """BASELINE config 3 exactly as named -- 20^3 x 64, mu = 0.01, degree 400, 50 deflated eigenpairs -- with TRUE
    eigenpairs: the closed-form lowest modes of K on a pure gauge.  D[mu] psi against the FFT closed form (the polynomial's
    error on this spectrum is < 1e-11), plus sign(K) phi_i = sign(lambda_i) phi_i on two of the deflated modes."""
    U, g = inputs.pure_gauge_links(DIMS, inputs.SEED_BASE + 34)
    G = golden_gammas()
    phi, lam = lowest_pure_gauge_eigenpairs(DIMS, g, G, 50)
    psi = inputs.gaussian_spinor(DIMS, inputs.SEED_BASE + 134)
    exact, omega = free_sign_fft(DIMS, psi, G, 1.5, g)
    alpha = inputs.chebyshev_sign_coeffs(400, 0.95 * omega.min() / 6.5)
    assert np.abs(inputs.chebyshev_eval(alpha, omega.ravel() / 6.5) - 1.0).max() < 1e-11
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[None, :, None]
    want = 0.5 * (1.01 * psi + 0.99 * g5 * exact)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side), api.Overlap(DIMS, dev(torch, U), prec, stream=side) as op:
        assert op.set_chebyshev(alpha) == 399
        op.set_deflation(dev(torch, phi), lam)
        got = op.overlap(dev(torch, psi, op.cdtype), 0.01).cpu().numpy().astype(np.complex128)
        e = [op.sign(dev(torch, phi[i], op.cdtype)).cpu().numpy().astype(np.complex128) for i in (0, 49)]
        side.synchronize()
    assert rel_err(got, want) < tol
    for i, ei in zip((0, 49), e):
        assert rel_err(ei, np.sign(lam[i]) * phi[i]) < (1e-12 if prec == "f64" else tol)


@pytest.mark.parametrize("nslabs", [2, 4])
def test_split_lattice_full_size_bit_identical(torch, api, rough, nslabs):
    """SURVEY §8(f) rank 3 at 20^3 x 64: the lattice split along t into 2 and 4 slabs (32 / 16 time slices each, 250 / 125
    tiles per slab), halo stores fused into the stencil kernel: D_W and a degree-21 polynomial sign function bit-identical
    to the undivided lattice (which the tests above hold against the oracle)."""
    U, psi = rough
    alpha = inputs.chebyshev_sign_coeffs(21, 0.3)
    Ud = dev(torch, U)
    with api.Overlap(DIMS, Ud) as ref, api.SplitOverlap(DIMS, Ud, nslabs) as sp:
        p = dev(torch, psi)
        for o in (ref, sp):
            o.set_chebyshev(alpha)
        assert torch.equal(sp.dw(p), ref.dw(p))
        assert torch.equal(sp.sign(p), ref.sign(p))
        sp.set_split_launch(True)    # boundary + interior launch per round (the multi-GPU default)
        assert torch.equal(sp.sign(p), ref.sign(p))
        assert torch.equal(sp.overlap(p, 0.01, dagger=True), ref.overlap(p, 0.01, dagger=True))
