"""The lattice split along t on ONE GPU: 1, 2 and 4 slab contexts
in their own streams, halo traffic fused into the stencil kernels (stores into the neighbour slab's halo buffers, which on
several GPUs are peer pointers), ordered by events only.  D_W, K^ and the polynomial sign function must be BIT-IDENTICAL to
the undivided lattice; with deflation and in CG the reductions are partitioned differently (rounding-level differences).
Everything is also held against the oracle."""
import numpy as np
import pytest

from paper_1510_06897_b200 import inputs
from tests.conftest import rel_err

pytestmark = pytest.mark.gpu


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


def dev(torch, a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t.to(dtype) if dtype is not None else t


def host(t):
    return t.detach().cpu().numpy().astype(np.complex128)


@pytest.mark.parametrize("split_launch", [False, True])
@pytest.mark.parametrize("nslabs", [1, 2, 4])
@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f64", 12), ("f32", 18)])
def test_split_stencil_and_polynomial_bit_identical(torch, api, orc, nslabs, prec, recon, split_launch):
    """split_launch: every stencil round as a boundary launch + an interior launch with the round's event in between (the
    multi-GPU default); 8 x 8 x 4 x 16 has 256-site time slices, i.e. whole 128-site tiles, so the split really happens
    (for 4 slabs of 4 time slices: 4 boundary + 4 interior tiles per slab)."""
    dims = (8, 8, 4, 16)
    U = inputs.config_links(dims, 0.4, 31, stout_steps=1)
    psi = inputs.gaussian_spinor(dims, 32)
    alpha = inputs.chebyshev_sign_coeffs(31, 0.09)
    alpha[0], alpha[4] = 0.3, -0.2          # generic table: psi term present in odd and even launches
    Ud = dev(torch, U)
    with api.Overlap(dims, Ud, prec, recon) as ref, api.SplitOverlap(dims, Ud, nslabs, prec, recon) as sp:
        p = dev(torch, psi, ref.cdtype)
        for o in (ref, sp):
            o.set_chebyshev(alpha)
        sp.set_split_launch(split_launch)
        assert torch.equal(sp.dw(p), ref.dw(p))
        assert torch.equal(sp.khat(p), ref.khat(p))
        s_split, s_ref = sp.sign(p), ref.sign(p)
        assert torch.equal(s_split, s_ref)
        assert torch.equal(sp.overlap(p, 0.05), ref.overlap(p, 0.05))
        assert torch.equal(sp.overlap(p, 0.05, dagger=True), ref.overlap(p, 0.05, dagger=True))
        # a second application reuses the halo buffers and the event chain
        assert torch.equal(sp.sign(s_split), ref.sign(s_ref))
        got_dw = host(sp.dw(p))
    tol = 1e-12 if prec == "f64" else 1e-5
    assert rel_err(got_dw, orc.dw(dims, U, psi)) < tol
    assert rel_err(host(s_split), orc.sign(dims, U, alpha, psi)) < (1e-10 if prec == "f64" else 1e-5)


@pytest.mark.parametrize("split_launch", [False, True])
@pytest.mark.parametrize("nslabs", [2, 4])
def test_split_deflated_overlap_and_cg(torch, api, orc, nslabs, split_launch):
    dims = (8, 4, 4, 16)
    U = inputs.config_links(dims, 0.3, 41, stout_steps=2)
    psi = inputs.gaussian_spinor(dims, 42)
    phi = inputs.orthonormal_vectors(dims, 5, 43)
    lam = np.array([0.5, -0.51, 0.52, -0.53, 0.54])
    alpha = inputs.chebyshev_sign_coeffs(61, 0.075)
    mu = 0.2
    Ud, phid = dev(torch, U), dev(torch, phi)
    with api.Overlap(dims, Ud) as ref, api.SplitOverlap(dims, Ud, nslabs) as sp:
        for o in (ref, sp):
            o.set_chebyshev(alpha)
            o.set_deflation(phid, lam)
        sp.set_split_launch(split_launch)
        p = dev(torch, psi)
        y, yr = host(sp.overlap(p, mu)), host(ref.overlap(p, mu))
        yd = host(sp.overlap(p, mu, dagger=True))
        xk, itk, _, okk = sp.cg(p, mu, tol=0.0, maxiter=6)
        x, it, rel, ok = sp.cg(p, mu, tol=1e-9, maxiter=500)
        xr, itr, relr, okr = ref.cg(p, mu, tol=1e-9, maxiter=500)
        hy = sp.overlap(psi, mu)             # host arrays in and out
    assert rel_err(y, yr) < 1e-13            # same operator, reductions partitioned differently
    assert rel_err(y, orc.overlap(dims, U, alpha, mu, psi, phi, lam)) < 1e-10
    assert rel_err(yd, orc.overlap(dims, U, alpha, mu, psi, phi, lam, dagger=True)) < 1e-10
    assert np.array_equal(hy, y)
    want, _, _ = orc.cg(dims, U, alpha, mu, psi, 0.0, 6, phi, lam)
    assert itk == 6 and okk and rel_err(host(xk), want) < 1e-10
    assert ok and okr and abs(it - itr) <= 1 and rel < 1.05e-9
    assert rel_err(host(x), host(xr)) < 1e-8


def test_split_argument_checks(torch, api):
    from paper_1510_06897_b200 import binding as B
    dims = (4, 4, 4, 8)
    Ud = dev(torch, inputs.random_links(dims, 0.3, 5))
    for bad in (3, 8, 0):                    # Lt % nslabs != 0, Lt / nslabs < 2, nslabs < 1
        with pytest.raises(B.OvlError):
            api.SplitOverlap(dims, Ud, bad)
    with api.SplitOverlap(dims, Ud, 2) as sp:
        with pytest.raises(B.OvlError) as e:
            sp.sign(dev(torch, inputs.gaussian_spinor(dims, 6)))
        assert e.value.code == B.OVL_ESTATE
