"""Worker of tests/test_gpu_split_ipc.py: run under `python -m torch.distributed.run --nproc-per-node 2` (gloo for the
plumbing; both ranks share cuda:0).  Every rank builds the same seeded global inputs, runs ITS slab of the lattice split
along t through the one-process-per-GPU wiring (CUDA IPC halos, interprocess events, shared-memory round counters), rank 0
gathers the slabs and compares with the undivided operator (bit-identical where there is no reduction) and the oracle."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    import torch
    import torch.distributed as dist

    from paper_1510_06897_b200 import api, binding, inputs
    binding.load_library()
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    torch.cuda.set_device(0)
    dims = (8, 8, 4, 16)
    V = int(np.prod(dims))
    Vl = V // world
    sl = slice(rank * Vl, (rank + 1) * Vl)
    U = inputs.config_links(dims, 0.4, 31, stout_steps=1)
    psi = inputs.gaussian_spinor(dims, 32)
    phi = inputs.orthonormal_vectors(dims, 3, 33)
    lam = np.array([0.5, -0.51, 0.52])
    alpha = inputs.chebyshev_sign_coeffs(31, 0.09)
    alpha[0], alpha[4] = 0.3, -0.2
    mu = 0.2

    def dev(a):
        return torch.from_numpy(np.ascontiguousarray(a)).cuda()

    out = {}
    with api.DistributedSplitOverlap(dims, dev(U[sl]), dist) as sp:
        sp.set_chebyshev(alpha)
        p = dev(psi[sl])
        out["dw"] = sp.dw(p).cpu().numpy()
        out["sign"] = sp.sign(p).cpu().numpy()
        out["sign2"] = sp.sign(sp.sign(p)).cpu().numpy()      # second and third apply: halo buffers and counters reused
        sp.set_deflation(dev(phi[:, sl]), lam)
        out["ovl"] = sp.overlap(p, mu).cpu().numpy()
        out["ovl_dag"] = sp.overlap(p, mu, dagger=True).cpu().numpy()
        xk, itk, _, okk = sp.cg(p, mu, tol=0.0, maxiter=5)
        out["cg5"] = xk.cpu().numpy()
        x, it, rel, ok = sp.cg(p, mu, tol=1e-9, maxiter=300)
        out["cg"] = x.cpu().numpy()
        out["cg_info"] = (it, rel, ok, itk, okk)
    gathered = [None] * world
    dist.all_gather_object(gathered, out)
    if rank == 0:
        from oracle import oracle as orc
        full = {k: np.concatenate([g[k] for g in gathered]) for k in out if k != "cg_info"}
        infos = [g["cg_info"] for g in gathered]
        assert all(i == infos[0] for i in infos), infos          # every rank saw the same scalars
        with api.Overlap(dims, dev(U)) as ref:
            ref.set_chebyshev(alpha)
            pd = dev(psi)
            assert np.array_equal(full["dw"], ref.dw(pd).cpu().numpy())
            s = ref.sign(pd)
            assert np.array_equal(full["sign"], s.cpu().numpy())
            assert np.array_equal(full["sign2"], ref.sign(s).cpu().numpy())
            ref.set_deflation(dev(phi), lam)
            yr = ref.overlap(pd, mu).cpu().numpy()
            xr, itr, relr, okr = ref.cg(pd, mu, tol=1e-9, maxiter=300)
            xr = xr.cpu().numpy()

        def rel_err(a, b):
            return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))

        assert rel_err(full["ovl"], yr) < 1e-13
        assert rel_err(full["ovl"], orc.overlap(dims, U, alpha, mu, psi, phi, lam)) < 1e-10
        assert rel_err(full["ovl_dag"], orc.overlap(dims, U, alpha, mu, psi, phi, lam, dagger=True)) < 1e-10
        want5, _, _ = orc.cg(dims, U, alpha, mu, psi, 0.0, 5, phi, lam)
        assert rel_err(full["cg5"], want5) < 1e-10
        it, rel, ok, itk, okk = infos[0]
        assert ok and okk and itk == 5 and rel < 1.05e-9 and abs(it - itr) <= 1
        assert rel_err(full["cg"], xr) < 1e-8
        print("IPC_SPLIT_OK", world, "ranks; cg iterations", it, flush=True)
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
