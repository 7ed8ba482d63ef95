"""Convenience wrapper over the C-ABI binding: owns an ovl_ctx, allocates outputs, accepts torch tensors
(CUDA or CPU) and numpy arrays.  Argument plumbing only -- every operation is one call into libovl.so."""
from __future__ import annotations

import numpy as np

from . import binding as B


def _torch():
    import torch
    return torch


class Overlap:
    """D[mu] = 1/2 (1 + mu + (1 - mu) gamma5 sign(K)), K = gamma5 (D_W - m_w)  (eq. 2.1-2.3).

    dims = (Lx, Ly, Lz, Lt); links: canonical (V,4,3,3) complex128 (numpy, CPU tensor or CUDA tensor).
    Spinors: (V,4,3) complex128 for prec='f64', complex64 for prec='f32'.
    """

    def __init__(self, dims, links, prec="f64", recon=18, stream=None, m_w=1.5, lambda_max=6.5, workspace=None):
        """workspace: None -> the library allocates its own device memory (ovl_create); a dict(max_nev=, max_rhs=,
        eig_block=) -> a torch-owned uint8 buffer of ovl_workspace_bytes is allocated here and the context lives in it
        (ovl_create_ws: no cudaMalloc / cudaFree inside any later call); a CUDA uint8 tensor with the dict under
        workspace["buffer"] is used as given."""
        torch = _torch()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1510_06897_b200 needs a CUDA device (no CPU fallback)")
        self.dims = tuple(int(d) for d in dims)
        self.V = int(np.prod(self.dims))
        self.prec = B.OVL_F64 if prec in ("f64", B.OVL_F64) else B.OVL_F32
        self.recon = int(recon)
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self.workspace = None
        if workspace is None:
            self.ctx = B.ovl_create(self.dims, links, self.prec, self.recon, self.stream.cuda_stream)
        else:
            caps = dict(max_nev=int(workspace.get("max_nev", 0)), max_rhs=int(workspace.get("max_rhs", 1)),
                        eig_block=int(workspace.get("eig_block", 0)))
            need = B.ovl_workspace_bytes(self.dims, self.prec, self.recon, **caps)
            buf = workspace.get("buffer")
            if buf is None:
                buf = torch.empty(need, dtype=torch.uint8, device="cuda")
            self.workspace, self.workspace_bytes = buf, need
            self.ctx = B.ovl_create_ws(self.dims, links, buf, self.prec, self.recon, stream=self.stream.cuda_stream, **caps)
        B.ovl_set_kernel(self.ctx, m_w, lambda_max)
        self.cdtype = torch.complex128 if self.prec == B.OVL_F64 else torch.complex64

    def close(self):
        if getattr(self, "ctx", None) is not None:
            B.ovl_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # ---- configuration
    def set_chebyshev(self, alpha):
        B.ovl_set_chebyshev(self.ctx, alpha)
        return B.ovl_poly_orders(self.ctx)

    def set_recurrence(self, mode):
        """'clenshaw' (default) or 'forward': evaluation order of the polynomial sum of eq. 2.3."""
        m = {"clenshaw": B.OVL_REC_CLENSHAW, "forward": B.OVL_REC_FORWARD}.get(mode, mode)
        B.ovl_set_recurrence(self.ctx, m)

    def set_fused_variant(self, variant):
        """'register' (default; picks the site order by lattice size), 'plain' / 'brick' (register kernel, that site order) or 'bulk' (cp.async.bulk
        landing zone for the links): same results bit for bit, see include/ovl.h."""
        v = {"register": B.OVL_FUSED_REGISTER, "bulk": B.OVL_FUSED_BULK, "plain": B.OVL_FUSED_PLAIN, "brick": B.OVL_FUSED_BRICK}.get(variant, variant)
        B.ovl_set_fused_variant(self.ctx, v)

    def set_graphs(self, on=True):
        """CUDA-graph replay of the polynomial loop (only effective when the context runs on a non-default stream)."""
        B.ovl_set_graphs(self.ctx, on)

    def set_deflation(self, phi, lam):
        B.ovl_set_deflation(self.ctx, phi, lam)

    # ---- helpers
    def _like(self, psi):
        if isinstance(psi, np.ndarray):
            return np.empty_like(psi)
        return _torch().empty_like(psi)

    def _run(self, fn, psi, *args):
        out = self._like(psi)
        fn(self.ctx, *args, psi, out)
        return out

    # ---- the path
    def dw(self, psi):
        return self._run(B.ovl_dw, psi)

    def khat(self, psi):
        return self._run(B.ovl_khat, psi)

    def sign(self, psi):
        return self._run(B.ovl_sign, psi)

    def overlap(self, psi, mu, dagger=False):
        return self._run(B.ovl_overlap, psi, mu, int(dagger))

    def overlap_multi(self, psi, mu, dagger=False):
        """psi: (nrhs, V, 4, 3); returns D[mu] psi_r for every r with the links read once per tile for all of them."""
        out = self._like(psi)
        B.ovl_overlap_multi(self.ctx, int(psi.shape[0]), mu, int(dagger), psi, out)
        return out

    def cg(self, b, mu, tol=1e-8, maxiter=1000):
        """Solve D^dag D x = b. Returns (x, iterations, true relative residual, converged)."""
        x = self._like(b)
        rc, it, rel = B.ovl_cg(self.ctx, mu, b, x, tol, maxiter)
        return x, it, rel, rc == B.OVL_OK

    def cg_chiral(self, b, mu, chirality, tol=1e-8, maxiter=1000):
        """Solve A_c x = P_c b in the chirality sector (one sign application per iteration instead of two; reading R23).
        Returns (x, iterations, true relative residual, converged)."""
        x = self._like(b)
        rc, it, rel = B.ovl_cg_chiral(self.ctx, mu, chirality, b, x, tol, maxiter)
        return x, it, rel, rc == B.OVL_OK

    def cg_multi(self, b, mu, tol=1e-8, maxiter=1000):
        """b: (nrhs, V, 4, 3). Solve D^dag D x_r = b_r in lockstep. Returns (x, iterations[], true relres[], converged)."""
        x = self._like(b)
        rc, it, rel = B.ovl_cg_multi(self.ctx, int(b.shape[0]), mu, b, x, tol, maxiter)
        return x, it, rel, rc == B.OVL_OK

    def cg_multi_chiral(self, b, mu, chirality, tol=1e-8, maxiter=1000):
        """b: (nrhs, V, 4, 3). The chiral-sector systems A_c x_r = P_c b_r in lockstep (one sign application per iteration).
        Returns (x, iterations[], true relres[], converged)."""
        x = self._like(b)
        rc, it, rel = B.ovl_cg_multi_chiral(self.ctx, int(b.shape[0]), mu, chirality, b, x, tol, maxiter)
        return x, it, rel, rc == B.OVL_OK

    def cg_mixed(self, inner, b, mu, tol=1e-8, inner_tol=1e-4, max_outer=20, max_inner=1000):
        """Mixed-precision CG: self is the fp64 operator, `inner` an fp32 Overlap on the same lattice and stream.
        Returns (x, outer steps, fp32 iterations, true fp64 relres, converged)."""
        x = self._like(b)
        rc, no, ni, rel = B.ovl_cg_mixed(self.ctx, inner.ctx, mu, b, x, tol, inner_tol, max_outer, max_inner)
        return x, no, ni, rel, rc == B.OVL_OK

    def cg_mixed_chiral(self, inner, b, mu, chirality, tol=1e-8, inner_tol=1e-4, max_outer=20, max_inner=1000):
        """cg_mixed on the chirality sector (A_c x = P_c b, one sign application per operator application).
        Returns (x, outer steps, fp32 iterations, true fp64 relres, converged)."""
        x = self._like(b)
        rc, no, ni, rel = B.ovl_cg_mixed_chiral(self.ctx, inner.ctx, mu, chirality, b, x, tol, inner_tol, max_outer, max_inner)
        return x, no, ni, rel, rc == B.OVL_OK

    def lowest_eigenpairs(self, nev, tol=1e-8, max_cycles=40, filter_degree=100, block=0):
        """Deflation space on the GPU: the nev lowest-|lambda| eigenpairs of K. Returns (phi (nev,V,4,3) complex128 CUDA
        tensor, lambda, residuals, cycles, converged)."""
        torch = _torch()
        phi = torch.empty((nev, self.V, 4, 3), dtype=torch.complex128, device="cuda")
        rc, lam, res, cyc = B.ovl_lowest_eigenpairs(self.ctx, nev, tol, max_cycles, filter_degree, block, phi)
        return phi, lam, res, cyc, rc == B.OVL_OK

    def lowest_eigenpairs_mixed(self, inner, nev, tol=1e-8, max_cycles=40, filter_degree=100, block=0):
        """The same with the filter on the fp32 kernels of `inner` (an 'f32' Overlap on the same lattice and stream) while the
        block is far from the tolerance. Returns (phi, lambda, residuals, cycles, fp32 cycles, converged)."""
        torch = _torch()
        phi = torch.empty((nev, self.V, 4, 3), dtype=torch.complex128, device="cuda")
        rc, lam, res, cyc, c32 = B.ovl_lowest_eigenpairs_mixed(self.ctx, inner.ctx, nev, tol, max_cycles, filter_degree, block, phi)
        return phi, lam, res, cyc, c32, rc == B.OVL_OK

    # ---- native-layout fields
    def native_empty(self, nrhs=1):
        torch = _torch()
        return torch.empty(B.ovl_field_bytes(self.ctx) * nrhs, dtype=torch.uint8, device="cuda")

    def to_native(self, psi):
        nat = self.native_empty()
        B.ovl_field_import(self.ctx, psi, nat)
        return nat

    def from_native(self, nat, like=None):
        torch = _torch()
        out = torch.empty((self.V, 4, 3), dtype=self.cdtype, device="cuda") if like is None else self._like(like)
        B.ovl_field_export(self.ctx, nat, out)
        return out

    def dw_native(self, nat_in, nat_out):
        B.ovl_dw_native(self.ctx, nat_in, nat_out)

    def overlap_native(self, nat_in, nat_out, mu, dagger=False):
        B.ovl_overlap_native(self.ctx, mu, int(dagger), nat_in, nat_out)

    def overlap_multi_native(self, nat_in, nat_out, nrhs, mu, dagger=False):
        B.ovl_overlap_multi_native(self.ctx, nrhs, mu, int(dagger), nat_in, nat_out)

    # ---- measurement
    def set_profiling(self, on=True):
        B.ovl_set_profiling(self.ctx, on)

    def last_poly_timing(self):
        return B.ovl_last_poly_timing(self.ctx)

    def poly_timings(self, max_n=64):
        return B.ovl_poly_timings(self.ctx, max_n)

    def launch_count(self):
        return B.ovl_launch_count(self.ctx)


class SplitOverlap:
    """The same operator on a lattice split along t into `nslabs` slabs (include/ovl.h, ovl_group_*): one slab per
    stream, optionally one per GPU (devices=[...]); halo traffic is fused into the stencil kernels as peer stores.
    Arguments and results are GLOBAL canonical fields, exactly as for Overlap."""

    def __init__(self, dims, links, nslabs, prec="f64", recon=18, devices=None, m_w=1.5, lambda_max=6.5):
        torch = _torch()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1510_06897_b200 needs a CUDA device (no CPU fallback)")
        self.dims = tuple(int(d) for d in dims)
        self.V = int(np.prod(self.dims))
        self.prec = B.OVL_F64 if prec in ("f64", B.OVL_F64) else B.OVL_F32
        self.nslabs = int(nslabs)
        self.devices = None if devices is None else [int(d) for d in devices]
        self.streams = []
        for r in range(self.nslabs):
            with torch.cuda.device(self.devices[r] if self.devices else torch.cuda.current_device()):
                self.streams.append(torch.cuda.Stream())
        torch.cuda.synchronize()
        self.grp = B.ovl_group_create(self.dims, self.nslabs, links, self.prec, int(recon),
                                      [s.cuda_stream for s in self.streams], self.devices)
        B.ovl_group_set_kernel(self.grp, m_w, lambda_max)
        self.cdtype = torch.complex128 if self.prec == B.OVL_F64 else torch.complex64

    def close(self):
        if getattr(self, "grp", None) is not None:
            B.ovl_group_destroy(self.grp)
            self.grp = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_split_launch(self, on=True):
        """Boundary launch + interior launch per stencil round (hides the cross-GPU event latency); same bits."""
        B.ovl_group_set_split_launch(self.grp, on)

    def set_chebyshev(self, alpha):
        B.ovl_group_set_chebyshev(self.grp, alpha)

    def set_deflation(self, phi, lam):
        B.ovl_group_set_deflation(self.grp, phi, lam)

    def _run(self, fn, psi, *args):
        torch = _torch()
        torch.cuda.synchronize()  # inputs may have been produced on another stream
        out = np.empty_like(psi) if isinstance(psi, np.ndarray) else torch.empty_like(psi)
        fn(self.grp, *args, psi, out)
        return out

    def dw(self, psi):
        return self._run(B.ovl_group_dw, psi)

    def khat(self, psi):
        return self._run(B.ovl_group_khat, psi)

    def sign(self, psi):
        return self._run(B.ovl_group_sign, psi)

    def overlap(self, psi, mu, dagger=False):
        return self._run(B.ovl_group_overlap, psi, mu, int(dagger))

    def cg(self, b, mu, tol=1e-8, maxiter=1000):
        torch = _torch()
        torch.cuda.synchronize()
        x = np.empty_like(b) if isinstance(b, np.ndarray) else torch.empty_like(b)
        rc, it, rel = B.ovl_group_cg(self.grp, mu, b, x, tol, maxiter)
        return x, it, rel, rc == B.OVL_OK

    def launch_count(self):
        return B.ovl_group_launch_count(self.grp)


class DistributedSplitOverlap(SplitOverlap):
    """One process per GPU (torchrun): this rank's slab of a lattice split along t over `dist.get_world_size()` ranks, wired
    to its neighbours through CUDA IPC (include/ovl.h, ovl_slab_*).  `dist` is an initialised torch.distributed (any
    backend: it only carries the handle exchange and the barriers).  Every method is collective; arguments and results are
    THIS RANK'S contiguous t-range of the canonical arrays (links (V/N,4,3,3), spinors (V/N,4,3), eigenvectors (nev,V/N,4,3))."""

    _counter = 0

    def __init__(self, dims, links_local, dist, prec="f64", recon=18, m_w=1.5, lambda_max=6.5):
        import os
        torch = _torch()
        self.dist = dist
        self.rank, self.nslabs = dist.get_rank(), dist.get_world_size()
        self.dims = tuple(int(d) for d in dims)
        self.V = int(np.prod(self.dims)) // self.nslabs
        self.prec = B.OVL_F64 if prec in ("f64", B.OVL_F64) else B.OVL_F32
        self.devices = None
        self.streams = [torch.cuda.Stream()]
        name = [f"/ovl_{os.getpid()}_{DistributedSplitOverlap._counter}"]
        DistributedSplitOverlap._counter += 1
        dist.broadcast_object_list(name, src=0)
        torch.cuda.synchronize()
        self.grp = B.ovl_slab_create(self.dims, self.rank, self.nslabs, links_local, self.prec, int(recon),
                                     self.streams[0].cuda_stream, name[0])
        blobs = [None] * self.nslabs
        dist.all_gather_object(blobs, B.ovl_slab_export(self.grp))
        B.ovl_slab_connect(self.grp, b"".join(blobs))
        dist.barrier()   # every rank's ghost links have landed before the first collective call
        B.ovl_group_set_kernel(self.grp, m_w, lambda_max)
        self.cdtype = torch.complex128 if self.prec == B.OVL_F64 else torch.complex64

    def close(self):
        if getattr(self, "grp", None) is not None:
            _torch().cuda.synchronize()
            self.dist.barrier()  # nobody unmaps memory a neighbour may still be writing
            B.ovl_group_destroy(self.grp)
            self.grp = None
