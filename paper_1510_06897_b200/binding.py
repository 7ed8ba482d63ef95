"""Thin ctypes binding of the C-ABI in include/ovl.h -- same names, argument marshalling only.

Every step of the path runs inside libovl.so's CUDA kernels.  There is no CPU fallback: if the library
is missing or cannot be loaded, importing a symbol from it raises.  PyTorch supplies device memory and
streams; numpy arrays are passed as host pointers (the library stages them itself).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

OVL_OK, OVL_EINVAL, OVL_ENOMEM, OVL_ECUDA, OVL_ESTATE, OVL_ENOTCONV = range(6)
OVL_F64, OVL_F32 = 0, 1
OVL_RECON18, OVL_RECON12 = 18, 12
OVL_REC_CLENSHAW, OVL_REC_FORWARD = 0, 1
OVL_FUSED_REGISTER, OVL_FUSED_BULK, OVL_FUSED_PLAIN, OVL_FUSED_BRICK = 0, 1, 2, 3
OVL_MAX_RHS = 12

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libovl.so")

# name -> (restype, argtypes); mirrors include/ovl.h one to one (tests/test_abi.py checks the header against this)
_P, _I, _D = C.c_void_p, C.c_int, C.c_double
SIGNATURES = {
    "ovl_version": (C.c_char_p, []),
    "ovl_workspace_bytes": (C.c_size_t, [C.POINTER(_I), _I, _I, _I, _I, _I]),
    "ovl_device_bytes": (C.c_size_t, [C.POINTER(_I), _I, _I, _I]),
    "ovl_create_ws": (_I, [C.POINTER(_P), C.POINTER(_I), _P, _I, _I, _I, _I, _I, _P, C.c_size_t, _P]),
    "ovl_create": (_I, [C.POINTER(_P), C.POINTER(_I), _P, _I, _I, _P]),
    "ovl_destroy": (_I, [_P]),
    "ovl_set_kernel": (_I, [_P, _D, _D]),
    "ovl_set_chebyshev": (_I, [_P, _I, C.POINTER(_D)]),
    "ovl_poly_orders": (_I, [_P]),
    "ovl_set_recurrence": (_I, [_P, _I]),
    "ovl_get_recurrence": (_I, [_P]),
    "ovl_set_graphs": (_I, [_P, _I]),
    "ovl_set_fused_variant": (_I, [_P, _I]),
    "ovl_set_deflation": (_I, [_P, _I, _P, C.POINTER(_D)]),
    "ovl_dw": (_I, [_P, _P, _P]),
    "ovl_khat": (_I, [_P, _P, _P]),
    "ovl_sign": (_I, [_P, _P, _P]),
    "ovl_overlap": (_I, [_P, _D, _I, _P, _P]),
    "ovl_overlap_multi": (_I, [_P, _I, _D, _I, _P, _P]),
    "ovl_cg": (_I, [_P, _D, _P, _P, _D, _I, C.POINTER(_I), C.POINTER(_D)]),
    "ovl_cg_chiral": (_I, [_P, _D, _I, _P, _P, _D, _I, C.POINTER(_I), C.POINTER(_D)]),
    "ovl_cg_multi": (_I, [_P, _I, _D, _P, _P, _D, _I, C.POINTER(_I), C.POINTER(_D)]),
    "ovl_cg_multi_chiral": (_I, [_P, _I, _D, _I, _P, _P, _D, _I, C.POINTER(_I), C.POINTER(_D)]),
    "ovl_cg_mixed": (_I, [_P, _P, _D, _P, _P, _D, _D, _I, _I, C.POINTER(_I), C.POINTER(_I), C.POINTER(_D)]),
    "ovl_cg_mixed_chiral": (_I, [_P, _P, _D, _I, _P, _P, _D, _D, _I, _I, C.POINTER(_I), C.POINTER(_I), C.POINTER(_D)]),
    "ovl_lowest_eigenpairs": (_I, [_P, _I, _D, _I, _I, _I, _P, C.POINTER(_D), C.POINTER(_D), C.POINTER(_I)]),
    "ovl_lowest_eigenpairs_mixed": (_I, [_P, _P, _I, _D, _I, _I, _I, _P, C.POINTER(_D), C.POINTER(_D), C.POINTER(_I), C.POINTER(_I)]),
    "ovl_last_error": (C.c_char_p, [_P]),
    "ovl_group_create": (_I, [C.POINTER(_P), C.POINTER(_I), _I, _P, _I, _I, C.POINTER(_P), C.POINTER(_I)]),
    "ovl_group_destroy": (_I, [_P]),
    "ovl_group_slabs": (_I, [_P]),
    "ovl_group_set_split_launch": (_I, [_P, _I]),
    "ovl_group_set_kernel": (_I, [_P, _D, _D]),
    "ovl_group_set_chebyshev": (_I, [_P, _I, C.POINTER(_D)]),
    "ovl_group_set_deflation": (_I, [_P, _I, _P, C.POINTER(_D)]),
    "ovl_group_dw": (_I, [_P, _P, _P]),
    "ovl_group_khat": (_I, [_P, _P, _P]),
    "ovl_group_sign": (_I, [_P, _P, _P]),
    "ovl_group_overlap": (_I, [_P, _D, _I, _P, _P]),
    "ovl_group_cg": (_I, [_P, _D, _P, _P, _D, _I, C.POINTER(_I), C.POINTER(_D)]),
    "ovl_slab_create": (_I, [C.POINTER(_P), C.POINTER(_I), _I, _I, _P, _I, _I, _P, C.c_char_p]),
    "ovl_slab_export": (_I, [_P, _P]),
    "ovl_slab_connect": (_I, [_P, _P]),
    "ovl_group_last_error": (C.c_char_p, [_P]),
    "ovl_group_launch_count": (C.c_longlong, [_P]),
    "ovl_field_bytes": (C.c_size_t, [_P]),
    "ovl_field_import": (_I, [_P, _P, _P]),
    "ovl_field_export": (_I, [_P, _P, _P]),
    "ovl_dw_native": (_I, [_P, _P, _P]),
    "ovl_overlap_native": (_I, [_P, _D, _I, _P, _P]),
    "ovl_overlap_multi_native": (_I, [_P, _I, _D, _I, _P, _P]),
    "ovl_set_profiling": (_I, [_P, _I]),
    "ovl_last_poly_timing": (_I, [_P, C.POINTER(C.c_float), C.POINTER(_I)]),
    "ovl_poly_timings": (_I, [_P, _I, C.POINTER(C.c_float), C.POINTER(_I)]),
    "ovl_launch_count": (C.c_longlong, [_P]),
}

_lib = None


class OvlError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"ovl status {code}: {msg}")
        self.code = code


def load_library(path: str = LIB_PATH) -> C.CDLL:
    """dlopen libovl.so and declare every prototype. Raises if the library is absent (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(path):
            raise ImportError(
                f"{path} is missing: build it with `python -m paper_1510_06897_b200.build` "
                "(there is no CPU fallback for the overlap path)")
        lib = C.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def _ptr(a):
    """Raw address of a torch tensor (device or CPU) or a numpy array; contiguity is the caller's contract."""
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("numpy arguments must be C-contiguous")
        return C.c_void_p(a.ctypes.data)
    if hasattr(a, "data_ptr"):
        if not a.is_contiguous():
            raise ValueError("tensor arguments must be contiguous")
        return C.c_void_p(a.data_ptr())
    if a is None:
        return C.c_void_p(0)
    return C.c_void_p(int(a))


def _dbl(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(_D))


def _check(ctx, rc, ok=(OVL_OK,)):
    if rc not in ok:
        msg = load_library().ovl_last_error(ctx).decode() if ctx else "no context"
        raise OvlError(rc, msg)
    return rc


# ------------------------------------------------------------------ same names as the C-ABI

def ovl_version() -> str:
    return load_library().ovl_version().decode()


def ovl_device_bytes(dims, prec=OVL_F64, recon=OVL_RECON18, max_nev=0) -> int:
    return int(load_library().ovl_device_bytes((_I * 4)(*map(int, dims)), prec, recon, max_nev))


def ovl_workspace_bytes(dims, prec=OVL_F64, recon=OVL_RECON18, max_nev=0, max_rhs=1, eig_block=0) -> int:
    return int(load_library().ovl_workspace_bytes((_I * 4)(*map(int, dims)), prec, recon, max_nev, max_rhs, eig_block))


def ovl_create_ws(dims, links, workspace, prec=OVL_F64, recon=OVL_RECON18, max_nev=0, max_rhs=1, eig_block=0, stream=0):
    """Context inside a caller-owned device workspace (a torch uint8 CUDA tensor of >= ovl_workspace_bytes bytes)."""
    ctx = _P()
    nbytes = workspace.numel() * workspace.element_size()
    rc = load_library().ovl_create_ws(C.byref(ctx), (_I * 4)(*map(int, dims)), _ptr(links), prec, recon, max_nev, max_rhs,
                                      eig_block, _ptr(workspace), nbytes, _P(int(stream)))
    if rc != OVL_OK:
        raise OvlError(rc, "ovl_create_ws failed (bad workspace / arguments)")
    return ctx


def ovl_create(dims, links, prec=OVL_F64, recon=OVL_RECON18, stream=0):
    ctx = _P()
    rc = load_library().ovl_create(C.byref(ctx), (_I * 4)(*map(int, dims)), _ptr(links), prec, recon, _P(int(stream)))
    if rc != OVL_OK:
        raise OvlError(rc, "ovl_create failed")
    return ctx


def ovl_destroy(ctx):
    return _check(None, load_library().ovl_destroy(ctx))


def ovl_set_kernel(ctx, m_w=1.5, lambda_max=6.5):
    return _check(ctx, load_library().ovl_set_kernel(ctx, m_w, lambda_max))


def ovl_set_chebyshev(ctx, alpha):
    a, p = _dbl(alpha)
    return _check(ctx, load_library().ovl_set_chebyshev(ctx, len(a) - 1, p))


def ovl_poly_orders(ctx) -> int:
    return int(load_library().ovl_poly_orders(ctx))


def ovl_set_recurrence(ctx, mode):
    return _check(ctx, load_library().ovl_set_recurrence(ctx, int(mode)))


def ovl_get_recurrence(ctx) -> int:
    return int(load_library().ovl_get_recurrence(ctx))


def ovl_set_fused_variant(ctx, variant):
    return _check(ctx, load_library().ovl_set_fused_variant(ctx, int(variant)))


def ovl_set_graphs(ctx, on=True):
    return _check(ctx, load_library().ovl_set_graphs(ctx, int(bool(on))))


def ovl_set_deflation(ctx, phi, lam):
    l, p = _dbl(lam)
    return _check(ctx, load_library().ovl_set_deflation(ctx, len(l), _ptr(phi) if len(l) else _P(0), p))


def ovl_dw(ctx, psi, out):
    return _check(ctx, load_library().ovl_dw(ctx, _ptr(psi), _ptr(out)))


def ovl_khat(ctx, psi, out):
    return _check(ctx, load_library().ovl_khat(ctx, _ptr(psi), _ptr(out)))


def ovl_sign(ctx, psi, out):
    return _check(ctx, load_library().ovl_sign(ctx, _ptr(psi), _ptr(out)))


def ovl_overlap(ctx, mu, dagger, psi, out):
    return _check(ctx, load_library().ovl_overlap(ctx, float(mu), int(dagger), _ptr(psi), _ptr(out)))


def ovl_overlap_multi(ctx, nrhs, mu, dagger, psi, out):
    return _check(ctx, load_library().ovl_overlap_multi(ctx, int(nrhs), float(mu), int(dagger), _ptr(psi), _ptr(out)))


def ovl_overlap_multi_native(ctx, nrhs, mu, dagger, in_native, out_native):
    return _check(ctx, load_library().ovl_overlap_multi_native(ctx, int(nrhs), float(mu), int(dagger), _ptr(in_native), _ptr(out_native)))


def ovl_cg(ctx, mu, b, x, tol, maxiter):
    """Returns (status, iterations, true relative residual); status is OVL_OK or OVL_ENOTCONV."""
    it, rel = _I(0), _D(0.0)
    rc = load_library().ovl_cg(ctx, float(mu), _ptr(b), _ptr(x), float(tol), int(maxiter), C.byref(it), C.byref(rel))
    _check(ctx, rc, ok=(OVL_OK, OVL_ENOTCONV))
    return rc, int(it.value), float(rel.value)


def ovl_cg_chiral(ctx, mu, chirality, b, x, tol, maxiter):
    """Returns (status, iterations, true relative residual) of the chiral-sector solve A_c x = P_c b."""
    it, rel = _I(0), _D(0.0)
    rc = load_library().ovl_cg_chiral(ctx, float(mu), int(chirality), _ptr(b), _ptr(x), float(tol), int(maxiter),
                                      C.byref(it), C.byref(rel))
    _check(ctx, rc, ok=(OVL_OK, OVL_ENOTCONV))
    return rc, int(it.value), float(rel.value)


def ovl_cg_multi(ctx, nrhs, mu, b, x, tol, maxiter):
    """Returns (status, iterations per system, true relative residual per system)."""
    it, rel = (_I * nrhs)(), (_D * nrhs)()
    rc = load_library().ovl_cg_multi(ctx, int(nrhs), float(mu), _ptr(b), _ptr(x), float(tol), int(maxiter), it, rel)
    _check(ctx, rc, ok=(OVL_OK, OVL_ENOTCONV))
    return rc, list(it), list(rel)


def ovl_cg_multi_chiral(ctx, nrhs, mu, chirality, b, x, tol, maxiter):
    """Returns (status, iterations per system, true relative residual per system) of the chiral-sector systems."""
    it, rel = (_I * nrhs)(), (_D * nrhs)()
    rc = load_library().ovl_cg_multi_chiral(ctx, int(nrhs), float(mu), int(chirality), _ptr(b), _ptr(x), float(tol), int(maxiter), it, rel)
    _check(ctx, rc, ok=(OVL_OK, OVL_ENOTCONV))
    return rc, list(it), list(rel)


def ovl_cg_mixed(ctx64, ctx32, mu, b, x, tol, inner_tol, max_outer, max_inner):
    """Returns (status, outer steps, total fp32 iterations, true fp64 relative residual)."""
    no, ni, rel = _I(0), _I(0), _D(0.0)
    rc = load_library().ovl_cg_mixed(ctx64, ctx32, float(mu), _ptr(b), _ptr(x), float(tol), float(inner_tol), int(max_outer),
                                     int(max_inner), C.byref(no), C.byref(ni), C.byref(rel))
    _check(ctx64, rc, ok=(OVL_OK, OVL_ENOTCONV))
    return rc, int(no.value), int(ni.value), float(rel.value)


def ovl_cg_mixed_chiral(ctx64, ctx32, mu, chirality, b, x, tol, inner_tol, max_outer, max_inner):
    """Returns (status, outer steps, total fp32 iterations, true fp64 relative residual of the sector system)."""
    no, ni, rel = _I(0), _I(0), _D(0.0)
    rc = load_library().ovl_cg_mixed_chiral(ctx64, ctx32, float(mu), int(chirality), _ptr(b), _ptr(x), float(tol), float(inner_tol),
                                            int(max_outer), int(max_inner), C.byref(no), C.byref(ni), C.byref(rel))
    _check(ctx64, rc, ok=(OVL_OK, OVL_ENOTCONV))
    return rc, int(no.value), int(ni.value), float(rel.value)


def ovl_lowest_eigenpairs(ctx, nev, tol, max_cycles, filter_degree, block, phi_out):
    """Returns (status, lambda[nev], residual[nev], cycles); phi_out is filled with nev canonical complex128 spinors."""
    lam, res, cyc = (_D * nev)(), (_D * nev)(), _I(0)
    rc = load_library().ovl_lowest_eigenpairs(ctx, int(nev), float(tol), int(max_cycles), int(filter_degree), int(block),
                                              _ptr(phi_out), lam, res, C.byref(cyc))
    _check(ctx, rc, ok=(OVL_OK, OVL_ENOTCONV))
    return rc, np.array(lam), np.array(res), int(cyc.value)


def ovl_lowest_eigenpairs_mixed(ctx64, ctx32, nev, tol, max_cycles, filter_degree, block, phi_out):
    """Returns (status, lambda[nev], residual[nev], cycles, fp32 filter cycles); phi_out as ovl_lowest_eigenpairs."""
    lam, res, cyc, c32 = (_D * nev)(), (_D * nev)(), _I(0), _I(0)
    rc = load_library().ovl_lowest_eigenpairs_mixed(ctx64, ctx32, int(nev), float(tol), int(max_cycles), int(filter_degree),
                                                    int(block), _ptr(phi_out), lam, res, C.byref(cyc), C.byref(c32))
    _check(ctx64, rc, ok=(OVL_OK, OVL_ENOTCONV))
    return rc, np.array(lam), np.array(res), int(cyc.value), int(c32.value)


def ovl_last_error(ctx) -> str:
    return load_library().ovl_last_error(ctx).decode()


def ovl_field_bytes(ctx) -> int:
    return int(load_library().ovl_field_bytes(ctx))


def ovl_field_import(ctx, canonical, native):
    return _check(ctx, load_library().ovl_field_import(ctx, _ptr(canonical), _ptr(native)))


def ovl_field_export(ctx, native, canonical):
    return _check(ctx, load_library().ovl_field_export(ctx, _ptr(native), _ptr(canonical)))


def ovl_dw_native(ctx, in_native, out_native):
    return _check(ctx, load_library().ovl_dw_native(ctx, _ptr(in_native), _ptr(out_native)))


def ovl_overlap_native(ctx, mu, dagger, in_native, out_native):
    return _check(ctx, load_library().ovl_overlap_native(ctx, float(mu), int(dagger), _ptr(in_native), _ptr(out_native)))


def ovl_set_profiling(ctx, on=True):
    return _check(ctx, load_library().ovl_set_profiling(ctx, int(bool(on))))


def ovl_last_poly_timing(ctx):
    """(milliseconds of the last profiled polynomial loop, fused-kernel launches in it)."""
    ms, n = C.c_float(0.0), _I(0)
    _check(ctx, load_library().ovl_last_poly_timing(ctx, C.byref(ms), C.byref(n)))
    return float(ms.value), int(n.value)


def ovl_poly_timings(ctx, max_n=64):
    """Loop times (ms) of the last up-to-max_n profiled polynomial loops, oldest first."""
    buf, n = (C.c_float * int(max_n))(), _I(0)
    _check(ctx, load_library().ovl_poly_timings(ctx, int(max_n), buf, C.byref(n)))
    return [float(buf[i]) for i in range(n.value)]


def ovl_launch_count(ctx) -> int:
    return int(load_library().ovl_launch_count(ctx))


# ------------------------------------------------------------------ t-split lattice (ovl_group_*)

def _gcheck(g, rc, ok=(OVL_OK,)):
    if rc not in ok:
        raise OvlError(rc, load_library().ovl_group_last_error(g).decode() if g else "no group")
    return rc


def ovl_group_create(dims, nslabs, links, prec=OVL_F64, recon=OVL_RECON18, streams=(), devices=None):
    g = _P()
    st = (_P * nslabs)(*[_P(int(s)) for s in streams])
    dv = (_I * nslabs)(*map(int, devices)) if devices is not None else None
    rc = load_library().ovl_group_create(C.byref(g), (_I * 4)(*map(int, dims)), int(nslabs), _ptr(links), prec, recon, st, dv)
    if rc != OVL_OK:
        raise OvlError(rc, "ovl_group_create failed")
    return g


OVL_SLAB_BLOB_BYTES = 256


def ovl_slab_create(dims, rank, nranks, links_local, prec=OVL_F64, recon=OVL_RECON18, stream=0, shm_name="/ovl_group"):
    """This process's slab of a lattice split along t over `nranks` processes (one per GPU)."""
    g = _P()
    rc = load_library().ovl_slab_create(C.byref(g), (_I * 4)(*map(int, dims)), int(rank), int(nranks), _ptr(links_local), prec, recon,
                                        _P(int(stream)), shm_name.encode())
    if rc != OVL_OK:
        raise OvlError(rc, "ovl_slab_create failed")
    return g


def ovl_slab_export(g) -> bytes:
    buf = C.create_string_buffer(OVL_SLAB_BLOB_BYTES)
    _gcheck(g, load_library().ovl_slab_export(g, buf))
    return buf.raw


def ovl_slab_connect(g, blobs: bytes):
    buf = C.create_string_buffer(blobs, len(blobs))
    return _gcheck(g, load_library().ovl_slab_connect(g, buf))


def ovl_group_destroy(g):
    return load_library().ovl_group_destroy(g)


def ovl_group_slabs(g) -> int:
    return int(load_library().ovl_group_slabs(g))


def ovl_group_set_split_launch(g, on=True):
    return _gcheck(g, load_library().ovl_group_set_split_launch(g, int(bool(on))))


def ovl_group_set_kernel(g, m_w=1.5, lambda_max=6.5):
    return _gcheck(g, load_library().ovl_group_set_kernel(g, float(m_w), float(lambda_max)))


def ovl_group_set_chebyshev(g, alpha):
    a, p = _dbl(alpha)
    return _gcheck(g, load_library().ovl_group_set_chebyshev(g, len(a) - 1, p))


def ovl_group_set_deflation(g, phi, lam):
    l, p = _dbl(lam)
    return _gcheck(g, load_library().ovl_group_set_deflation(g, len(l), _ptr(phi), p))


def ovl_group_dw(g, psi, out):
    return _gcheck(g, load_library().ovl_group_dw(g, _ptr(psi), _ptr(out)))


def ovl_group_khat(g, psi, out):
    return _gcheck(g, load_library().ovl_group_khat(g, _ptr(psi), _ptr(out)))


def ovl_group_sign(g, psi, out):
    return _gcheck(g, load_library().ovl_group_sign(g, _ptr(psi), _ptr(out)))


def ovl_group_overlap(g, mu, dagger, psi, out):
    return _gcheck(g, load_library().ovl_group_overlap(g, float(mu), int(dagger), _ptr(psi), _ptr(out)))


def ovl_group_cg(g, mu, b, x, tol, maxiter):
    it, rel = _I(0), _D(0.0)
    rc = load_library().ovl_group_cg(g, float(mu), _ptr(b), _ptr(x), float(tol), int(maxiter), C.byref(it), C.byref(rel))
    _gcheck(g, rc, ok=(OVL_OK, OVL_ENOTCONV))
    return rc, int(it.value), float(rel.value)


def ovl_group_last_error(g) -> str:
    return load_library().ovl_group_last_error(g).decode()


def ovl_group_launch_count(g) -> int:
    return int(load_library().ovl_group_launch_count(g))
