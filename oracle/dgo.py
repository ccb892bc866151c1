"""ctypes front end of the CPU oracle oracle/dgo.c (test infrastructure, not the product).

All arrays are HOST numpy arrays in the structure-of-arrays layouts of include/dg.h
(rho_g[ncells], rho_d[N][ncells], t_s[N][ncells], p[3][n][ncells], A/E[n*n][ncells]); inputs are
float64, results are numpy.longdouble (x87 80-bit) so that the comparison with the CUDA output is
itself carried out in extended precision.
"""
import ctypes as C

import numpy as np

from . import build as _build

_lib = None
LD = np.longdouble


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        if L.dgo_sizeof_long_double() != np.dtype(LD).itemsize or L.dgo_ldbl_mant_dig() != np.finfo(LD).nmant + 1:
            raise RuntimeError("numpy.longdouble does not match the C compiler's long double")
        L.dgo_max_threads.restype = C.c_int
        _lib = L
    return _lib


def max_threads() -> int:
    return int(lib().dgo_max_threads())


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.c_void_p)


def _shape_check(rho_g, rho_d, t_s, N):
    ncells = rho_g.shape[0]
    assert rho_g.shape == (ncells,) and rho_d.shape == (N, ncells) and t_s.shape == (N, ncells)
    return ncells


def drag_matrix_build(rho_g, rho_d, t_s, dt, nthreads=0):
    """Stage a1 (Eq. 14, 15, 17): returns A = dt*Omega as longdouble [n*n][ncells]."""
    N = rho_d.shape[0]
    rho_g, prg = _f64(rho_g); rho_d, prd = _f64(rho_d); t_s, pts = _f64(t_s)
    ncells = _shape_check(rho_g, rho_d, t_s, N)
    n = N + 1
    A = np.empty((n * n, ncells), dtype=LD)
    rc = lib().dgo_drag_matrix_build(prg, prd, pts, C.c_double(dt), C.c_int(N), C.c_longlong(ncells),
                                     A.ctypes.data_as(C.c_void_p), C.c_int(nthreads))
    assert rc == 0
    return A


def expm_batch(A, N, rebuild_diag=True, nthreads=0):
    """Stages a2-a4 on fp64 drag matrices A[n*n][ncells]: returns (E longdouble [n*n][ncells], s int32[ncells])."""
    A, pA = _f64(A)
    n = N + 1
    ncells = A.shape[1]
    assert A.shape == (n * n, ncells)
    E = np.empty((n * n, ncells), dtype=LD)
    s = np.empty(ncells, dtype=np.int32)
    rc = lib().dgo_expm_batch(pA, C.c_int(N), C.c_longlong(ncells), C.c_int(1 if rebuild_diag else 0),
                              E.ctypes.data_as(C.c_void_p), s.ctypes.data_as(C.c_void_p), C.c_int(nthreads))
    assert rc == 0
    return E, s


def drag_apply(E, p_in, N, nthreads=0):
    """Stage a5 (Eq. 18) with E given in fp64: returns p_out longdouble [3][n][ncells]."""
    E, pE = _f64(E); p_in, pp = _f64(p_in)
    n = N + 1
    ncells = E.shape[1]
    assert E.shape == (n * n, ncells) and p_in.shape == (3, n, ncells)
    out = np.empty((3, n, ncells), dtype=LD)
    rc = lib().dgo_drag_apply(pE, pp, C.c_int(N), C.c_longlong(ncells), out.ctypes.data_as(C.c_void_p), C.c_int(nthreads))
    assert rc == 0
    return out


def drag_update(rho_g, rho_d, t_s, dt, p_in, want_E=False, nthreads=0):
    """Whole path a1..a5: returns p_out longdouble [3][n][ncells] (and E [n*n][ncells], s[ncells] if want_E)."""
    N = rho_d.shape[0]
    rho_g, prg = _f64(rho_g); rho_d, prd = _f64(rho_d); t_s, pts = _f64(t_s); p_in, pp = _f64(p_in)
    ncells = _shape_check(rho_g, rho_d, t_s, N)
    n = N + 1
    assert p_in.shape == (3, n, ncells)
    out = np.empty((3, n, ncells), dtype=LD)
    E = np.empty((n * n, ncells), dtype=LD) if want_E else None
    s = np.empty(ncells, dtype=np.int32) if want_E else None
    rc = lib().dgo_drag_update(prg, prd, pts, C.c_double(dt), pp, C.c_int(N), C.c_longlong(ncells),
                               out.ctypes.data_as(C.c_void_p),
                               E.ctypes.data_as(C.c_void_p) if want_E else None,
                               s.ctypes.data_as(C.c_void_p) if want_E else None, C.c_int(nthreads))
    assert rc == 0
    return (out, E, s) if want_E else out


def rk1_update(rho_g, rho_d, t_s, dt, p_in, nthreads=0):
    """First-order implicit RK1 drag step (App. A.1, Eq. A.6): p_out = (I - dt*Omega)^-1 p_in by a dense solve,
    longdouble [3][n][ncells]."""
    N = rho_d.shape[0]
    rho_g, prg = _f64(rho_g); rho_d, prd = _f64(rho_d); t_s, pts = _f64(t_s); p_in, pp = _f64(p_in)
    ncells = _shape_check(rho_g, rho_d, t_s, N)
    n = N + 1
    assert p_in.shape == (3, n, ncells)
    out = np.empty((3, n, ncells), dtype=LD)
    rc = lib().dgo_rk1_update(prg, prd, pts, C.c_double(dt), pp, C.c_int(N), C.c_longlong(ncells),
                              out.ctypes.data_as(C.c_void_p), C.c_int(nthreads))
    assert rc == 0
    return out


def energy_update(rho_g, rho_d, t_s, dt, p_in, E_in, w, nthreads=0):
    """Gas energy after one exact drag step with frictional heating (Eq. 4; R20): returns
    (E_out longdouble [ncells], p_out longdouble [3][n][ncells])."""
    N = rho_d.shape[0]
    rho_g, prg = _f64(rho_g); rho_d, prd = _f64(rho_d); t_s, pts = _f64(t_s); p_in, pp = _f64(p_in); E_in, pe = _f64(E_in)
    ncells = _shape_check(rho_g, rho_d, t_s, N)
    n = N + 1
    assert p_in.shape == (3, n, ncells) and E_in.shape == (ncells,)
    E_out = np.empty(ncells, dtype=LD)
    p_out = np.empty((3, n, ncells), dtype=LD)
    rc = lib().dgo_energy_update(prg, prd, pts, C.c_double(dt), pp, pe, C.c_double(w), C.c_int(N), C.c_longlong(ncells),
                                 E_out.ctypes.data_as(C.c_void_p), p_out.ctypes.data_as(C.c_void_p), C.c_int(nthreads))
    assert rc == 0
    return E_out, p_out


def parity_error(p_gpu, p_ref, p_in):
    """DESIGN.md reading R13: per cell, max_{k,comp}|p_gpu - p_ref| / max_{k,comp}|p_in|, in long double."""
    d = np.abs(np.asarray(p_gpu, dtype=LD) - np.asarray(p_ref, dtype=LD)).reshape(-1, p_ref.shape[-1]).max(axis=0)
    scale = np.abs(np.asarray(p_in, dtype=LD)).reshape(-1, p_ref.shape[-1]).max(axis=0)
    return d / scale


def conservation_error(p_out, p_in):
    """R13: per cell and component |sum_k p_out - sum_k p_in| / sum_k |p_in|, sums in long double. Needs no oracle."""
    po = np.asarray(p_out, dtype=LD); pi = np.asarray(p_in, dtype=LD)
    return np.abs(po.sum(axis=1) - pi.sum(axis=1)) / np.abs(pi).sum(axis=1)
