"""Thin ctypes binding over libdg.so (include/dg.h): argument marshalling only — every step of the path runs in
the CUDA kernels of the library.  Function names are those of the C ABI.

Device entry points take torch CUDA float64 tensors in the layouts of include/dg.h and enqueue on torch's current
stream; PyTorch is used for device memory and streams only.  There is no CPU fallback: if libdg.so is missing or
cannot be loaded, importing this module raises.
"""
import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libdg.so")

DG_NMAX = 16
DG_OK, DG_EINVAL, DG_ENULL, DG_EALIGN, DG_ERANGE, DG_ECUDA, DG_ECAPACITY = range(7)
DG_STATIC_STAGE_BYTES = 32 << 20
(DG_VARIANT_DEFAULT, DG_VARIANT_TPC, DG_VARIANT_WPC, DG_VARIANT_PAPER, DG_VARIANT_PPC, DG_VARIANT_PAPER_ALG2,
 DG_VARIANT_PAPER_BOUND, DG_VARIANT_TPS) = range(8)

EXPORTS = ("dg_drag_matrix_build", "dg_expm_scale_square", "dg_drag_apply", "dg_drag_update", "dg_drag_update_ex",
           "dg_drag_update_variant", "dg_drag_update_steps", "dg_drag_rk1", "dg_drag_update_energy", "dg_drag_update_f32",
           "dg_drag_update_host", "dg_host_release", "dg_host_set_max_pitch", "dg_drag_update_host_static", "dg_peak_kernel", "dg_launches_per_update", "dg_variant_name",
           "dg_status_string", "dg_last_cuda_error", "dg_version")


class DgError(RuntimeError):
    def __init__(self, status, where):
        self.status = int(status)
        msg = _lib.dg_status_string(self.status).decode()
        if self.status == DG_ECUDA:
            msg += " — " + _lib.dg_last_cuda_error().decode()
        super().__init__(f"{where}: {msg}")


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2509_25347_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, dbl, ll, i32 = C.c_void_p, C.c_double, C.c_longlong, C.c_int
    lib.dg_drag_matrix_build.argtypes = [vp, vp, vp, dbl, i32, ll, vp, vp]
    lib.dg_expm_scale_square.argtypes = [vp, i32, ll, vp, vp, vp]
    lib.dg_drag_apply.argtypes = [vp, vp, i32, ll, vp, vp]
    lib.dg_drag_update.argtypes = [vp, vp, vp, dbl, vp, i32, ll, vp, vp]
    lib.dg_drag_update_ex.argtypes = [vp, vp, vp, dbl, vp, i32, ll, vp, vp, vp, vp]
    lib.dg_drag_update_variant.argtypes = [vp, vp, vp, dbl, vp, i32, ll, vp, vp, vp, i32, vp]
    lib.dg_drag_update_steps.argtypes = [vp, vp, vp, dbl, vp, i32, ll, i32, vp, vp]
    lib.dg_drag_rk1.argtypes = [vp, vp, vp, dbl, vp, i32, ll, vp, vp]
    lib.dg_drag_update_f32.argtypes = [vp, vp, vp, C.c_float, vp, i32, ll, vp, vp, vp, vp]
    lib.dg_drag_update_energy.argtypes = [vp, vp, vp, dbl, vp, vp, dbl, i32, ll, vp, vp, vp]
    lib.dg_drag_update_host.argtypes = [vp, vp, vp, dbl, vp, i32, ll, vp, ll, i32]
    lib.dg_host_release.argtypes = []
    lib.dg_host_set_max_pitch.argtypes = [ll]
    lib.dg_drag_update_host_static.argtypes = [vp, vp, vp, dbl, vp, i32, ll, vp, vp]
    lib.dg_peak_kernel.argtypes = [i32, i32, vp, ll, C.POINTER(dbl), vp]
    lib.dg_launches_per_update.argtypes = [i32, ll]
    lib.dg_variant_name.argtypes = [i32]
    lib.dg_variant_name.restype = C.c_char_p
    lib.dg_status_string.argtypes = [i32]
    lib.dg_status_string.restype = C.c_char_p
    lib.dg_last_cuda_error.argtypes = []
    lib.dg_last_cuda_error.restype = C.c_char_p
    lib.dg_version.argtypes = []
    for name in EXPORTS:
        fn = getattr(lib, name)
        if fn.restype is C.c_int and name not in ("dg_launches_per_update", "dg_version"):
            fn.restype = C.c_int
    return lib


_lib = _load()


def raw():
    """The ctypes library handle (tests call it with deliberately bad arguments)."""
    return _lib


def _check(st, where):
    if st != DG_OK:
        raise DgError(st, where)


def _dev(t, name, shape=None, dtype=torch.float64):
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name}: expected a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous {dtype} tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t.data_ptr()


def _stream():
    return torch.cuda.current_stream().cuda_stream


def dg_drag_matrix_build(rho_g, rho_d, t_s, dt, A=None):
    """Stage a1.  Returns A [n*n, ncells] = dt*Omega (Eq. 17)."""
    N, ncells = rho_d.shape
    n = N + 1
    if A is None:
        A = torch.empty((n * n, ncells), dtype=torch.float64, device=rho_g.device)
    st = _lib.dg_drag_matrix_build(_dev(rho_g, "rho_g", (ncells,)), _dev(rho_d, "rho_d", (N, ncells)),
                                   _dev(t_s, "t_s", (N, ncells)), float(dt), N, ncells,
                                   _dev(A, "A", (n * n, ncells)), _stream())
    _check(st, "dg_drag_matrix_build")
    return A


def dg_expm_scale_square(A, N, E=None, want_s=False):
    """Stages a2-a4.  Returns E [n*n, ncells] = exp(A) (and the per-cell scaling exponent s if want_s)."""
    n = N + 1
    ncells = A.shape[1]
    if E is None:
        E = torch.empty_like(A)
    s = torch.empty(ncells, dtype=torch.int32, device=A.device) if want_s else None
    st = _lib.dg_expm_scale_square(_dev(A, "A", (n * n, ncells)), N, ncells, _dev(E, "E", (n * n, ncells)),
                                   _dev(s, "s_out", (ncells,), torch.int32) if want_s else None, _stream())
    _check(st, "dg_expm_scale_square")
    return (E, s) if want_s else E


def dg_drag_apply(E, p_in, N, p_out=None):
    """Stage a5.  Returns p_out [3, n, ncells] = E p_in."""
    n = N + 1
    ncells = E.shape[1]
    if p_out is None:
        p_out = torch.empty_like(p_in)
    st = _lib.dg_drag_apply(_dev(E, "E", (n * n, ncells)), _dev(p_in, "p_in", (3, n, ncells)), N, ncells,
                            _dev(p_out, "p_out", (3, n, ncells)), _stream())
    _check(st, "dg_drag_apply")
    return p_out


def dg_drag_update(rho_g, rho_d, t_s, dt, p_in, p_out=None):
    """Fused a1..a5 (the timed path).  Returns p_out [3, n, ncells]."""
    N, ncells = rho_d.shape
    n = N + 1
    if p_out is None:
        p_out = torch.empty_like(p_in)
    st = _lib.dg_drag_update(_dev(rho_g, "rho_g", (ncells,)), _dev(rho_d, "rho_d", (N, ncells)),
                             _dev(t_s, "t_s", (N, ncells)), float(dt), _dev(p_in, "p_in", (3, n, ncells)), N, ncells,
                             _dev(p_out, "p_out", (3, n, ncells)), _stream())
    _check(st, "dg_drag_update")
    return p_out


def dg_drag_update_ex(rho_g, rho_d, t_s, dt, p_in, p_out=None, variant=DG_VARIANT_DEFAULT):
    """Fused update that also returns the per-cell (s, m) choices: (p_out, s int32[ncells], m int32[ncells]).
    `variant` forces the thread mapping (dg_drag_update_variant)."""
    N, ncells = rho_d.shape
    n = N + 1
    if p_out is None:
        p_out = torch.empty_like(p_in)
    s = torch.empty(ncells, dtype=torch.int32, device=rho_g.device)
    m = torch.empty(ncells, dtype=torch.int32, device=rho_g.device)
    st = _lib.dg_drag_update_variant(_dev(rho_g, "rho_g", (ncells,)), _dev(rho_d, "rho_d", (N, ncells)),
                                     _dev(t_s, "t_s", (N, ncells)), float(dt), _dev(p_in, "p_in", (3, n, ncells)), N,
                                     ncells, _dev(p_out, "p_out", (3, n, ncells)),
                                     _dev(s, "s", (ncells,), torch.int32), _dev(m, "m", (ncells,), torch.int32),
                                     int(variant), _stream())
    _check(st, "dg_drag_update_variant")
    return p_out, s, m


def dg_drag_update_steps(rho_g, rho_d, t_s, dt, p_in, nsteps, p_out=None):
    """nsteps fused drag updates in a row with the same dt (the Dustybox driver)."""
    N, ncells = rho_d.shape
    n = N + 1
    if p_out is None:
        p_out = torch.empty_like(p_in)
    st = _lib.dg_drag_update_steps(_dev(rho_g, "rho_g", (ncells,)), _dev(rho_d, "rho_d", (N, ncells)),
                                   _dev(t_s, "t_s", (N, ncells)), float(dt), _dev(p_in, "p_in", (3, n, ncells)), N,
                                   ncells, int(nsteps), _dev(p_out, "p_out", (3, n, ncells)), _stream())
    _check(st, "dg_drag_update_steps")
    return p_out


def dg_drag_rk1(rho_g, rho_d, t_s, dt, p_in, p_out=None):
    """First-order implicit RK1 drag step (App. A.2, Eq. A.8-A.9): p_out = (I - dt Omega)^-1 p_in."""
    N, ncells = rho_d.shape
    n = N + 1
    if p_out is None:
        p_out = torch.empty_like(p_in)
    st = _lib.dg_drag_rk1(_dev(rho_g, "rho_g", (ncells,)), _dev(rho_d, "rho_d", (N, ncells)),
                          _dev(t_s, "t_s", (N, ncells)), float(dt), _dev(p_in, "p_in", (3, n, ncells)), N, ncells,
                          _dev(p_out, "p_out", (3, n, ncells)), _stream())
    _check(st, "dg_drag_rk1")
    return p_out


def dg_drag_update_energy(rho_g, rho_d, t_s, dt, p_in, E_in, w, p_out=None, E_out=None):
    """Fused drag update plus the gas energy with frictional heating (Eq. 4; w in [0, 1]): returns (p_out, E_out)."""
    N, ncells = rho_d.shape
    n = N + 1
    if p_out is None:
        p_out = torch.empty_like(p_in)
    if E_out is None:
        E_out = torch.empty_like(E_in)
    st = _lib.dg_drag_update_energy(_dev(rho_g, "rho_g", (ncells,)), _dev(rho_d, "rho_d", (N, ncells)),
                                    _dev(t_s, "t_s", (N, ncells)), float(dt), _dev(p_in, "p_in", (3, n, ncells)),
                                    _dev(E_in, "E_in", (ncells,)), float(w), N, ncells,
                                    _dev(p_out, "p_out", (3, n, ncells)), _dev(E_out, "E_out", (ncells,)), _stream())
    _check(st, "dg_drag_update_energy")
    return p_out, E_out


def dg_drag_update_f32(rho_g, rho_d, t_s, dt, p_in, p_out=None):
    """The fused update in single precision (Eq. B.8 with u = 2^-24): float32 tensors in, (p_out, s, m) out."""
    N, ncells = rho_d.shape
    n = N + 1
    f32 = torch.float32
    if p_out is None:
        p_out = torch.empty_like(p_in)
    s = torch.empty(ncells, dtype=torch.int32, device=rho_g.device)
    m = torch.empty(ncells, dtype=torch.int32, device=rho_g.device)
    st = _lib.dg_drag_update_f32(_dev(rho_g, "rho_g", (ncells,), f32), _dev(rho_d, "rho_d", (N, ncells), f32),
                                 _dev(t_s, "t_s", (N, ncells), f32), float(dt), _dev(p_in, "p_in", (3, n, ncells), f32),
                                 N, ncells, _dev(p_out, "p_out", (3, n, ncells), f32),
                                 _dev(s, "s", (ncells,), torch.int32), _dev(m, "m", (ncells,), torch.int32), _stream())
    _check(st, "dg_drag_update_f32")
    return p_out, s, m


def _host(t, name, shape):
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous float64 CPU tensor")
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t.data_ptr()


def dg_drag_update_host(rho_g, rho_d, t_s, dt, p_in, p_out=None, chunk_cells=0, device=-1):
    """The fused update on HOST tensors (pinned memory makes the copies asynchronous).  Synchronous."""
    N, ncells = rho_d.shape
    n = N + 1
    if p_out is None:
        p_out = torch.empty_like(p_in)
    st = _lib.dg_drag_update_host(_host(rho_g, "rho_g", (ncells,)), _host(rho_d, "rho_d", (N, ncells)),
                                  _host(t_s, "t_s", (N, ncells)), float(dt), _host(p_in, "p_in", (3, n, ncells)), N,
                                  ncells, _host(p_out, "p_out", (3, n, ncells)), int(chunk_cells), int(device))
    _check(st, "dg_drag_update_host")
    return p_out


def dg_host_release():
    _check(_lib.dg_host_release(), "dg_host_release")


def dg_host_set_max_pitch(nbytes):
    """Test hook: rows of dg_drag_update_host whose pitch exceeds `nbytes` are copied one by one (0 = device limit)."""
    _check(_lib.dg_host_set_max_pitch(int(nbytes)), "dg_host_set_max_pitch")


def dg_drag_update_host_static(rho_g, rho_d, t_s, dt, p_in, p_out=None):
    """The fused update on HOST tensors for callers that must not allocate device memory (a host code whose pool owns
    the whole GPU, a loop that cannot take cudaMalloc's device-wide stall, a fixed memory quota): the library call
    stages in a fixed 32 MiB array built into libdg.so instead of asking for memory.  At most
    DG_STATIC_STAGE_BYTES // (8 * (8N + 7)) cells per call, DgError(DG_ECAPACITY) beyond; runs on the current device and
    torch's current stream and returns when p_out is complete.  Calls share that one array: never let two overlap.
    (Only the C call is allocation-free; this wrapper still makes the host result tensor when p_out is None.)"""
    N, ncells = rho_d.shape
    n = N + 1
    if p_out is None:
        p_out = torch.empty_like(p_in)
    st = _lib.dg_drag_update_host_static(_host(rho_g, "rho_g", (ncells,)), _host(rho_d, "rho_d", (N, ncells)),
                                         _host(t_s, "t_s", (N, ncells)), float(dt), _host(p_in, "p_in", (3, n, ncells)),
                                         N, ncells, _host(p_out, "p_out", (3, n, ncells)), _stream())
    _check(st, "dg_drag_update_host_static")
    return p_out


def dg_peak_kernel(kind, iters, scratch):
    """Enqueues one microbenchmark launch on the current stream; returns the flops (kinds 0-2) or bytes (kind 3)."""
    work = C.c_double(0.0)
    st = _lib.dg_peak_kernel(int(kind), int(iters), _dev(scratch, "scratch"), scratch.numel() * 8, C.byref(work),
                             _stream())
    _check(st, "dg_peak_kernel")
    return work.value


def dg_launches_per_update(N, ncells):
    return int(_lib.dg_launches_per_update(int(N), int(ncells)))


def dg_variant_name(N):
    return _lib.dg_variant_name(int(N)).decode()


def dg_version():
    return int(_lib.dg_version())
