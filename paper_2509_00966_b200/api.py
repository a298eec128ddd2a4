"""ctypes binding of include/mlmd.h: same names, argument marshalling only.

Arrays may be numpy arrays (host) or torch CUDA tensors (device); the binding passes their
pointers and the matching MLMD_HOST / MLMD_DEVICE tag.  ``Domain`` is a small convenience owner
of the handle and its torch-allocated workspace.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmlmd.so")
TEST_LIB_PATH = os.path.join(HERE, "libmlmd_test.so")   # product objects + kernel-level test hooks; tests/ only

OK, ERR_ARG, ERR_SHAPE, ERR_STATE, ERR_CUDA, ERR_NOMEM, ERR_NONFINITE, WARN_UNSTABLE = range(8)
HOST, DEVICE = 0, 1
BETA_REAL32, BETA_COMPLEX64 = 0, 1
GEMM_FP32GRADE, GEMM_FP64, GEMM_LOWP_BF16, GEMM_TF32X1, GEMM_FP32_SIMT, GEMM_FP32GRADE_STAGED = range(6)
KEEP_PSI0, CHECK_FINITE, BORROW_PSI = 1, 2, 4
OPT_GRAPH, OPT_STENCIL, OPT_GEMM_PATH, OPT_KICK_NORM, OPT_FD_ORDER, OPT_LOCAL_SOLVER = range(6)

EXPORTED_SYMBOLS = [
    "mlmd_workspace_bytes", "mlmd_domain_create", "mlmd_domain_destroy", "mlmd_set_orbitals",
    "mlmd_get_orbitals", "mlmd_set_vloc", "mlmd_set_projectors", "mlmd_set_gemm_mode", "mlmd_set_option", "mlmd_propagate",
    "mlmd_propagate_split", "mlmd_occupations", "mlmd_energy_nl", "mlmd_current", "mlmd_current_nl",
    "mlmd_density", "mlmd_overlap", "mlmd_orbital_norms_static", "mlmd_launch_count", "mlmd_last_error", "mlmd_profile", "mlmd_profile_read", "mlmd_gemm_path",
]
K_STENCIL, K_PROJ, K_BACK, K_GLUE, K_DENSITY, K_NLP, K_NORM = range(7)
KERNEL_CLASSES = ["stencil", "proj", "back", "glue", "density", "nlp", "norm"]


class MlmdError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("mlmd error %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib() -> ctypes.CDLL:
    """Load libmlmd.so (built in-tree by paper_2509_00966_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise MlmdError(ERR_CUDA, "%s not found: run `python -c 'import __graft_entry__ as g; g.build()'` "
                            "(there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        i, d, p, u, z = ctypes.c_int, ctypes.c_double, ctypes.c_void_p, ctypes.c_uint, ctypes.c_size_t
        L.mlmd_workspace_bytes.argtypes = [i, i, i, i, i, i, u]
        L.mlmd_workspace_bytes.restype = z
        L.mlmd_domain_create.argtypes = [ctypes.POINTER(p), i, i, i, i, d, d, d, i, i, p, z, p, u]
        L.mlmd_domain_destroy.argtypes = [p]
        L.mlmd_set_orbitals.argtypes = [p, p, p, i]
        L.mlmd_get_orbitals.argtypes = [p, p, i]
        L.mlmd_set_vloc.argtypes = [p, p, i]
        L.mlmd_set_projectors.argtypes = [p, i, p, i, p, i]
        L.mlmd_set_gemm_mode.argtypes = [p, i]
        L.mlmd_set_option.argtypes = [p, i, i]
        L.mlmd_propagate.argtypes = [p, i, d, p, i]
        L.mlmd_propagate_split.argtypes = [p, i, d, p, i]
        L.mlmd_density.argtypes = [p, p, i]
        L.mlmd_overlap.argtypes = [p, i, p, i]
        L.mlmd_orbital_norms_static.argtypes = [p, i, ctypes.c_longlong, i, d, p, p]
        L.mlmd_occupations.argtypes = [p, p, p, i]
        L.mlmd_energy_nl.argtypes = [p, p, i]
        L.mlmd_current.argtypes = [p, p, i, p, i]
        L.mlmd_current_nl.argtypes = [p, p, i, p, i]
        L.mlmd_profile.argtypes = [p, i]
        L.mlmd_profile_read.argtypes = [p, i, ctypes.POINTER(d), ctypes.POINTER(ctypes.c_longlong)]
        L.mlmd_launch_count.argtypes = [p]
        L.mlmd_gemm_path.argtypes = [p]
        L.mlmd_launch_count.restype = ctypes.c_longlong
        L.mlmd_last_error.restype = ctypes.c_char_p
        for name in EXPORTED_SYMBOLS:
            if name not in ("mlmd_workspace_bytes", "mlmd_launch_count", "mlmd_last_error", "mlmd_profile_read"):
                getattr(L, name).restype = i
        _lib = L
    return _lib


def mlmd_last_error() -> str:
    return lib().mlmd_last_error().decode()


def _check(rc: int) -> int:
    if rc not in (OK, WARN_UNSTABLE):
        raise MlmdError(rc, mlmd_last_error())
    return rc


def _ptr_where(a, dtype=None):
    """(pointer, where) of a numpy array or a torch tensor; checks contiguity and dtype."""
    if a is None:
        return None, HOST
    if isinstance(a, np.ndarray):
        if dtype is not None and a.dtype != dtype:
            raise TypeError("expected dtype %s, got %s" % (dtype, a.dtype))
        if not a.flags.c_contiguous:
            raise ValueError("array must be C-contiguous")
        return ctypes.c_void_p(a.ctypes.data), HOST
    import torch
    if isinstance(a, torch.Tensor):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        if dtype is not None and np.dtype(str(a.dtype).replace("torch.", "")) != dtype:
            raise TypeError("expected dtype %s, got %s" % (dtype, a.dtype))
        return ctypes.c_void_p(a.data_ptr()), (DEVICE if a.is_cuda else HOST)
    raise TypeError("expected numpy array or torch tensor, got %r" % type(a))


def _host_f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


# ---- the C calls, same names ---------------------------------------------------------------------
def mlmd_workspace_bytes(ndom, nx, ny, nz, norb, nproj_max, flags=0) -> int:
    return int(lib().mlmd_workspace_bytes(ndom, nx, ny, nz, norb, nproj_max, flags))


def mlmd_domain_create(ndom, nx, ny, nz, hx, hy, hz, norb, nproj_max, workspace_ptr, workspace_bytes,
                       stream_ptr=0, flags=0):
    h = ctypes.c_void_p()
    _check(lib().mlmd_domain_create(ctypes.byref(h), ndom, nx, ny, nz, hx, hy, hz, norb, nproj_max,
                                    ctypes.c_void_p(workspace_ptr), workspace_bytes, ctypes.c_void_p(stream_ptr), flags))
    return h


def mlmd_domain_destroy(h):
    _check(lib().mlmd_domain_destroy(h))


def mlmd_set_orbitals(h, psi, occ=None):
    p, where = _ptr_where(psi, np.dtype(np.complex64))
    o = _host_f64(occ)
    _check(lib().mlmd_set_orbitals(h, p, None if o is None else o.ctypes.data_as(ctypes.c_void_p), where))


def mlmd_get_orbitals(h, out):
    p, where = _ptr_where(out, np.dtype(np.complex64))
    _check(lib().mlmd_get_orbitals(h, p, where))
    return out


def mlmd_set_vloc(h, vloc):
    p, where = _ptr_where(vloc, np.dtype(np.float32))
    _check(lib().mlmd_set_vloc(h, p, where))


def mlmd_set_projectors(h, nproj, beta, D):
    if nproj == 0:
        _check(lib().mlmd_set_projectors(h, 0, None, BETA_REAL32, None, HOST))
        return
    if isinstance(beta, np.ndarray):
        cplx = beta.dtype == np.complex64
    else:
        cplx = "complex" in str(beta.dtype)
    p, where = _ptr_where(beta, np.dtype(np.complex64 if cplx else np.float32))
    d = _host_f64(D)
    _check(lib().mlmd_set_projectors(h, nproj, p, BETA_COMPLEX64 if cplx else BETA_REAL32,
                                     d.ctypes.data_as(ctypes.c_void_p), where))


def mlmd_set_gemm_mode(h, mode):
    _check(lib().mlmd_set_gemm_mode(h, mode))


def mlmd_set_option(h, key, value):
    _check(lib().mlmd_set_option(h, key, value))


def mlmd_propagate(h, nsteps, dt, A) -> int:
    """A: [nsteps, a_ndom, 3] float64 host array (a_ndom = 1 or ndom).  Returns OK or WARN_UNSTABLE."""
    a = _host_f64(A)
    if nsteps > 0 and (a.ndim != 3 or a.shape[0] < nsteps or a.shape[2] != 3):
        raise ValueError("A must have shape [nsteps, a_ndom, 3]")
    a_ndom = a.shape[1] if a is not None and a.ndim == 3 else 1
    return _check(lib().mlmd_propagate(h, nsteps, dt, None if a is None else a.ctypes.data_as(ctypes.c_void_p), a_ndom))


def mlmd_propagate_split(h, nsteps, dt, A) -> int:
    """The paper's literal Eq. (2) step (half-kick, Taylor-4 of h_loc, half-kick); arguments as mlmd_propagate."""
    a = _host_f64(A)
    if nsteps > 0 and (a.ndim != 3 or a.shape[0] < nsteps or a.shape[2] != 3):
        raise ValueError("A must have shape [nsteps, a_ndom, 3]")
    a_ndom = a.shape[1] if a is not None and a.ndim == 3 else 1
    return _check(lib().mlmd_propagate_split(h, nsteps, dt, None if a is None else a.ctypes.data_as(ctypes.c_void_p), a_ndom))


def mlmd_density(h, out):
    p, where = _ptr_where(out, np.dtype(np.float32))
    _check(lib().mlmd_density(h, p, where))
    return out


def mlmd_overlap(h, which, out):
    p, where = _ptr_where(out, np.dtype(np.complex64))
    _check(lib().mlmd_overlap(h, which, p, where))
    return out


def mlmd_orbital_norms_static(psi, dv, out, stream_ptr=0):
    """norm2[dom][n] = dv sum_r |psi[dom][r][n]|^2 with no handle, workspace or allocation (include/mlmd.h).
    psi: CUDA tensor complex64 [ndom, ngrid, ld]; out: CUDA tensor float64 [ndom, ld] (the caller's); returns out."""
    if psi.dim() != 3 or tuple(out.shape) != (psi.shape[0], psi.shape[2]):
        raise ValueError("psi must be [ndom, ngrid, ld] and out [ndom, ld]")
    pp, wp = _ptr_where(psi, np.dtype(np.complex64))
    po, wo = _ptr_where(out, np.dtype(np.float64))
    if wp != DEVICE or wo != DEVICE:
        raise ValueError("psi and out must be CUDA tensors")
    _check(lib().mlmd_orbital_norms_static(pp, psi.shape[0], psi.shape[1], psi.shape[2], float(dv), po, ctypes.c_void_p(stream_ptr)))
    return out


def mlmd_occupations(h, f, n_exc):
    """f: [ndom, norb] float64, n_exc: [ndom] float64 (numpy host arrays or CUDA tensors, both of one kind)."""
    pf, wf = _ptr_where(f, np.dtype(np.float64))
    pn, wn = _ptr_where(n_exc, np.dtype(np.float64))
    if wf != wn:
        raise ValueError("f and n_exc must both be host arrays or both be device tensors")
    _check(lib().mlmd_occupations(h, pf, pn, wf))
    return f, n_exc


def mlmd_energy_nl(h, E):
    """E: [ndom] float64 (numpy host array or CUDA tensor)."""
    p, where = _ptr_where(E, np.dtype(np.float64))
    _check(lib().mlmd_energy_nl(h, p, where))
    return E


def mlmd_current(h, A, J):
    """A: [a_ndom, 3] host float64; J: [ndom, 3] float64 (numpy host array or CUDA tensor)."""
    a = _host_f64(A).reshape(-1, 3)
    p, where = _ptr_where(J, np.dtype(np.float64))
    _check(lib().mlmd_current(h, a.ctypes.data_as(ctypes.c_void_p), a.shape[0], p, where))
    return J


def mlmd_current_nl(h, rbeta, J):
    """rbeta: [3, ndom, ngrid, nproj] = (r - R_p)_d beta_p(r), dtype of the projectors (numpy host array or CUDA tensor);
    J: [ndom, 3] float64 (numpy host array or CUDA tensor)."""
    pr, wr = _ptr_where(rbeta)
    p, where = _ptr_where(J, np.dtype(np.float64))
    _check(lib().mlmd_current_nl(h, pr, wr, p, where))
    return J


def mlmd_profile(h, enable: bool):
    _check(lib().mlmd_profile(h, 1 if enable else 0))


def mlmd_profile_read(h, kind: int):
    """(milliseconds summed over launches, number of launches) of kernel class `kind`."""
    ms, n = ctypes.c_double(), ctypes.c_longlong()
    _check(lib().mlmd_profile_read(h, kind, ctypes.byref(ms), ctypes.byref(n)))
    return ms.value, n.value


def mlmd_launch_count(h) -> int:
    return int(lib().mlmd_launch_count(h))


# ---- convenience owner ------------------------------------------------------------------------------
class Domain:
    """Owns a handle and its workspace (a torch uint8 CUDA tensor).  Methods mirror the C calls."""

    def __init__(self, ndom, grid, h, norb, nproj_max, flags=0, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise MlmdError(ERR_CUDA, "no CUDA device: libmlmd has no CPU fallback")
        self.ndom, self.grid, self.h, self.norb, self.nproj_max = ndom, tuple(grid), tuple(h), norb, nproj_max
        self.device = torch.device(device)
        nbytes = mlmd_workspace_bytes(ndom, *self.grid, norb, nproj_max, flags)
        if nbytes == 0:
            raise MlmdError(ERR_SHAPE, "invalid shape")
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            st = torch.cuda.current_stream(self.device) if stream is None else stream
            self.stream = st
            self.handle = mlmd_domain_create(ndom, *self.grid, *self.h, norb, nproj_max, self.workspace.data_ptr(),
                                             nbytes, st.cuda_stream, flags)

    def close(self):
        if getattr(self, "handle", None) is not None:
            mlmd_domain_destroy(self.handle)
            self.handle = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_orbitals(self, psi, occ=None):
        mlmd_set_orbitals(self.handle, psi, occ)

    def get_orbitals(self, out=None):
        if out is None:
            out = np.empty((self.ndom, *self.grid, self.norb), dtype=np.complex64)
        return mlmd_get_orbitals(self.handle, out)

    def set_vloc(self, vloc):
        mlmd_set_vloc(self.handle, vloc)

    def set_projectors(self, beta, D):
        nproj = 0 if beta is None else beta.shape[-1]
        mlmd_set_projectors(self.handle, nproj, beta, D)

    def set_gemm_mode(self, mode):
        mlmd_set_gemm_mode(self.handle, mode)

    def set_option(self, key, value):
        mlmd_set_option(self.handle, key, value)

    def propagate(self, nsteps, dt, A):
        return mlmd_propagate(self.handle, nsteps, dt, A)

    def propagate_split(self, nsteps, dt, A):
        return mlmd_propagate_split(self.handle, nsteps, dt, A)

    def density(self, out=None):
        if out is None:
            out = np.empty((self.ndom, *self.grid), dtype=np.float32)
        return mlmd_density(self.handle, out)

    def overlap(self, which=0, out=None):
        if out is None:
            out = np.empty((self.ndom, self.norb, self.norb), dtype=np.complex64)
        return mlmd_overlap(self.handle, which, out)

    def occupations(self):
        """(f_s(t) [ndom, norb], n_exc [ndom]) as float64 host arrays (needs flags=KEEP_PSI0)."""
        f = np.empty((self.ndom, self.norb), dtype=np.float64)
        n_exc = np.empty((self.ndom,), dtype=np.float64)
        return mlmd_occupations(self.handle, f, n_exc)

    def energy_nl(self):
        return mlmd_energy_nl(self.handle, np.empty((self.ndom,), dtype=np.float64))

    def current(self, A):
        return mlmd_current(self.handle, A, np.empty((self.ndom, 3), dtype=np.float64))

    def current_nl(self, rbeta):
        return mlmd_current_nl(self.handle, rbeta, np.empty((self.ndom, 3), dtype=np.float64))

    def profile(self, enable=True):
        mlmd_profile(self.handle, enable)

    def profile_read(self):
        """{class name: (ms_total, launches)} for the classes that ran."""
        out = {}
        for k, name in enumerate(KERNEL_CLASSES):
            ms, n = mlmd_profile_read(self.handle, k)
            if n:
                out[name] = (ms, n)
        return out

    def gemm_path(self):
        return "tcgen05" if lib().mlmd_gemm_path(self.handle) else "simt"

    def launch_count(self):
        return mlmd_launch_count(self.handle)
