"""numpy-facing wrapper around the FP64 C oracle (oracle/mlmd_ref.c).

TEST INFRASTRUCTURE ONLY: import this from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs, never from the product package.  It promotes the
float32/complex64 inputs produced by ``workloads`` to float64/complex128 (reading D21) and
calls the C functions; there is no arithmetic of the method in this file.
"""
from __future__ import annotations

import ctypes
from typing import Optional, Sequence, Tuple

import numpy as np

from . import build as _build

NO_KINETIC = 1
HORNER = 2
NO_LOCAL = 4
ORDER2 = 8      # 2nd-order (7-point) stencil: the paper's own local discretisation (NEXT-3)

_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        i, d, p, l = ctypes.c_int, ctypes.c_double, ctypes.c_void_p, ctypes.c_long
        _lib.mlmd_ref_num_threads.restype = i
        _lib.mlmd_ref_apply_h.argtypes = [i, i, i, d, d, d, i, i, p, p, p, p, p, p, i]
        _lib.mlmd_ref_apply_h.restype = i
        _lib.mlmd_ref_density.argtypes = [i, l, i, p, p, p]
        _lib.mlmd_ref_density.restype = i
        _lib.mlmd_ref_overlap.argtypes = [i, l, i, d, p, p, p]
        _lib.mlmd_ref_overlap.restype = i
        _lib.mlmd_ref_propagate.argtypes = [i, i, i, i, d, d, d, i, i, p, p, p, p, p, i, d, p, i, p, i]
        _lib.mlmd_ref_propagate.restype = i
        _lib.mlmd_ref_propagate_split.argtypes = [i, i, i, i, d, d, d, i, i, p, p, p, p, p, i, d, p, i, p, i]
        _lib.mlmd_ref_propagate_split.restype = i
        _lib.mlmd_ref_local_richardson.argtypes = [i, i, i, d, d, d, i, p, p, p, d]
        _lib.mlmd_ref_local_richardson.restype = i
        _lib.mlmd_ref_occupations.argtypes = [i, i, p, p, p, p]
        _lib.mlmd_ref_occupations.restype = i
        _lib.mlmd_ref_energy_nl.argtypes = [i, l, i, i, d, p, p, p, p, p]
        _lib.mlmd_ref_energy_nl.restype = i
        _lib.mlmd_ref_current.argtypes = [i, i, i, i, d, d, d, i, p, p, p, i, p, i]
        _lib.mlmd_ref_current.restype = i
        _lib.mlmd_ref_current_nl.argtypes = [i, l, i, i, d, p, p, p, p, p, p]
        _lib.mlmd_ref_current_nl.restype = i
    return _lib


def num_threads() -> int:
    return int(lib().mlmd_ref_num_threads())


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def apply_h(u, vloc, beta, D, A: Sequence[float], h: Sequence[float], flags: int = 0) -> np.ndarray:
    """H u for one domain.  u: [nx,ny,nz,norb]; vloc: [nx,ny,nz]; beta: [ngrid,nproj] or None."""
    u = _c128(u)
    nx, ny, nz, norb = u.shape
    vloc = _f64(vloc)
    nproj = 0 if beta is None else beta.shape[-1]
    b = _c128(beta.reshape(-1, nproj)) if nproj else None
    dd = _f64(D) if nproj else None
    Av = _f64(A)
    out = np.empty_like(u)
    rc = lib().mlmd_ref_apply_h(nx, ny, nz, h[0], h[1], h[2], norb, nproj, _ptr(u), _ptr(out), _ptr(vloc),
                                _ptr(b), _ptr(dd), _ptr(Av), flags)
    if rc:
        raise RuntimeError("mlmd_ref_apply_h failed: %d" % rc)
    return out


def propagate(psi, occ, vloc, beta, D, A, dt: float, h: Sequence[float], nsteps: Optional[int] = None,
              flags: int = 0) -> Tuple[np.ndarray, np.ndarray]:
    """nsteps Taylor-4 steps.  psi: [ndom,nx,ny,nz,norb]; A: [nsteps, a_ndom, 3].
    Returns (psi_new complex128, rho float64 [ndom,nx,ny,nz])."""
    p = _c128(psi).copy()
    ndom, nx, ny, nz, norb = p.shape
    vloc = _f64(vloc)
    occ = _f64(occ)
    nproj = 0 if beta is None else beta.shape[-1]
    b = _c128(beta.reshape(ndom, -1, nproj)) if nproj else None
    dd = _f64(D) if nproj else None
    A = _f64(A)
    if nsteps is None:
        nsteps = A.shape[0]
    assert A.ndim == 3 and A.shape[0] >= nsteps and A.shape[1] in (1, ndom) and A.shape[2] == 3
    rho = np.empty((ndom, nx, ny, nz), dtype=np.float64)
    rc = lib().mlmd_ref_propagate(ndom, nx, ny, nz, h[0], h[1], h[2], norb, nproj, _ptr(p), _ptr(occ),
                                  _ptr(vloc), _ptr(b), _ptr(dd), nsteps, dt, _ptr(A), A.shape[1], _ptr(rho), flags)
    if rc:
        raise RuntimeError("mlmd_ref_propagate failed: %d" % rc)
    return p, rho


def propagate_split(psi, occ, vloc, beta, D, A, dt: float, h: Sequence[float], nsteps: Optional[int] = None,
                    kick_only: bool = False, local: str = "taylor", order: int = 4) -> Tuple[np.ndarray, np.ndarray]:
    """nsteps steps of the paper's literal Eq. (2): half-kick, exp(-i dt h_loc), half-kick.  local = "taylor": the
    4th-order Taylor sum on 4th-order differences (reading D28); "richardson": the paper's own block-diagonal
    split-operator solver on 2nd-order differences (reading D33).  order = 2: the Taylor sum on the 2nd-order (7-point)
    differences of reading D32.  Same arguments and return values as ``propagate``."""
    assert local in ("taylor", "richardson") and order in (2, 4)
    p = _c128(psi).copy()
    ndom, nx, ny, nz, norb = p.shape
    vloc = _f64(vloc)
    occ = _f64(occ)
    nproj = 0 if beta is None else beta.shape[-1]
    b = _c128(beta.reshape(ndom, -1, nproj)) if nproj else None
    dd = _f64(D) if nproj else None
    A = _f64(A)
    if nsteps is None:
        nsteps = A.shape[0]
    assert A.ndim == 3 and A.shape[0] >= nsteps and A.shape[1] in (1, ndom) and A.shape[2] == 3
    rho = np.empty((ndom, nx, ny, nz), dtype=np.float64)
    rc = lib().mlmd_ref_propagate_split(ndom, nx, ny, nz, h[0], h[1], h[2], norb, nproj, _ptr(p), _ptr(occ),
                                        _ptr(vloc), _ptr(b), _ptr(dd), nsteps, dt, _ptr(A), A.shape[1], _ptr(rho),
                                        (1 if kick_only else 0) | (2 if local == "richardson" else 0) | (4 if order == 2 else 0))
    if rc:
        raise RuntimeError("mlmd_ref_propagate_split failed: %d" % rc)
    return p, rho


def local_richardson(psi, vloc, A, dt: float, h: Sequence[float]) -> np.ndarray:
    """One application of U_loc(dt) of reading D33 to psi [nx, ny, nz, norb] (one domain); A: [3]."""
    p = _c128(psi).copy()
    nx, ny, nz, norb = p.shape
    v, a = _f64(vloc), _f64(A)
    rc = lib().mlmd_ref_local_richardson(nx, ny, nz, h[0], h[1], h[2], norb, _ptr(p), _ptr(v), _ptr(a), dt)
    if rc:
        raise RuntimeError("mlmd_ref_local_richardson failed: %d" % rc)
    return p


def density(psi, occ) -> np.ndarray:
    p = _c128(psi)
    ndom, nx, ny, nz, norb = p.shape
    occ = _f64(occ)
    rho = np.empty((ndom, nx, ny, nz), dtype=np.float64)
    lib().mlmd_ref_density(ndom, nx * ny * nz, norb, _ptr(p), _ptr(occ), _ptr(rho))
    return rho


def overlap(phi, psi, dv: float) -> np.ndarray:
    """S[dom] = dv * phi^H psi, [ndom, norb, norb] complex128."""
    a, b = _c128(phi), _c128(psi)
    ndom, nx, ny, nz, norb = b.shape
    S = np.empty((ndom, norb, norb), dtype=np.complex128)
    lib().mlmd_ref_overlap(ndom, nx * ny * nz, norb, dv, _ptr(a), _ptr(b), _ptr(S))
    return S


def occupations(S, occ) -> Tuple[np.ndarray, np.ndarray]:
    """(f_s(t) [ndom, norb], n_exc [ndom]) from S = overlap(Psi(0), Psi(t)) and the occupations (reading D29)."""
    S = _c128(S)
    occ = _f64(occ)
    ndom, norb, _ = S.shape
    f = np.empty((ndom, norb), dtype=np.float64)
    nexc = np.empty((ndom,), dtype=np.float64)
    lib().mlmd_ref_occupations(ndom, norb, _ptr(S), _ptr(occ), _ptr(f), _ptr(nexc))
    return f, nexc


def energy_nl(psi, occ, beta, D, dv: float) -> np.ndarray:
    """E_nl[dom] = sum_n f_n <psi_n|V_NL|psi_n>."""
    p = _c128(psi)
    ndom, nx, ny, nz, norb = p.shape
    nproj = beta.shape[-1]
    b = _c128(beta.reshape(ndom, -1, nproj))
    E = np.empty((ndom,), dtype=np.float64)
    lib().mlmd_ref_energy_nl(ndom, nx * ny * nz, norb, nproj, dv, _ptr(p), _ptr(_f64(occ)), _ptr(b), _ptr(_f64(D)), _ptr(E))
    return E


def current(psi, occ, A, h: Sequence[float], flags: int = 0) -> np.ndarray:
    """J[dom][d] = sum_n f_n Re<psi_n| -i D1_d + A_d |psi_n>; A: [a_ndom, 3]; flags=ORDER2: the 2nd-order D1."""
    p = _c128(psi)
    ndom, nx, ny, nz, norb = p.shape
    A = _f64(A).reshape(-1, 3)
    assert A.shape[0] in (1, ndom)
    J = np.empty((ndom, 3), dtype=np.float64)
    lib().mlmd_ref_current(ndom, nx, ny, nz, h[0], h[1], h[2], norb, _ptr(p), _ptr(_f64(occ)), _ptr(A), A.shape[0], _ptr(J), flags)
    return J


def current_nl(psi, occ, beta, rbeta, D, dv: float) -> np.ndarray:
    """Nonlocal part of the current: J[dom][d] = sum_n f_n <psi_n| -i [r_d, V_NL] |psi_n>.
    rbeta: [3, ndom, ngrid, nproj] = (r - R_p)_d beta_p(r), supplied by the caller."""
    p = _c128(psi)
    ndom, nx, ny, nz, norb = p.shape
    nproj = beta.shape[-1]
    b = _c128(beta.reshape(ndom, -1, nproj))
    rb = _c128(rbeta.reshape(3, ndom, -1, nproj))
    J = np.empty((ndom, 3), dtype=np.float64)
    rc = lib().mlmd_ref_current_nl(ndom, nx * ny * nz, norb, nproj, dv, _ptr(p), _ptr(_f64(occ)), _ptr(b), _ptr(rb),
                                   _ptr(_f64(D)), _ptr(J))
    if rc:
        raise RuntimeError("mlmd_ref_current_nl failed: %d" % rc)
    return J
