"""Kernel-level GPU checks of the tcgen05 GEMMs (csrc/gemm_tc.cu) against a dense FP64 product of the
same operands (torch on the GPU), through the test hooks of csrc/test_hooks.cu
(libmlmd_test.so: the product objects plus the hooks; the product library does not export them).  Shapes span several M / N
tiles, a ragged projector count, several split-K slices and accumulation chains.

What they pin: operand layouts (MN-major 32B-atom swizzle, K-major SW32), descriptor strides, the
hi/lo split, chain draining through TMA store / reduce-add, and the accuracy of each product mode.
"""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def L():
    import paper_2509_00966_b200 as M
    M.lib()
    lib = ctypes.CDLL(M.api.TEST_LIB_PATH)
    i, p, l = ctypes.c_int, ctypes.c_void_p, ctypes.c_long
    lib.mlmd_debug_proj.argtypes = [i, p, i, l, p, p, i, i, p, i, i, p, i, i, i, i]
    lib.mlmd_debug_back.argtypes = [i, p, i, l, p, p, i, i, p, p, p, i, i, i, i]
    return lib


def hi_lo(x):
    import torch
    h = (x.view(torch.int32) & -8192).view(torch.float32)
    return h, x - h


def run_proj(L, path, ndom, ngrid, P, N, nsplit, nprod, chain, positive=False, split_in_kernel=True):
    """split_in_kernel (the product path): A is ONE plain FP32 array, the kernel forms hi / lo in shared memory;
    False: a pre-split (hi, lo) pair is handed over (the kernel's second operand stream, kept for callers that have it)."""
    import torch
    g = torch.Generator(device="cuda").manual_seed(1234)
    lda = (P + 7) // 8 * 8
    A = torch.zeros(ndom * ngrid * lda + 64, device="cuda")          # + slack for the last 32-column chunk
    Av = A[: ndom * ngrid * lda].view(ndom, ngrid, lda)
    rnd = (lambda *s: torch.rand(*s, device="cuda", generator=g)) if positive else (lambda *s: torch.randn(*s, device="cuda", generator=g))
    Av[:, :, :P] = rnd(ndom, ngrid, P)
    Y = rnd(ndom, ngrid, N)
    Ah, Al = hi_lo(A)
    prows = (max(lda, N) + 127) // 128 * 128
    z = torch.full((ndom, nsplit, prows, N), 7.0, device="cuda")
    a_hi = A if split_in_kernel else Ah
    a_lo = None if (split_in_kernel or nprod != 3) else Al.data_ptr()
    rc = L.mlmd_debug_proj(path, None, ndom, ngrid, a_hi.data_ptr(), a_lo, lda, P, Y.data_ptr(), N, N, z.data_ptr(), prows,
                           nsplit, nprod, chain)
    assert rc == 0
    Z = z.sum(1)[:, :P, :].double()
    ref = torch.einsum("drp,drc->dpc", Av[:, :, :P].double(), Y.double())
    return float((Z - ref).abs().max() / ref.abs().max())


def run_back(L, path, ndom, ngrid, P, N, nprod, stored_remainder=True):
    """stored_remainder: hand the kernel A - trunc_tf32(A) as its second operand stream (the product path: CTA-pair
    kernel); False: the single-CTA kernel forms the operand pair in shared memory."""
    import torch
    g = torch.Generator(device="cuda").manual_seed(4321)
    lda = (P + 7) // 8 * 8
    A = torch.zeros(ndom, ngrid, lda, device="cuda")
    A[:, :, :P] = torch.randn(ndom, ngrid, P, device="cuda", generator=g)
    prows = (max(lda, N) + 127) // 128 * 128
    W = torch.zeros(ndom, prows, N, device="cuda")
    W[:, :P] = torch.randn(ndom, P, N, device="cuda", generator=g)
    Y0 = torch.randn(ndom, ngrid, N, device="cuda", generator=g)
    Y = Y0.clone()
    Wh, Wl = hi_lo(W)
    Al = hi_lo(A)[1]
    rc = L.mlmd_debug_back(path, None, ndom, ngrid, A.data_ptr(), Al.data_ptr() if stored_remainder else None, lda, P,
                           Wh.data_ptr(), Wl.data_ptr(), Y.data_ptr(), N, N, prows, nprod)
    assert rc == 0
    ref = Y0.double() + torch.einsum("drp,dpc->drc", A.double(), W[:, :lda].double())
    return float((Y.double() - ref).abs().max() / ref.abs().max())


SHAPES = [(1, 1024, 32, 128), (2, 4096, 240, 448), (1, 2048, 300, 704), (3, 512, 5, 32)]


@pytest.mark.parametrize("ndom,ngrid,P,N", SHAPES)
def test_projection_3xtf32(L, ndom, ngrid, P, N):
    for nsplit, chain in ((1, 0), (3, 8), (2, 2)):
        err = run_proj(L, 1, ndom, ngrid, P, N, nsplit, 3, chain)
        assert err < (4e-6 if chain else 1e-4), (nsplit, chain, err)   # unchained: ~2.3e-8 per MMA (R2)


def test_projection_chain_bounds_truncation_drift(L):
    """Reading R2 of DESIGN.md: tensor-core accumulation truncates; same-sign sums drift linearly with
    the chain length and the bounded chains remove the drift."""
    long_chain = run_proj(L, 1, 2, 8192, 240, 448, 1, 3, 0, positive=True)
    short_chain = run_proj(L, 1, 2, 8192, 240, 448, 1, 3, 4, positive=True)
    assert short_chain < 4e-6 and long_chain > 4 * short_chain


def test_projection_with_presplit_operand_pair(L):
    assert run_proj(L, 1, 2, 2048, 448, 448, 2, 3, 4, split_in_kernel=False) < 4e-6


@pytest.mark.parametrize("nprod,tol", [(1, 2e-3), (0, 1.5e-2)])
def test_projection_low_precision_rungs(L, nprod, tol):
    err = run_proj(L, 1, 2, 4096, 240, 448, 3, nprod, 8)
    assert 1e-5 < err < tol


@pytest.mark.parametrize("ndom,ngrid,P,N", SHAPES)
def test_back_application(L, ndom, ngrid, P, N):
    assert run_back(L, 1, ndom, ngrid, P, N, 3) < 6e-6
    assert run_back(L, 1, ndom, ngrid, P, N, 3, stored_remainder=False) < 6e-6
    assert run_back(L, 1, ndom, ngrid, P, N, 1) < 3e-3
    assert run_back(L, 1, ndom, ngrid, P, N, 0) < 2e-2


def test_cuda_core_kernels_agree(L):
    assert run_proj(L, 0, 2, 1024, 37, 96, 4, 3, 0) < 2e-6
    assert run_back(L, 0, 2, 1000, 37, 96, 3) < 2e-6
