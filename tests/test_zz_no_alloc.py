"""mlmd_orbital_norms_static: the allocation-free entry point (include/mlmd.h; scratch in a file-scope device array,
csrc/noalloc.cu) against the existing paths on the same data, on two calls in a row:
  * the split step's norm pass as the library runs it, with its partial sums in caller scratch (test hook
    mlmd_debug_colnorm2 of libmlmd_test.so): same summation order, so agreement to FP64 rounding;
  * the diagonal of mlmd_overlap's Gram matrix (through a handle), at the Gram tolerance of the parity tests (1e-5);
  * a plain FP64 sum.
The second call uses a smaller batch with other values, so anything stale in the shared array would show.
Collected last on purpose (pytest -x): a failure here hides nothing.
"""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hook():
    import paper_2509_00966_b200 as M
    M.lib()
    lib = ctypes.CDLL(M.api.TEST_LIB_PATH)
    i, p, l = ctypes.c_int, ctypes.c_void_p, ctypes.c_long
    lib.mlmd_debug_colnorm2.argtypes = [p, i, l, i, p, p, p]
    return lib


def _case(seed, ndom, grid, norb):
    import torch
    ld = (norb + 15) // 16 * 16
    ngrid = grid[0] * grid[1] * grid[2]
    g = torch.Generator(device="cuda").manual_seed(seed)
    psi = torch.zeros(ndom, ngrid, ld, dtype=torch.complex64, device="cuda")
    re = torch.randn(ndom, ngrid, norb, device="cuda", generator=g)
    im = torch.randn(ndom, ngrid, norb, device="cuda", generator=g)
    scale = 0.25 + torch.rand(ndom, 1, norb, device="cuda", generator=g)      # orbitals of different norms
    psi[:, :, :norb] = torch.complex(re, im) * scale
    return psi, ld, ngrid


def _existing_paths(M, hook, psi, grid, h, norb, dv):
    import torch
    ndom, ngrid, ld = psi.shape
    part = torch.empty(ndom, 64, ld, dtype=torch.float64, device="cuda")
    raw = torch.empty(ndom, ld, dtype=torch.float64, device="cuda")
    assert hook.mlmd_debug_colnorm2(None, ndom, ngrid, ld, psi.data_ptr(), part.data_ptr(), raw.data_ptr()) == 0
    dom = M.Domain(ndom, grid, h, norb, 0)
    dom.set_vloc(np.zeros((ndom, ngrid), np.float32))
    dom.set_orbitals(psi[:, :, :norb].reshape(ndom, *grid, norb).contiguous())
    gram = dom.overlap(0)
    gram = gram.cpu().numpy() if hasattr(gram, "cpu") else np.asarray(gram)
    dom.close() if hasattr(dom, "close") else None
    return raw * dv, np.real(np.diagonal(gram, axis1=1, axis2=2))


def test_static_scratch_entry_point_matches_the_existing_paths_twice_in_a_row(hook):
    import torch
    import paper_2509_00966_b200 as M
    h = (0.4, 0.45, 0.5)
    dv = h[0] * h[1] * h[2]
    cases = [(11, 3, (16, 16, 16), 40), (12, 2, (12, 10, 14), 24)]     # second: smaller batch, ragged slabs
    data = [_case(*c) for c in cases]
    outs = [torch.full((c[1], d[1]), -1.0, dtype=torch.float64, device="cuda") for c, d in zip(cases, data)]
    # warm-up (module load), then two calls in a row with no allocation between them
    M.mlmd_orbital_norms_static(data[0][0], dv, outs[0])
    torch.cuda.synchronize()
    outs[0].fill_(-1.0)
    free0 = torch.cuda.mem_get_info()[0]
    for (psi, ld, ngrid), out in zip(data, outs):
        M.mlmd_orbital_norms_static(psi, dv, out, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0, "the entry point must not allocate device memory"
    for (seed, ndom, grid, norb), (psi, ld, ngrid), out in zip(cases, data, outs):
        same_order, gram_diag = _existing_paths(M, hook, psi, grid, h, norb, dv)
        got = out.cpu().numpy()
        assert np.all(got[:, norb:] == 0.0)                                   # padded columns hold zeros
        np.testing.assert_allclose(got, same_order.cpu().numpy(), rtol=1e-14, atol=0.0)
        plain = ((psi.real.double() ** 2 + psi.imag.double() ** 2).sum(1) * dv).cpu().numpy()
        np.testing.assert_allclose(got, plain, rtol=1e-6)
        assert np.max(np.abs(got[:, :norb] - gram_diag) / np.abs(gram_diag)) <= 1e-5


def test_static_scratch_limit_and_argument_errors():
    import torch
    import paper_2509_00966_b200 as M
    L = M.lib()
    small = torch.zeros(1, 8, 16, dtype=torch.complex64, device="cuda")
    out = torch.zeros(1, 16, dtype=torch.float64, device="cuda")
    # 80 domains x 224 columns x 64 slabs x 8 B = 9.2 MB > the 8 MiB array: rejected before anything is launched
    rc = L.mlmd_orbital_norms_static(ctypes.c_void_p(small.data_ptr()), 80, 110592, 224, 1.0, ctypes.c_void_p(out.data_ptr()), None)
    assert rc == M.api.ERR_SHAPE and "MLMD_STATIC_SCRATCH_BYTES" in M.mlmd_last_error()
    host = np.zeros((1, 8, 16), np.complex64)
    rc = L.mlmd_orbital_norms_static(ctypes.c_void_p(host.ctypes.data), 1, 8, 16, 1.0, ctypes.c_void_p(out.data_ptr()), None)
    assert rc == M.api.ERR_ARG
    assert L.mlmd_orbital_norms_static(None, 1, 8, 16, 1.0, ctypes.c_void_p(out.data_ptr()), None) == M.api.ERR_ARG
    # the largest benchmarked batch shape (configs[3]: 64 domains x 224 orbitals) fits
    assert 64 * 64 * 224 * 8 <= 8 << 20
    torch.cuda.synchronize()
    assert float(out.abs().sum()) == 0.0
