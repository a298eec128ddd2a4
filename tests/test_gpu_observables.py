"""GPU parity of mlmd_energy_nl and mlmd_current (reading D30) against the FP64 oracle on
the same seeded inputs, through the C ABI.

Tolerances (derived from north_star's): E_nl is a sum of |projection coefficient|^2 with the GEMM's FP32-grade
error (Gram tolerance 1e-5), so relative 1e-5 of sum_n f_n sum_p |D_p| |<beta_p|psi_n>|^2 (the same sum without
cancellation between projectors of opposite sign); the current is an FP32 dot product per point summed in FP64:
1e-5 of N_e / h_min (its natural scale: every electron at the largest finite-difference velocity).
"""
import numpy as np
import pytest

import workloads as W
from test_gpu_parity import make_domain

pytestmark = pytest.mark.gpu


def check_observables(dom, psi, occ, beta, D, A, h, lowp=False):
    from oracle import ref
    dv = float(np.prod(h))
    tol = 1e-3 if lowp else 1e-5
    if beta is not None:
        E = dom.energy_nl()
        E_ref = ref.energy_nl(psi, occ, beta, D, dv)
        scale = ref.energy_nl(psi, occ, beta, np.abs(D), dv)
        print("E_nl", E, E_ref, "rel", np.abs(E - E_ref) / scale)
        assert (np.abs(E - E_ref) <= tol * scale).all()
    J = dom.current(A)
    J_ref = ref.current(psi, occ, A, h)
    ne = (np.asarray(occ) * dv * (np.abs(psi.astype(np.complex128)) ** 2).sum(axis=(1, 2, 3))).sum(axis=1)
    print("J", J, J_ref, "scaled err", np.abs(J - J_ref).max(axis=1) / (ne / min(h)))
    assert (np.abs(J - J_ref).max(axis=1) <= 1e-5 * ne / min(h)).all()


def test_observables_config1_after_the_pulse_starts():
    """Config 1 (one 32^3 domain, 64 orbitals, 32 projectors) after 5 steps in the field: GPU observables of the
    GPU state against oracle observables of the oracle state."""
    from oracle import ref
    c = W.get_config(1)
    d = W.generate(c)
    A = d["A"][:5] * 10.0
    dom = make_domain(c, d)
    dom.propagate(5, c.dt, A)
    r, _ = ref.propagate(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], A, c.dt, c.h)
    check_observables(dom, r, d["occ"], d["beta"], d["D"], A[4], c.h)
    dom.close()


@pytest.mark.parametrize("grid,norb,cplx", [((6, 5, 7), 3, True), ((8, 16, 8), 5, False), ((16, 16, 32), 12, True)])
def test_observables_ragged_shapes_complex_projectors_per_domain_field(grid, norb, cplx):
    import paper_2509_00966_b200 as M
    rng = np.random.default_rng(11 + norb)
    ndom, nproj, h = 3, 4, (0.5, 0.45, 0.4)
    ngrid = int(np.prod(grid))
    psi = (rng.standard_normal((ndom, *grid, norb)) + 1j * rng.standard_normal((ndom, *grid, norb))).astype(np.complex64)
    occ = rng.uniform(0, 2, (ndom, norb))
    beta = rng.standard_normal((ndom, ngrid, nproj)) + (1j * rng.standard_normal((ndom, ngrid, nproj)) if cplx else 0)
    beta = beta.astype(np.complex64 if cplx else np.float32)
    D = rng.uniform(-2, 2, (ndom, nproj))
    A = rng.uniform(-0.3, 0.3, (ndom, 3))
    dom = M.Domain(ndom, grid, h, norb, nproj * (2 if cplx else 1))
    dom.set_vloc(np.zeros((ndom, *grid), dtype=np.float32))
    dom.set_orbitals(psi, occ)
    dom.set_projectors(beta, D)
    check_observables(dom, psi, occ, beta, D, A, h)
    check_observables(dom, psi, occ, beta, D, A[:1], h)          # one field for all domains
    dom.close()


def test_observables_perovskite_domain_tensor_core_projection_and_plane_wave_current():
    """One configs[2]-shaped domain: E_nl through the tcgen05 projection; then plane waves, whose current is the
    closed form of oracle pin J1, on the GPU itself."""
    import paper_2509_00966_b200 as M
    c = W.get_config(2, ndom=1, nsteps=1)
    d = W.generate(c)
    dom = make_domain(c, d)
    assert M.lib().mlmd_gemm_path(dom.handle) == 1
    A = np.array([[0.05, -0.02, 0.03]])
    check_observables(dom, d["psi"], d["occ"], d["beta"], d["D"], A, c.h)
    dom.set_gemm_mode(M.GEMM_LOWP_BF16)
    check_observables(dom, d["psi"], d["occ"], d["beta"], d["D"], A, c.h, lowp=True)
    dom.close()
    grid, h = (16, 16, 16), (0.5, 0.45, 0.4)
    box = [n * s for n, s in zip(grid, h)]
    X, Y, Z = np.meshgrid(*[np.arange(n) * s for n, s in zip(grid, h)], indexing="ij")
    ms = [(1, 0, 0), (0, -2, 0), (2, -1, 4), (-5, 3, -7)]
    f = np.array([[2.0, 1.0, 0.5, 1.5]])
    psi = np.zeros((1, *grid, 4), dtype=np.complex64)
    want = np.zeros(3)
    lam1 = lambda p: (4.0 / 3.0) * np.sin(p) - (1.0 / 6.0) * np.sin(2 * p)
    for n, m in enumerate(ms):
        k = [2 * np.pi * mi / b for mi, b in zip(m, box)]
        psi[0, ..., n] = np.exp(1j * (k[0] * X + k[1] * Y + k[2] * Z)) / np.sqrt(np.prod(box))
        want += f[0, n] * (np.array([lam1(k[d] * h[d]) / h[d] for d in range(3)]) + A[0])
    dom = M.Domain(1, grid, h, 4, 0)
    dom.set_vloc(np.zeros((1, *grid), dtype=np.float32))
    dom.set_orbitals(psi, f)
    assert np.abs(dom.current(A)[0] - want).max() <= 1e-5 * f.sum() / min(h)
    assert dom.energy_nl()[0] == 0.0                               # no projectors
    with pytest.raises(M.MlmdError):
        dom.current(np.zeros((2, 3)))                              # a_ndom must be 1 or ndom
    dom.close()
