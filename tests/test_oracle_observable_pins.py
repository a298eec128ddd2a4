"""Pins of the oracle's observables (oracle/mlmd_ref.c: mlmd_ref_energy_nl, mlmd_ref_current; SURVEY.md 8(f)
NEXT-2, reading D30).  The paper prints no numbers for them: closed forms (rank-1 projector,
plane waves with the finite-difference symbol, real orbitals) and dense Kronecker matrices built here.  CPU only.
"""
import numpy as np

from oracle import ref
from test_oracle_pins import circulant_derivative, rand_c
from test_oracle_split_pins import orthonormal_projectors

RNG = np.random.default_rng(6620259)


def test_e1_rank_one_projector_closed_form():
    """E1: one normalised projector b, psi_n = a_n b + c_n chi (chi orthogonal to b): <b|psi_n> = a_n, so
    E_nl = D sum_n f_n |a_n|^2."""
    grid, h, D = (6, 5, 7), (0.4, 0.5, 0.45), -2.3
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    B = orthonormal_projectors(ngrid, 2, dv)
    a = np.array([0.8 - 0.3j, 0.0, 1.1j])
    c = np.array([0.5 + 0.2j, 1.3, 0.0])
    f = np.array([[2.0, 1.0, 0.5]])
    psi = (a[None, :] * B[:, :1] + c[None, :] * B[:, 1:]).reshape(1, *grid, 3)
    E = ref.energy_nl(psi, f, B[:, :1].reshape(1, ngrid, 1), np.array([[D]]), dv)
    assert abs(E[0] - D * (f[0] * np.abs(a) ** 2).sum()) < 1e-13


def test_e2_dense_matrix_and_batch():
    """E2: E_nl = sum_n f_n dv psi_n^H (dv B D B^H) psi_n with dense numpy matrices, complex non-orthogonal
    projectors, two domains with different data (index order of occ, D, beta per domain)."""
    grid, h = (5, 6, 5), (0.5, 0.4, 0.45)
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    psi = rand_c(2, *grid, 3)
    beta = rand_c(2, ngrid, 4)
    D = RNG.uniform(-2, 2, (2, 4))
    f = RNG.uniform(0, 2, (2, 3))
    E = ref.energy_nl(psi, f, beta, D, dv)
    for dom in range(2):
        x = psi[dom].reshape(ngrid, 3)
        V = dv * (beta[dom] * D[dom][None, :]) @ beta[dom].conj().T
        want = sum(f[dom, n] * dv * np.real(x[:, n].conj() @ V @ x[:, n]) for n in range(3))
        assert abs(E[dom] - want) < 1e-11 * max(1.0, abs(want))


def test_j1_plane_waves_carry_the_finite_difference_velocity():
    """J1: psi = e^{i k.r}/sqrt(Vol): D1 e^{ikx} = i lam1(k h)/h e^{ikx}, lam1(p) = 4/3 sin p - 1/6 sin 2p, so
    J_d = sum_n f_n (lam1(k_nd h_d)/h_d + A_d)."""
    grid, h = (12, 10, 16), (0.5, 0.45, 0.4)
    box = [n * s for n, s in zip(grid, h)]
    ax = [np.arange(n) * s for n, s in zip(grid, h)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    ms = [(1, 0, 0), (0, -2, 0), (2, -1, 4), (-5, 3, -7)]
    f = np.array([[2.0, 1.0, 0.5, 1.5]])
    A = np.array([[0.07, -0.04, 0.11]])
    psi = np.zeros((1, *grid, len(ms)), dtype=np.complex128)
    want = np.zeros(3)
    lam1 = lambda p: (4.0 / 3.0) * np.sin(p) - (1.0 / 6.0) * np.sin(2 * p)
    for n, m in enumerate(ms):
        k = [2 * np.pi * mi / b for mi, b in zip(m, box)]
        psi[0, ..., n] = np.exp(1j * (k[0] * X + k[1] * Y + k[2] * Z)) / np.sqrt(np.prod(box))
        want += f[0, n] * (np.array([lam1(k[d] * h[d]) / h[d] for d in range(3)]) + A[0])
    J = ref.current(psi, f, A, h)
    assert np.abs(J[0] - want).max() < 1e-12


def test_j2_real_orbitals_carry_only_the_diamagnetic_current():
    """J2: for real psi, <psi|-i D1|psi> is purely imaginary: J = A * sum_n f_n ||psi_n||^2."""
    grid, h = (6, 5, 7), (0.4, 0.5, 0.45)
    dv = float(np.prod(h))
    psi = RNG.standard_normal((1, *grid, 3)).astype(np.complex128)
    f = np.array([[2.0, 1.0, 0.5]])
    A = np.array([[0.3, -0.2, 0.1]])
    ne = (f[0] * dv * (np.abs(psi[0]) ** 2).sum(axis=(0, 1, 2))).sum()
    assert np.abs(ref.current(psi, f, A, h)[0] - A[0] * ne).max() < 1e-12


def test_j3_dense_kronecker_derivatives_per_domain_field():
    """J3: J_d = sum_n f_n dv Re psi_n^H (-i D1_d + A_d) psi_n with circulant first-derivative matrices put on
    the right axis by Kronecker products; two domains, each with its own field."""
    grid, h = (5, 6, 7), (0.5, 0.4, 0.45)
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    psi = rand_c(2, *grid, 2)
    f = RNG.uniform(0, 2, (2, 2))
    A = RNG.uniform(-0.3, 0.3, (2, 3))
    J = ref.current(psi, f, A, h)
    eye = [np.eye(n) for n in grid]
    for dom in range(2):
        x = psi[dom].reshape(ngrid, 2)
        for d in range(3):
            parts = list(eye)
            parts[d] = circulant_derivative(grid[d], h[d], 1)
            D1 = np.kron(np.kron(parts[0], parts[1]), parts[2])
            want = sum(f[dom, n] * dv * np.real(x[:, n].conj() @ (-1j * (D1 @ x[:, n]) + A[dom, d] * x[:, n])) for n in range(2))
            assert abs(J[dom, d] - want) < 1e-11
