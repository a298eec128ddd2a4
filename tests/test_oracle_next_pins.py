"""Pins of the oracle functions added for SURVEY.md 8(f) NEXT-2 (nonlocal part of the current) and
NEXT-3 (the paper's own 2nd-order / 7-point local discretisation).  The paper prints no
numbers for either, so the expected values come from independent routes: weights solved from their Taylor-matching
definition, plane-wave symbols, polynomial exactness, convergence order, dense commutators and a gauge derivative.
CPU only.
"""
import math

import numpy as np

from oracle import ref
from test_oracle_pins import p4, rand_c

RNG = np.random.default_rng(966203)


# ---- NEXT-3: 2nd-order central differences (flag ref.ORDER2) ------------------------------------------------
def fd_weights3(order_of_derivative):
    """3-point central weights from their definition: sum_j w_j j^m = m! delta(m, order), m = 0..2 (solved)."""
    j = np.arange(-1, 2, dtype=np.float64)
    V = np.vander(j, 3, increasing=True).T
    rhs = np.zeros(3)
    rhs[order_of_derivative] = math.factorial(order_of_derivative)
    return np.linalg.solve(V, rhs)


def dense_h_order2(grid, h, vloc, A):
    I = [np.eye(n) for n in grid]
    H = np.zeros((int(np.prod(grid)),) * 2, dtype=np.complex128)
    for d in range(3):
        for order, coef in ((2, -0.5), (1, -1j * A[d])):
            w = fd_weights3(order) / h[d] ** order
            M = np.zeros((grid[d], grid[d]))
            for i in range(grid[d]):
                for jj, wj in zip((-1, 0, 1), w):
                    M[i, (i + jj) % grid[d]] += wj
            parts = list(I)
            parts[d] = M
            H += coef * np.kron(np.kron(parts[0], parts[1]), parts[2])
    return H + np.diag(vloc.reshape(-1) + 0.5 * float(np.dot(A, A)))


def test_o2a_weights_are_the_seven_point_star():
    assert np.allclose(fd_weights3(2), [1, -2, 1], atol=1e-14) and np.allclose(fd_weights3(1), [-0.5, 0, 0.5], atol=1e-14)


def test_o2b_plane_wave_symbol_and_taylor_factor():
    """e^{ik.r} is an eigenvector with eps = sum_d [ (1 - cos p_d)/h_d^2 + A_d sin(p_d)/h_d ] + |A|^2/2, p = k h
    (lambda2 = 2 - 2 cos p, lambda1 = sin p); n steps multiply it by P4(-i dt eps)^n."""
    grid, h, dt, nsteps = (12, 10, 16), (0.5, 0.45, 0.4), 0.02, 5
    A = np.array([0.07, -0.04, 0.11])
    box = [n * s for n, s in zip(grid, h)]
    ax = [np.arange(n) * s for n, s in zip(grid, h)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    ms = [(0, 0, 0), (1, 0, 0), (0, -2, 0), (2, -1, 4), (-5, 3, -7), (6, 5, 8)]
    psi = np.zeros((1, *grid, len(ms)), dtype=np.complex128)
    eps = []
    for n, m in enumerate(ms):
        k = [2 * np.pi * mi / b for mi, b in zip(m, box)]
        psi[0, ..., n] = np.exp(1j * (k[0] * X + k[1] * Y + k[2] * Z))
        eps.append(sum(0.5 * (2 - 2 * np.cos(k[d] * h[d])) / h[d] ** 2 + A[d] * np.sin(k[d] * h[d]) / h[d] for d in range(3))
                   + 0.5 * A @ A)
    out, _ = ref.propagate(psi, np.ones((1, len(ms))), np.zeros((1, *grid)), None, None, np.tile(A, (nsteps, 1, 1)), dt, h,
                           flags=ref.ORDER2)
    for n, e in enumerate(eps):
        assert np.abs(out[0, ..., n] - p4(-1j * dt * e) ** nsteps * psi[0, ..., n]).max() < 1e-13


def test_o2c_dense_operator_anisotropic_grid():
    """applyH(flag ORDER2) against a dense matrix built from the SOLVED 3-point weights on a 6x5x7 grid."""
    grid, h = (6, 5, 7), (0.41, 0.37, 0.45)
    vloc = RNG.uniform(-1, 1, grid)
    A = np.array([0.2, -0.1, 0.15])
    u = rand_c(*grid, 2)
    got = ref.apply_h(u, vloc, None, None, A, h, flags=ref.ORDER2)
    want = (dense_h_order2(grid, h, vloc, A) @ u.reshape(-1, 2)).reshape(*grid, 2)
    assert np.abs(got - want).max() < 1e-12 * np.abs(want).max()
    # and it is NOT the 4th-order operator
    assert np.abs(ref.apply_h(u, vloc, None, None, A, h) - got).max() > 1e-2 * np.abs(want).max()


def test_o2d_second_order_convergence_and_polynomial_exactness():
    """-1/2 D2 applied to sin(kx) converges to k^2/2 sin(kx) with error ratio 4 when h halves (4th order would give
    16); a quadratic is differentiated exactly in the interior of a long axis."""
    errs = []
    for n in (16, 32, 64):
        L = 2 * np.pi
        h = L / n
        x = np.arange(n) * h
        u = np.zeros((n, 5, 5, 1), dtype=np.complex128)
        u[:, :, :, 0] = np.sin(2 * x)[:, None, None]
        out = ref.apply_h(u, np.zeros((n, 5, 5)), None, None, np.zeros(3), (h, 1.0, 1.0), flags=ref.ORDER2)
        errs.append(np.abs(out[:, 0, 0, 0] - 2.0 * np.sin(2 * x)).max())
    assert 3.7 < errs[0] / errs[1] < 4.3 and 3.85 < errs[1] / errs[2] < 4.15
    n, h = 24, 0.3
    x = (np.arange(n) - 12) * h
    u = np.zeros((n, 5, 5, 1), dtype=np.complex128)
    u[:, :, :, 0] = (1.5 * x ** 2 - 0.7 * x + 2.0)[:, None, None]
    A = np.array([0.3, 0.0, 0.0])
    out = ref.apply_h(u, np.zeros((n, 5, 5)), None, None, A, (h, 1.0, 1.0), flags=ref.ORDER2)[:, 0, 0, 0]
    want = -0.5 * 3.0 - 1j * A[0] * (3.0 * x - 0.7) + 0.5 * A[0] ** 2 * (1.5 * x ** 2 - 0.7 * x + 2.0)
    assert np.abs(out[2:-2] - want[2:-2]).max() < 1e-11       # away from the periodic seam


def test_o2e_plane_waves_carry_the_second_order_velocity():
    """The local current with the 2nd-order first difference: D1 e^{ikx} = i sin(k h)/h e^{ikx}."""
    grid, h = (12, 10, 16), (0.5, 0.45, 0.4)
    box = [n * s for n, s in zip(grid, h)]
    ax = [np.arange(n) * s for n, s in zip(grid, h)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    ms = [(1, 0, 0), (0, -2, 0), (2, -1, 4), (-5, 3, -7)]
    f = np.array([[2.0, 1.0, 0.5, 1.5]])
    A = np.array([[0.07, -0.04, 0.11]])
    psi = np.zeros((1, *grid, len(ms)), dtype=np.complex128)
    want = np.zeros(3)
    for n, m in enumerate(ms):
        k = [2 * np.pi * mi / b for mi, b in zip(m, box)]
        psi[0, ..., n] = np.exp(1j * (k[0] * X + k[1] * Y + k[2] * Z)) / np.sqrt(np.prod(box))
        want += f[0, n] * (np.array([np.sin(k[d] * h[d]) / h[d] for d in range(3)]) + A[0])
    assert np.abs(ref.current(psi, f, A, h, flags=ref.ORDER2)[0] - want).max() < 1e-12


# ---- NEXT-2: nonlocal part of the current --------------------------------------------------------------------
def test_c1_dense_commutator_any_diagonal_position_operator():
    """<psi| -i [X_d, V_NL] |psi> with V_NL = dv B D B^H as a dense matrix and X_d ANY real diagonal matrix; the
    oracle gets rbeta_d = X_d beta.  Complex non-orthogonal projectors, two domains with their own data."""
    grid, h = (6, 5, 7), (0.41, 0.37, 0.45)
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    psi = rand_c(2, *grid, 3)
    beta = rand_c(2, ngrid, 4)
    D = RNG.uniform(-2, 2, (2, 4))
    f = RNG.uniform(0, 2, (2, 3))
    X = RNG.uniform(-3, 3, (3, 2, ngrid))
    rbeta = X[:, :, :, None] * beta[None]
    J = ref.current_nl(psi, f, beta, rbeta, D, dv)
    for dom in range(2):
        V = dv * (beta[dom] * D[dom][None, :]) @ beta[dom].conj().T
        x = psi[dom].reshape(ngrid, 3)
        for d in range(3):
            Xd = np.diag(X[d, dom])
            comm = -1j * (Xd @ V - V @ Xd)
            want = sum(f[dom, n] * dv * (x[:, n].conj() @ comm @ x[:, n]) for n in range(3))
            assert abs(want.imag) < 1e-10 and abs(J[dom, d] - want.real) < 1e-10 * max(1.0, abs(want.real))


def test_c2_gauge_derivative_of_the_nonlocal_energy():
    """A uniform field enters the nonlocal operator through the gauge phases beta_p -> e^{-i A.(r - R_p)} beta_p, so
    dE_nl/dA_d at A = 0 is the nonlocal current.  Central finite difference of the (separately pinned, E1-E2)
    nonlocal energy of the phased projectors against the oracle's current_nl."""
    grid, h = (6, 5, 7), (0.4, 0.5, 0.45)
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    psi = rand_c(1, *grid, 3)
    beta = RNG.standard_normal((1, ngrid, 4)).astype(np.complex128)
    D = RNG.uniform(-2, 2, (1, 4))
    f = np.array([[2.0, 1.0, 0.5]])
    X = RNG.uniform(-2, 2, (3, 1, ngrid, 4))          # (r - R_p)_d: may differ per projector (its own centre)
    J = ref.current_nl(psi, f, beta, X * beta[None], D, dv)
    eps = 1e-5
    for d in range(3):
        E = [ref.energy_nl(psi, f, np.exp(-1j * s * eps * X[d]) * beta, D, dv)[0] for s in (+1, -1)]
        assert abs((E[0] - E[1]) / (2 * eps) - J[0, d]) < 1e-7 * max(1.0, abs(J[0, d]))


def test_c3_real_orbitals_and_real_projectors_carry_no_nonlocal_current():
    grid, h = (5, 6, 5), (0.5, 0.4, 0.45)
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    psi = RNG.standard_normal((1, *grid, 2)).astype(np.complex128)
    beta = RNG.standard_normal((1, ngrid, 3)).astype(np.complex128)
    X = RNG.uniform(-2, 2, (3, 1, ngrid, 1))
    J = ref.current_nl(psi, np.array([[2.0, 1.0]]), beta, X * beta[None], RNG.uniform(-1, 1, (1, 3)), dv)
    assert np.abs(J).max() < 1e-12


def test_o2f_eq2_step_on_second_order_differences_from_dense_matrices():
    """O2f: mlmd_ref_propagate_split(order=2) = kick, Taylor-4 of the dense 2nd-order h_loc (Vandermonde-solved weights), kick:
    the order switch reaches the local propagator of the Eq. (2) step and nothing else."""
    from oracle import ref
    from test_oracle_pins import rand_c, rel
    grid, h, dt, nsteps = (5, 6, 5), (0.5, 0.4, 0.45), 0.04, 2
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    psi = rand_c(1, *grid, 3)
    vloc = RNG.uniform(-1, 0.5, (1, *grid))
    beta = rand_c(1, ngrid, 4) * 0.6
    D = RNG.uniform(-2, 2, (1, 4))
    A = RNG.uniform(-0.2, 0.2, (nsteps, 1, 3))
    out, _ = ref.propagate_split(psi, np.full((1, 3), 2.0), vloc, beta, D, A, dt, h, order=2)
    x = psi[0].reshape(ngrid, 3).astype(np.complex128)
    V = dv * (beta[0] * D[0][None, :]) @ beta[0].conj().T

    def kick(y):
        z = y - 0.5j * dt * (V @ y)
        return z * (np.linalg.norm(y, axis=0) / np.linalg.norm(z, axis=0))[None, :]
    for n in range(nsteps):
        x = kick(x)
        z = -1j * dt * dense_h_order2(grid, h, vloc[0], A[n, 0])
        term, acc = x.copy(), x.copy()
        for m in range(1, 5):
            term = z @ term / m
            acc = acc + term
        x = kick(acc)
    assert rel(out[0].reshape(ngrid, 3), x) < 1e-12
    o4, _ = ref.propagate_split(psi, np.full((1, 3), 2.0), vloc, beta, D, A, dt, h)
    assert rel(o4, out) > 1e-4          # the 4th-order step is a different operator
