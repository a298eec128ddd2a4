"""Pins of the oracle's block-diagonal split-operator local solver (oracle/mlmd_ref.c: mlmd_ref_local_richardson and
the `local="richardson"` form of mlmd_ref_propagate_split, reading D33).

PAPER.md L147 names the solver ("a block-diagonal split-operator solver for electronic wave functions [41]",
"uniform operations on nearest-neighbor mesh points") and L283 the 7-point stencil it is based on; it prints neither a
formula nor a number.  The pins therefore are: the pair matrices built HERE add up to the 2nd-order operator whose
weights are solved from their Taylor-matching definition (test_oracle_next_pins.dense_h_order2); every factor as a dense
scipy expm (not the oracle's closed 2 x 2 form); closed-form eigenvectors of all pair blocks at once; unitarity for any
dt; time reversal; the order of convergence against expm of the whole operator; the whole Eq. (2) step from dense
matrices.  CPU only; nothing re-calls the oracle to check itself.
"""
import numpy as np
import pytest
import scipy.linalg

from oracle import ref
from test_oracle_pins import rand_c, rel
from test_oracle_next_pins import dense_h_order2

RNG = np.random.default_rng(96620341)


def pair_matrix(n, parity, a, b):
    """Dense 1-D matrix that couples the pairs (j, j+1 mod n), j = parity, parity + 2, ...: a/2 on both diagonal
    entries of a pair, b from j+1 to j, conj(b) back."""
    M = np.zeros((n, n), dtype=np.complex128)
    for j in range(parity, n, 2):
        jn = (j + 1) % n
        M[j, j] += a / 2
        M[jn, jn] += a / 2
        M[j, jn] += b
        M[jn, j] += np.conj(b)
    return M


def on_axis(grid, d, M):
    parts = [np.eye(n) for n in grid]
    parts[d] = M
    return np.kron(np.kron(parts[0], parts[1]), parts[2])


def pair_operators(grid, h, A):
    """[(E_d, O_d)] as dense matrices on the whole grid."""
    out = []
    for d in range(3):
        a = 1.0 / h[d] ** 2
        b = -0.5 / h[d] ** 2 - 1j * A[d] / (2 * h[d])
        out.append((on_axis(grid, d, pair_matrix(grid[d], 0, a, b)), on_axis(grid, d, pair_matrix(grid[d], 1, a, b))))
    return out


def dense_u_loc(grid, h, vloc, A, dt):
    E = scipy.linalg.expm
    P = np.diag(np.exp(-0.5j * dt * (vloc.reshape(-1) + 0.5 * float(np.dot(A, A)))))
    U = np.eye(int(np.prod(grid)), dtype=np.complex128)
    for Ed, Od in pair_operators(grid, h, A):
        U = U @ (E(-0.5j * dt * Ed) @ E(-1j * dt * Od) @ E(-0.5j * dt * Ed))
    return P @ U @ P


def test_r1_pair_matrices_add_up_to_the_pinned_second_order_operator():
    """R1: sum_d (E_d + O_d) + diag(V + 1/2|A|^2) is the 2nd-order h_loc whose weights are solved from their definition
    (pins O2a-O2c fix the oracle's own apply_h to the same matrix): fixes a_d, b_d, the sign of the A term, the wrap."""
    grid, h = (4, 6, 8), (0.5, 0.4, 0.45)
    vloc = RNG.uniform(-1, 0.5, grid)
    A = np.array([0.2, -0.15, 0.1])
    H = np.diag(vloc.reshape(-1) + 0.5 * float(np.dot(A, A))).astype(np.complex128)
    for Ed, Od in pair_operators(grid, h, A):
        H += Ed + Od
    assert np.abs(H - dense_h_order2(grid, h, vloc, A)).max() < 1e-13
    u = rand_c(*grid, 2)
    got = ref.apply_h(u, vloc, None, None, A, h, flags=ref.ORDER2)
    assert rel(got.reshape(-1, 2), H @ u.reshape(-1, 2)) < 1e-13


def test_r2_every_factor_as_a_dense_matrix_exponential():
    """R2: U_loc = P S_x S_y S_z P with each exp(-i tau E_d), exp(-i tau O_d) taken by scipy expm of the dense pair
    matrix: fixes the closed 2 x 2 exponential, the pairing (even / odd / wrap pair), tau = dt/2, dt, dt/2 and the phases."""
    grid, h, dt = (4, 6, 4), (0.5, 0.4, 0.45), 0.35
    vloc = RNG.uniform(-1, 0.5, grid)
    A = np.array([0.2, -0.15, 0.1])
    psi = rand_c(*grid, 3)
    got = ref.local_richardson(psi, vloc, A, dt, h)
    want = dense_u_loc(grid, h, vloc, A, dt) @ psi.reshape(-1, 3)
    assert rel(got.reshape(-1, 3), want) < 1e-12


def test_r3_joint_eigenvectors_of_all_pair_blocks_closed_form():
    """R3: with V = 0, A = 0 the constant function is annihilated by every pair block (a/2 + b = 0) and the alternating
    function (-1)^(i+j+k) is an eigenvector of every block with eigenvalue a_d: U_loc multiplies it by
    exp(-2 i dt sum_d 1/h_d^2) for ANY dt, no matrix involved.  (2/h^2 is the top of the 2nd-order kinetic band.)"""
    grid, h, dt = (6, 4, 8), (0.5, 0.4, 0.3), 0.8
    i, j, k = np.meshgrid(*[np.arange(n) for n in grid], indexing="ij")
    alt = ((-1.0) ** (i + j + k)).astype(np.complex128)
    psi = np.stack([np.ones(grid, dtype=np.complex128), alt, (0.3 - 0.7j) * alt + 2.0], axis=-1)
    got = ref.local_richardson(psi, np.zeros(grid), np.zeros(3), dt, h)
    ph = np.exp(-2j * dt * sum(1.0 / x ** 2 for x in h))
    want = np.stack([np.ones(grid, dtype=np.complex128), ph * alt, (0.3 - 0.7j) * ph * alt + 2.0], axis=-1)
    assert np.abs(got - want).max() < 1e-13


def test_r4_unitary_for_any_dt_and_time_reversible():
    """R4: every factor is unitary, so norms and overlaps are kept for any dt (the Taylor step is stable only for
    dt |h| <= 2 sqrt 2), and the symmetric product gives U(-dt) U(dt) = 1."""
    grid, h = (6, 8, 6), (0.4, 0.35, 0.45)
    vloc = RNG.uniform(-2, 1, grid)
    A = np.array([0.3, 0.1, -0.2])
    psi = rand_c(*grid, 4)
    g0 = psi.reshape(-1, 4).conj().T @ psi.reshape(-1, 4)
    for dt in (0.02, 0.7, 25.0):
        out = ref.local_richardson(psi, vloc, A, dt, h)
        g1 = out.reshape(-1, 4).conj().T @ out.reshape(-1, 4)
        assert np.abs(g1 - g0).max() / np.abs(g0).max() < 1e-13
        back = ref.local_richardson(out, vloc, A, -dt, h)
        assert rel(back, psi) < 1e-12


def test_r5_second_order_in_dt_against_expm_of_the_whole_operator():
    """R5: one step differs from expm(-i dt h_loc) by O(dt^3) (halving dt divides the error by 8), n steps over a fixed
    time by O(dt^2): the symmetric splitting, not a first-order one (E O instead of E/2 O E/2 would give 4 and 2)."""
    grid, h = (4, 6, 4), (0.5, 0.45, 0.4)
    vloc = RNG.uniform(-1, 0.5, grid)
    A = np.array([0.2, -0.1, 0.15])
    psi = rand_c(*grid, 2)
    H = dense_h_order2(grid, h, vloc, A)
    errs = []
    for dt in (0.04, 0.02, 0.01):
        want = scipy.linalg.expm(-1j * dt * H) @ psi.reshape(-1, 2)
        errs.append(rel(ref.local_richardson(psi, vloc, A, dt, h).reshape(-1, 2), want))
    assert 7.0 < errs[0] / errs[1] < 9.0 and 7.0 < errs[1] / errs[2] < 9.0
    T, tot = 0.32, []
    for n in (8, 16, 32):
        x = psi
        for _ in range(n):
            x = ref.local_richardson(x, vloc, A, T / n, h)
        tot.append(rel(x.reshape(-1, 2), scipy.linalg.expm(-1j * T * H) @ psi.reshape(-1, 2)))
    assert 3.5 < tot[0] / tot[1] < 4.5 and 3.5 < tot[1] / tot[2] < 4.5


def test_r6_whole_eq2_step_with_the_split_operator_local_solver():
    """R6: mlmd_ref_propagate_split(local="richardson") = kick, U_loc, kick from dense matrices (complex non-orthogonal
    projectors, per-domain midpoint field, three steps), and its density."""
    grid, h, dt, nsteps = (4, 6, 4), (0.5, 0.4, 0.45), 0.05, 3
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    psi = rand_c(2, *grid, 3)
    vloc = RNG.uniform(-1, 0.5, (2, *grid))
    beta = rand_c(2, ngrid, 4) * 0.6
    D = RNG.uniform(-2, 2, (2, 4))
    A = RNG.uniform(-0.2, 0.2, (nsteps, 2, 3))
    occ = np.array([[2.0, 1.0, 0.5]] * 2)
    out, rho = ref.propagate_split(psi, occ, vloc, beta, D, A, dt, h, local="richardson")

    def kick(x, V):
        y = x - 0.5j * dt * (V @ x)
        return y * (np.linalg.norm(x, axis=0) / np.linalg.norm(y, axis=0))[None, :]
    for dom in range(2):
        x = psi[dom].reshape(ngrid, 3).astype(np.complex128)
        V = dv * (beta[dom] * D[dom][None, :]) @ beta[dom].conj().T
        for n in range(nsteps):
            x = kick(dense_u_loc(grid, h, vloc[dom], A[n, dom], dt) @ kick(x, V), V)
        assert rel(out[dom].reshape(ngrid, 3), x) < 1e-12
        assert np.allclose(rho[dom].reshape(-1), (np.abs(x) ** 2 * occ[dom][None, :]).sum(1), rtol=1e-12, atol=0)
    # without projectors the step is U_loc alone
    o2, _ = ref.propagate_split(psi[:1], occ[:1], vloc[:1], None, None, A[:1, :1], dt, h, local="richardson")
    assert rel(o2[0], ref.local_richardson(psi[0], vloc[0], A[0, 0], dt, h)) < 1e-15


def test_r7_odd_axis_is_rejected():
    """R7: the pairing needs an even number of points on every periodic axis."""
    with pytest.raises(RuntimeError):
        ref.local_richardson(rand_c(4, 5, 6, 1), np.zeros((4, 5, 6)), np.zeros(3), 0.1, (0.4, 0.4, 0.4))
