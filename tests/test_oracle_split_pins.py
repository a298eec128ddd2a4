"""Pins of the oracle's literal Eq. (2) step (oracle/mlmd_ref.c: mlmd_ref_propagate_split).

PAPER.md Eq. (2): psi <- K exp(-i dt h_loc) K psi with K = (1 - i dt/2 v_nl)/||1 - i dt/2 v_nl||
(readings D27, D28 in DESIGN.md).  The paper prints no numbers for it, so the pins are closed forms,
a special case that reduces to the already-pinned Taylor step, dense linear algebra built here from
Kronecker products, and the splitting order.  CPU only; nothing re-calls the oracle to check itself.
"""
import numpy as np
import scipy.linalg

from oracle import ref
from test_oracle_pins import dense_h, rand_c, rel

RNG = np.random.default_rng(96620250)


def orthonormal_projectors(ngrid, nproj, dv):
    """Columns with <b_p|b_q> = dv sum conj(b_p) b_q = delta_pq."""
    q, _ = np.linalg.qr(RNG.standard_normal((ngrid, nproj)) + 1j * RNG.standard_normal((ngrid, nproj)))
    return q / np.sqrt(dv)


def test_s1_rank_one_kick_closed_form():
    """S1: one normalised projector b, psi = a b + c chi with chi orthogonal to b.  v_nl psi = D a b, so
    a half-kick maps (a, c) -> (a (1 - i tau D), c) * sqrt((|a|^2+|c|^2)/(|a|^2 (1+tau^2 D^2)+|c|^2)):
    two-number arithmetic, no grid."""
    grid, h, dt, D = (6, 5, 7), (0.4, 0.5, 0.45), 0.07, 3.1
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    B = orthonormal_projectors(ngrid, 2, dv)
    b, chi = B[:, 0], B[:, 1]
    coef = np.array([[0.8 - 0.3j, 0.5 + 0.2j], [0.0, 1.3], [1.1j, 0.0]])     # (a, c) per orbital
    psi = (coef[:, 0][None, :] * b[:, None] + coef[:, 1][None, :] * chi[:, None]).reshape(1, *grid, 3)
    out, _ = ref.propagate_split(psi, np.full((1, 3), 2.0), np.zeros((1, *grid)), b.reshape(1, ngrid, 1),
                                 np.array([[D]]), np.zeros((2, 1, 3)), dt, h, nsteps=2, kick_only=True)
    tau = dt / 2
    exp = coef.astype(np.complex128).copy()
    for _ in range(4):                                                      # 2 steps x 2 half-kicks
        for n in range(3):
            a, c = exp[n]
            s = np.sqrt((abs(a) ** 2 + abs(c) ** 2) / (abs(a) ** 2 * (1 + tau ** 2 * D ** 2) + abs(c) ** 2))
            exp[n] = [a * (1 - 1j * tau * D) * s, c * s]
    want = (exp[:, 0][None, :] * b[:, None] + exp[:, 1][None, :] * chi[:, None]).reshape(1, *grid, 3)
    assert rel(out, want) < 1e-13


def test_s2_without_nonlocal_part_it_is_the_taylor_step():
    """S2: nproj = 0 or D = 0 turns K into the identity; the step is then the Taylor-4 step of h_loc,
    which pins P1..P12 already fix (same bits for nproj = 0)."""
    grid, h, dt = (6, 7, 5), (0.5, 0.45, 0.4), 0.03
    ngrid = int(np.prod(grid))
    psi = rand_c(2, *grid, 3)
    vloc = RNG.uniform(-1, 0.5, (2, *grid))
    A = RNG.uniform(-0.1, 0.1, (3, 2, 3))
    occ = np.full((2, 3), 2.0)
    a, ra = ref.propagate_split(psi, occ, vloc, None, None, A, dt, h)
    b, rb = ref.propagate(psi, occ, vloc, None, None, A, dt, h)
    assert np.array_equal(a, b) and np.array_equal(ra, rb)
    beta = rand_c(2, ngrid, 4)
    c, _ = ref.propagate_split(psi, occ, vloc, beta, np.zeros((2, 4)), A, dt, h)
    assert rel(c, b) < 1e-14


def test_s3_eigenvectors_of_vnl_pick_up_the_kick_phase():
    """S3: orthonormal projectors are eigenvectors of v_nl with eigenvalue D_p; the normalised kick is
    then the pure phase (1 - i tau D)/|1 - i tau D| = exp(-i atan(tau D)), twice per step."""
    grid, h, dt, nsteps = (5, 6, 5), (0.5, 0.4, 0.45), 0.11, 3
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    D = np.array([2.0, -1.5, 0.3, 7.0])
    B = orthonormal_projectors(ngrid, 4, dv)
    psi = (B * np.array([1.0, 0.5j, -2.0, 0.1 + 0.1j])[None, :]).reshape(1, *grid, 4)
    out, _ = ref.propagate_split(psi, np.full((1, 4), 2.0), np.zeros((1, *grid)), B.reshape(1, ngrid, 4), D[None, :],
                                 np.zeros((nsteps, 1, 3)), dt, h, kick_only=True)
    want = psi * np.exp(-2j * nsteps * np.arctan(0.5 * dt * D))[None, None, None, None, :]
    assert rel(out, want) < 1e-13


def dense_split_step(psi, Hloc, V, dt):
    def kick(x):
        y = x - 0.5j * dt * (V @ x)
        return y * (np.linalg.norm(x, axis=0) / np.linalg.norm(y, axis=0))[None, :]
    x = kick(psi)
    z = -1j * dt * Hloc
    term, acc = x.copy(), x.copy()
    for m in range(1, 5):
        term = z @ term / m
        acc += term
    return kick(acc)


def test_s4_dense_matrices_on_a_tiny_grid():
    """S4: the whole step rebuilt from dense matrices (Kronecker-product h_loc, dv B D B^H) with complex,
    non-orthogonal projectors, a field, a local potential, per-domain A and three steps: fixes the order
    kick / local / kick, the dt/2, the sign, the midpoint field and the per-orbital normalisation."""
    grid, h, dt, nsteps = (5, 6, 5), (0.5, 0.4, 0.45), 0.04, 3
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    psi = rand_c(2, *grid, 3)
    vloc = RNG.uniform(-1, 0.5, (2, *grid))
    beta = rand_c(2, ngrid, 4) * 0.6
    D = RNG.uniform(-2, 2, (2, 4))
    A = RNG.uniform(-0.2, 0.2, (nsteps, 2, 3))
    out, rho = ref.propagate_split(psi, np.array([[2.0, 1.0, 0.5]] * 2), vloc, beta, D, A, dt, h)
    for dom in range(2):
        x = psi[dom].reshape(ngrid, 3).astype(np.complex128)
        V = dv * (beta[dom] * D[dom][None, :]) @ beta[dom].conj().T
        for n in range(nsteps):
            x = dense_split_step(x, dense_h(grid, h, vloc[dom], None, None, A[n, dom]), V, dt)
        assert rel(out[dom].reshape(ngrid, 3), x) < 1e-12
        want_rho = (np.abs(x) ** 2 * np.array([2.0, 1.0, 0.5])[None, :]).sum(1)
        assert np.allclose(rho[dom].reshape(-1), want_rho, rtol=1e-12, atol=0)


def test_s5_leading_error_term_of_the_first_order_kick():
    """S5: K(tau) psi = (1 - i tau V - tau^2 <V^2>/2 + ..) psi while exp(-i tau V) psi =
    (1 - i tau V - tau^2 V^2/2 + ..) psi, <V^2> = <psi|V^2|psi>/<psi|psi>; the symmetric arrangement cancels
    the commutator term, so against expm(-i dt (h_loc + v_nl)) one step errs by
        dt^2/4 (V^2 - <V^2>) psi + O(dt^3)
    ("first-order" nonlocal correction, Eq. (2)).  A kick of dt instead of dt/2 makes the error
    4x this, a single kick half of it, an un-normalised kick a different vector, kicks on one side add a
    commutator term: each fails the 4% match; the O(dt^3) remainder is checked by halving dt."""
    grid, h = (5, 6, 5), (0.5, 0.4, 0.45)
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    psi = rand_c(1, *grid, 2)
    vloc = RNG.uniform(-1, 0.5, (1, *grid))
    beta = rand_c(1, ngrid, 3) * 0.5
    D = np.array([[1.0, -0.7, 0.4]])
    A = np.array([[[0.05, -0.02, 0.03]]])
    H = dense_h(grid, h, vloc[0], beta[0], D[0], A[0, 0])
    V = dv * (beta[0] * D[0][None, :]) @ beta[0].conj().T
    x = psi[0].reshape(ngrid, 2)
    V2x = V @ (V @ x)
    ev = np.real(np.sum(x.conj() * V2x, 0) / np.sum(np.abs(x) ** 2, 0))
    mism = []
    for dt in (0.002, 0.001):
        out, _ = ref.propagate_split(psi, np.full((1, 2), 2.0), vloc, beta, D, A, dt, h)
        exact = scipy.linalg.expm(-1j * dt * H) @ x
        pred = dt ** 2 / 4 * (V2x - ev[None, :] * x)
        mism.append(rel(out[0].reshape(ngrid, 2) - exact, pred))
    assert mism[1] < 0.04, mism
    assert 1.7 < mism[0] / mism[1] < 2.3, mism


def test_o1_two_level_rotation_closed_form():
    """O1 (reading D29): Psi(t) = Psi(0) U with a rotation by theta between a filled (f=2) and an empty orbital
    and a pure phase on a third, half-filled one: f(t) = (2 cos^2, 2 sin^2, 1), n_exc = 2 sin^2 theta."""
    th = 0.37
    U = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, np.exp(0.9j)]], dtype=np.complex128)
    f, nexc = ref.occupations(U[None], np.array([[2.0, 0.0, 1.0]]))
    assert np.allclose(f[0], [2 * np.cos(th) ** 2, 2 * np.sin(th) ** 2, 1.0], atol=1e-15)
    assert abs(nexc[0] - 2 * np.sin(th) ** 2) < 1e-15


def test_o2_sum_rule_phases_and_t0():
    """O2: for unitary S the electrons are conserved (sum_s f_s(t) = sum_n f_n) and n_exc = (sum_s |f_s(t) - f_s(0)|)/2;
    column phases of S do not matter; S = 1 gives f(t) = f(0), n_exc = 0; the s and n indices are not interchangeable
    (a non-normal S distinguishes them)."""
    n = 6
    q, _ = np.linalg.qr(RNG.standard_normal((n, n)) + 1j * RNG.standard_normal((n, n)))
    occ = np.array([[2.0, 2.0, 1.5, 0.5, 0.0, 0.0]])
    f, nexc = ref.occupations(q[None], occ)
    assert abs(f.sum() - occ.sum()) < 1e-13
    assert abs(nexc[0] - 0.5 * np.abs(f - occ).sum()) < 1e-13
    f2, nexc2 = ref.occupations((q * np.exp(1j * RNG.uniform(0, 6, n))[None, :])[None], occ)
    assert np.allclose(f, f2, atol=1e-14) and abs(nexc[0] - nexc2[0]) < 1e-14
    f0, n0 = ref.occupations(np.eye(n, dtype=np.complex128)[None], occ)
    assert np.array_equal(f0, occ) and n0[0] == 0.0
    S = np.zeros((1, 2, 2), dtype=np.complex128)
    S[0, 0, 1] = 1.0                                   # <psi_0(0)|psi_1(t)> = 1: orbital 1's electrons sit on reference 0
    f3, n3 = ref.occupations(S, np.array([[0.0, 2.0]]))
    assert np.array_equal(f3, [[2.0, 0.0]]) and n3[0] == 2.0


def test_o3_occupations_from_the_oracles_own_overlap():
    """O3: end to end through mlmd_ref_overlap: orbitals mixed by a known unitary give the O1 numbers on a grid."""
    grid, h = (5, 6, 5), (0.5, 0.4, 0.45)
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    B = orthonormal_projectors(ngrid, 2, dv)
    th = 1.1
    U = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    psi0 = B.reshape(1, *grid, 2)
    psit = (B @ U).reshape(1, *grid, 2)
    f, nexc = ref.occupations(ref.overlap(psi0, psit, dv), np.array([[2.0, 0.0]]))
    assert np.allclose(f[0], [2 * np.cos(th) ** 2, 2 * np.sin(th) ** 2], atol=1e-13)
    assert abs(nexc[0] - 2 * np.sin(th) ** 2) < 1e-13


def test_s6_scissor_kick_is_eq5():
    """S6: with beta = Psi(0) and D_p = D the half-kick is PAPER.md Eq. (5), psi + delta Psi(0) Psi^H(0) psi with
    delta = -i dt/2 D dv, followed by the per-orbital renormalisation of reading D27 (plain numpy matrices)."""
    grid, h, dt, D = (5, 6, 5), (0.5, 0.4, 0.45), 0.05, 0.35
    ngrid, dv = int(np.prod(grid)), float(np.prod(h))
    x = rand_c(ngrid, 4)
    delta = -0.5j * dt * D * dv
    y = x
    for _ in range(2):                                        # kick_only: the two half-kicks of one step
        z = y + delta * (x @ (x.conj().T @ y))
        y = z * (np.linalg.norm(y, axis=0) / np.linalg.norm(z, axis=0))[None, :]
    out, _ = ref.propagate_split(x.reshape(1, *grid, 4), np.full((1, 4), 2.0), np.zeros((1, *grid)), x.reshape(1, ngrid, 4),
                                 np.full((1, 4), D), np.zeros((1, 1, 3)), dt, h, kick_only=True)
    assert rel(out[0].reshape(ngrid, 4), y) < 1e-13
