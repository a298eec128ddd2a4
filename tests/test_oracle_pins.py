"""Pins of the FP64 oracle (oracle/mlmd_ref.c) against what the paper and the mathematics fix.

The paper prints no value of psi, rho or any overlap, so every pin is mathematical
(DESIGN.md "Pins").  Nothing here re-calls the oracle to check the
oracle: each expected value is built by an independent route (closed form, dense matrices from
Kronecker products or hand loops, scipy's expm/eigh, Taylor-matching conditions, identities).
All tests are CPU-only.
"""
import math

import numpy as np
import pytest
import scipy.linalg

import workloads as W
from oracle import ref

RNG = np.random.default_rng(20250966)


# ----------------------------------------------------------------------------------------
# independent building blocks
def fd_weights(order_of_derivative: int) -> np.ndarray:
    """5-point central-difference weights from their DEFINITION (Taylor matching):
    sum_j w_j j^m = m! * delta(m, order) for m = 0..4.  Not typed in; solved."""
    j = np.arange(-2, 3, dtype=np.float64)
    V = np.vander(j, 5, increasing=True).T           # V[m, j] = j^m
    rhs = np.zeros(5)
    rhs[order_of_derivative] = math.factorial(order_of_derivative)
    return np.linalg.solve(V, rhs)


def circulant_derivative(n: int, h: float, order: int) -> np.ndarray:
    w = fd_weights(order) / h ** order
    M = np.zeros((n, n))
    for i in range(n):
        for jj, wj in zip(range(-2, 3), w):
            M[i, (i + jj) % n] += wj
    return M


def dense_h(grid, h, vloc, beta, D, A):
    """H as a dense matrix over r=(ix*ny+iy)*nz+iz, built from Kronecker products."""
    nx, ny, nz = grid
    I = [np.eye(n) for n in grid]
    H = np.zeros((nx * ny * nz,) * 2, dtype=np.complex128)
    for d in range(3):
        parts2 = [I[0], I[1], I[2]]
        parts1 = [I[0], I[1], I[2]]
        parts2[d] = circulant_derivative(grid[d], h[d], 2)
        parts1[d] = circulant_derivative(grid[d], h[d], 1)
        H += -0.5 * np.kron(np.kron(parts2[0], parts2[1]), parts2[2])
        H += -1j * A[d] * np.kron(np.kron(parts1[0], parts1[1]), parts1[2])
    H += np.diag(vloc.reshape(-1).astype(np.float64) + 0.5 * float(np.dot(A, A)))
    if beta is not None:
        B = beta.astype(np.complex128)
        dv = h[0] * h[1] * h[2]
        H += dv * (B * np.asarray(D, dtype=np.float64)[None, :]) @ B.conj().T
    return H


def p4(z):
    return 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24


def rand_c(*shape):
    return RNG.standard_normal(shape) + 1j * RNG.standard_normal(shape)


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(np.asarray(b).ravel())


@pytest.fixture(scope="module")
def cfg0():
    c = W.get_config(0)
    d = W.generate(c)
    return c, d


@pytest.fixture(scope="module")
def cfg0_dense(cfg0):
    c, d = cfg0
    A = np.array([0.05, -0.03, 0.02])
    H = dense_h(c.grid, c.h, d["vloc"][0], d["beta"][0], d["D"][0], A)
    lam, V = np.linalg.eigh(H)
    return A, H, lam, V


# ----------------------------------------------------------------------------------------
def test_weights_are_the_textbook_ones():
    """Sanity of the independent derivation itself (textbook 4th-order central differences)."""
    assert np.allclose(fd_weights(2), [-1 / 12, 4 / 3, -5 / 2, 4 / 3, -1 / 12], atol=1e-14)
    assert np.allclose(fd_weights(1), [1 / 12, -2 / 3, 0, 2 / 3, -1 / 12], atol=1e-14)


@pytest.mark.parametrize("A", [(0.0, 0.0, 0.0), (0.1, 0.0, 0.0), (0.07, -0.04, 0.11)])
def test_p1_plane_wave_closed_form(A):
    """P1: V=0, no projectors: e^{ik.r} is an eigenvector with symbol eps(k,A) (reading D5), so
    n steps multiply it by P4(-i dt eps)^n exactly (BASELINE.json north_star, first pin)."""
    grid, h, dt, nsteps = (12, 10, 16), (0.5, 0.45, 0.4), 0.02, 7
    box = [n * s for n, s in zip(grid, h)]
    ax = [np.arange(n) * s for n, s in zip(grid, h)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    ms = [(0, 0, 0), (1, 0, 0), (0, -2, 0), (0, 0, 3), (2, -1, 4), (-5, 3, -7), (6, 5, 8)]
    psi = np.zeros((1, *grid, len(ms)), dtype=np.complex128)
    eps = []
    lam2 = lambda p: 2.5 - (8.0 / 3.0) * np.cos(p) + (1.0 / 6.0) * np.cos(2 * p)
    lam1 = lambda p: (4.0 / 3.0) * np.sin(p) - (1.0 / 6.0) * np.sin(2 * p)
    for n, m in enumerate(ms):
        k = [2 * np.pi * mi / L for mi, L in zip(m, box)]
        psi[0, ..., n] = np.exp(1j * (k[0] * X + k[1] * Y + k[2] * Z))
        e = 0.5 * np.dot(A, A)
        for d in range(3):
            ph = k[d] * h[d]
            e += 0.5 * lam2(ph) / h[d] ** 2 + A[d] * lam1(ph) / h[d]
        eps.append(e)
    Aarr = np.tile(np.array(A, dtype=np.float64), (nsteps, 1, 1))
    out, rho = ref.propagate(psi, np.ones((1, len(ms))), np.zeros((1, *grid)), None, None, Aarr, dt, h)
    for n, e in enumerate(eps):
        expect = p4(-1j * dt * e) ** nsteps * psi[0, ..., n]
        assert rel(out[0, ..., n], expect) < 1e-13
    # P8 corollary: the density of plane waves is uniform
    assert np.ptp(rho) < 1e-12 * rho.mean()


def test_p12_polynomial_exactness():
    """Definition of '4th-order central differences' (north_star): the 5-point D1 is exact on
    polynomials up to degree 4 and D2 up to degree 5.  Away from the periodic seam
    H p = -1/2 p'' - i A p' + 1/2 A^2 p must hold to rounding, separately along each axis."""
    n, h = 16, 0.37
    x = (np.arange(n) - n / 2) * h
    coef = [0.3, -1.1, 0.7, 0.45, -0.25]                       # degree 4
    pol = np.polynomial.Polynomial(coef)
    for axis in range(3):
        A = np.zeros(3)
        A[axis] = 0.23
        shape = [1, 1, 1]
        shape[axis] = n
        u = np.broadcast_to(pol(x).reshape(shape), (n, n, n)).astype(np.complex128)[..., None]
        out = ref.apply_h(u, np.zeros((n, n, n)), None, None, A, (h, h, h))
        expect = -0.5 * pol.deriv(2)(x) - 1j * A[axis] * pol.deriv(1)(x) + 0.5 * A[axis] ** 2 * pol(x)
        sl = [0, 0, 0, 0]
        sl[axis] = slice(2, n - 2)
        assert np.allclose(out[tuple(sl)], expect[2:n - 2], rtol=0, atol=1e-11)
    # degree 5 is still exact for D2 (A = 0)
    pol5 = np.polynomial.Polynomial(coef + [0.15])
    u = np.broadcast_to(pol5(x).reshape(n, 1, 1), (n, n, n)).astype(np.complex128)[..., None]
    out = ref.apply_h(u, np.zeros((n, n, n)), None, None, np.zeros(3), (h, h, h))
    assert np.allclose(out[2:n - 2, 0, 0, 0], -0.5 * pol5.deriv(2)(x)[2:n - 2], atol=1e-10)


def test_p13_fourth_order_convergence_to_continuum():
    """h -> 0: H e^{ikx} -> 1/2 |k+A|^2 e^{ikx} (Eq. 3) with error ratio 2^4."""
    L, kx, A = 6.0, 2 * np.pi * 2 / 6.0, np.array([0.3, 0.0, 0.0])
    exact = 0.5 * (kx + A[0]) ** 2
    errs = []
    for n in (16, 32, 64):
        h = L / n
        x = np.arange(n) * h
        u = np.broadcast_to(np.exp(1j * kx * x).reshape(n, 1, 1), (n, 5, 5)).astype(np.complex128)[..., None]
        out = ref.apply_h(u, np.zeros((n, 5, 5)), None, None, A, (h, 0.5, 0.5))
        ratio = out[..., 0] / u[..., 0]
        assert np.ptp(ratio.real) < 1e-10 and np.abs(ratio.imag).max() < 1e-10
        errs.append(abs(ratio.real.mean() - exact))
    assert 14.0 < errs[0] / errs[1] < 17.0 and 15.0 < errs[1] / errs[2] < 16.5


def test_p2_dense_operator(cfg0, cfg0_dense):
    """P2: applyH == H_dense u on the 16^3 grid of config 0 (projectors, V_loc and A all on)."""
    c, d = cfg0
    A, H, _, _ = cfg0_dense
    u = rand_c(*c.grid, 3)
    out = ref.apply_h(u, d["vloc"][0], d["beta"][0], d["D"][0], A, c.h)
    assert rel(out.reshape(c.ngrid, 3), H @ u.reshape(c.ngrid, 3)) < 1e-12
    assert np.abs(H - H.conj().T).max() < 1e-12                     # the independent H is Hermitian


def test_p3_dense_polynomial_and_expm(cfg0, cfg0_dense):
    """P3: one oracle step == V P4(-i dt Lambda) V^H psi; and it approximates expm(-i dt H) psi within
    the Lagrange remainder theta^5/120, the error falling ~32x when dt is halved (north_star pin 2)."""
    c, d = cfg0
    A, H, lam, V = cfg0_dense
    psi = d["psi"][0].astype(np.complex128).reshape(c.ngrid, c.norb)
    Aarr = A.reshape(1, 1, 3)

    def one_step(dt):
        out, _ = ref.propagate(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], Aarr, dt, c.h, nsteps=1)
        return out.reshape(c.ngrid, c.norb)

    dt = c.dt
    poly = V @ (p4(-1j * dt * lam)[:, None] * (V.conj().T @ psi))
    assert rel(one_step(dt), poly) < 1e-12
    exact = V @ (np.exp(-1j * dt * lam)[:, None] * (V.conj().T @ psi))
    # library cross-check of the eigen-route itself on a few columns
    E = scipy.linalg.expm(-1j * dt * H)
    assert rel(E @ psi[:, :2], exact[:, :2]) < 1e-10
    theta = dt * np.abs(lam).max()
    err = np.linalg.norm(one_step(dt) - exact, axis=0) / np.linalg.norm(exact, axis=0)
    assert err.max() <= theta ** 5 / 120
    exact_half = V @ (np.exp(-0.5j * dt * lam)[:, None] * (V.conj().T @ psi))
    err_half = np.linalg.norm(one_step(dt / 2) - exact_half, axis=0) / np.linalg.norm(exact_half, axis=0)
    ratio = err / err_half
    assert ratio.min() > 24 and ratio.max() < 40


def test_p4_hermiticity(cfg0):
    """P4: <phi|H psi> = <H phi|psi> with A != 0, V != 0, projectors on (north_star pin 3)."""
    c, d = cfg0
    A = np.array([0.08, 0.05, -0.02])
    phi, psi = rand_c(*c.grid, 4), rand_c(*c.grid, 4)
    Hpsi = ref.apply_h(psi, d["vloc"][0], d["beta"][0], d["D"][0], A, c.h)
    Hphi = ref.apply_h(phi, d["vloc"][0], d["beta"][0], d["D"][0], A, c.h)
    lhs = np.einsum("xyzn,xyzn->n", phi.conj(), Hpsi)
    rhs = np.einsum("xyzn,xyzn->n", Hphi.conj(), psi)
    assert np.abs(lhs - rhs).max() < 1e-12 * np.abs(lhs).max()


def test_p5_exact_norm_identity(cfg0):
    """P5: H Hermitian  =>  P4(-iX)^H P4(-iX) = 1 - X^6/72 + X^8/576 with X = dt H, hence
    G_new = G - <X^3 psi|X^3 psi>/72 + <X^4 psi|X^4 psi>/576 exactly (sharpens north_star's
    'norm and orthonormality drift O(dt^5)'; the diagonal is the per-orbital norm)."""
    c, d = cfg0
    A = np.array([0.1, 0.0, 0.0])
    dt = c.dt
    psi = d["psi"].astype(np.complex128)
    out, _ = ref.propagate(psi, d["occ"], d["vloc"], d["beta"], d["D"], A.reshape(1, 1, 3), dt, c.h, nsteps=1)
    x = psi[0]
    xs = []
    for m in range(4):
        x = dt * ref.apply_h(x, d["vloc"][0], d["beta"][0], d["D"][0], A, c.h)
        xs.append(x.reshape(c.ngrid, c.norb))
    gram = lambda a: c.dv * a.conj().T @ a
    G0 = gram(psi.reshape(c.ngrid, c.norb))
    expect = G0 - gram(xs[2]) / 72 + gram(xs[3]) / 576
    G1 = gram(out.reshape(c.ngrid, c.norb))
    assert np.abs(G1 - expect).max() < 1e-12
    # the defect is sixth order in dt*H: nothing larger hides in it
    assert np.abs(G1 - G0).max() < 2 * (dt * 8 / min(c.h) ** 2 * 1.2) ** 6 / 72


def test_p6_rank1_projector_closed_form():
    """P6: kinetic term off, V=0, one normalised beta with strength d:
    H = d |beta><beta| is d times a projector, so psi_new = psi + (P4(-i d dt) - 1) beta <beta|psi>."""
    grid, h, dt, dstr = (8, 6, 10), (0.4, 0.5, 0.3), 0.05, -0.8
    dv = h[0] * h[1] * h[2]
    ngrid = grid[0] * grid[1] * grid[2]
    b = rand_c(ngrid, 1)
    b /= np.sqrt(dv * np.vdot(b, b).real)
    psi = rand_c(1, *grid, 3)
    out, _ = ref.propagate(psi, np.ones((1, 3)), np.zeros((1, *grid)), b[None], np.array([[dstr]]),
                           np.zeros((1, 1, 3)), dt, h, flags=ref.NO_KINETIC)
    flat = psi.reshape(ngrid, 3)
    expect = flat + (p4(-1j * dstr * dt) - 1) * b @ (dv * b.conj().T @ flat)
    assert rel(out.reshape(ngrid, 3), expect) < 1e-13


def test_p7_eq5_special_case():
    """P7: PAPER.md Eq. (5) (L199) is the case beta = Psi(0) (orthonormal, complex), D = const:
    V_NL Psi(0) = delta0 Psi(0).  Exercises complex projectors."""
    c = W.get_config(0)
    d = W.generate_domain(c, 0)
    psi0 = d["psi"].astype(np.complex128)
    delta0 = 0.37
    out = ref.apply_h(psi0, np.zeros(c.grid), psi0.reshape(c.ngrid, c.norb), np.full(c.norb, delta0),
                      np.zeros(3), c.h, flags=ref.NO_KINETIC)
    # complex64-rounded orbitals are orthonormal to ~1e-7 only; compare with the Gram-corrected form
    flat = psi0.reshape(c.ngrid, c.norb)
    G = c.dv * flat.conj().T @ flat
    assert rel(out.reshape(c.ngrid, c.norb), delta0 * flat @ G) < 1e-13
    assert rel(out, delta0 * psi0) < 1e-6


def test_p8_density_sum_rule(cfg0):
    """P8: dv * sum_r rho = sum_n f_n ||psi_n||^2 and rho >= 0."""
    c, d = cfg0
    psi = rand_c(2, *c.grid, 5)
    occ = np.array([[2.0, 1.5, 0.0, 0.25, 1.0], [0.0, 2.0, 2.0, 0.5, 0.1]])
    rho = ref.density(psi, occ)
    norms = c.dv * np.einsum("dxyzn,dxyzn->dn", psi.conj(), psi).real
    assert np.allclose(c.dv * rho.sum(axis=(1, 2, 3)), (occ * norms).sum(axis=1), rtol=1e-13)
    assert rho.min() >= 0.0
    r = (3, 7, 11)
    assert np.isclose(rho[1][r], np.sum(occ[1] * np.abs(psi[1][r]) ** 2), rtol=1e-13)


def test_overlap_matches_definition():
    """S = dv Phi^H Psi ('overlap matrix between KS orbitals at time t and 0')."""
    grid, dv = (5, 6, 7), 0.123
    phi, psi = rand_c(2, *grid, 4), rand_c(2, *grid, 4)
    S = ref.overlap(phi, psi, dv)
    for dom in range(2):
        a, b = phi[dom].reshape(-1, 4), psi[dom].reshape(-1, 4)
        assert np.allclose(S[dom], dv * a.conj().T @ b, rtol=1e-13, atol=1e-13)


def test_p9_batch_independence():
    """P9: a batch of domains == the same domains run one by one, bitwise."""
    c = W.get_config(0, ndom=3, nsteps=3)
    d = W.generate(c)
    A = np.tile(np.array([0.05, 0.0, -0.02]), (3, 3, 1)) * np.arange(1, 4)[None, :, None]   # per-domain A (D8)
    both, rho = ref.propagate(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], A, c.dt, c.h)
    for dom in range(3):
        one, rho1 = ref.propagate(d["psi"][dom:dom + 1], d["occ"][dom:dom + 1], d["vloc"][dom:dom + 1],
                                  d["beta"][dom:dom + 1], d["D"][dom:dom + 1], A[:, dom:dom + 1], c.dt, c.h)
        assert np.array_equal(one[0], both[dom]) and np.array_equal(rho1[0], rho[dom])
    assert not np.array_equal(both[0], both[1])


def test_p10_horner_equals_term_sum(cfg0):
    """P10: the GPU's Horner form is the same polynomial (licenses S2 of SURVEY.md section 8(a))."""
    c, d = cfg0
    A = W.laser_samples(W.get_config(1), nsteps=5, t0=0.6)
    a, _ = ref.propagate(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], A, c.dt, c.h)
    b, _ = ref.propagate(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], A, c.dt, c.h, flags=ref.HORNER)
    assert rel(a, b) < 1e-14


def test_p11_brute_force_anisotropic():
    """P11: 6x5x7 grid, hx != hy != hz, 2 orbitals, 1 complex projector: dense 210x210 H from
    hand-rolled loops (index order (ix*ny+iy)*nz+iz), step by dense matrix powers."""
    grid, h, dt = (6, 5, 7), (0.31, 0.47, 0.39), 0.015
    nx, ny, nz = grid
    n = nx * ny * nz
    dv = h[0] * h[1] * h[2]
    A = np.array([0.09, -0.06, 0.04])
    vloc = RNG.standard_normal(grid)
    b = rand_c(n, 1)
    b /= np.sqrt(dv * np.vdot(b, b).real)
    dstr = 0.6
    w2, w1 = fd_weights(2), fd_weights(1)
    H = np.zeros((n, n), dtype=np.complex128)
    for ix in range(nx):
        for iy in range(ny):
            for iz in range(nz):
                r = (ix * ny + iy) * nz + iz
                H[r, r] += vloc[ix, iy, iz] + 0.5 * A @ A
                for jj in range(-2, 3):
                    for d, (qx, qy, qz) in enumerate((((ix + jj) % nx, iy, iz), (ix, (iy + jj) % ny, iz),
                                                      (ix, iy, (iz + jj) % nz))):
                        rr = (qx * ny + qy) * nz + qz
                        H[r, rr] += -0.5 * w2[jj + 2] / h[d] ** 2 - 1j * A[d] * w1[jj + 2] / h[d]
    H += dv * dstr * b @ b.conj().T
    psi = rand_c(1, *grid, 2)
    out, _ = ref.propagate(psi, np.ones((1, 2)), vloc[None], b[None], np.array([[dstr]]),
                           np.tile(A, (2, 1, 1)), dt, h)
    X = -1j * dt * H
    U = np.eye(n) + X + X @ X / 2 + X @ X @ X / 6 + X @ X @ X @ X / 24
    assert rel(out.reshape(n, 2), U @ U @ psi.reshape(n, 2)) < 1e-13


def test_laser_and_workload_shapes():
    """The generator reproduces BASELINE.json's shapes: 240 / 810 projectors, 352 / 1188 electrons,
    a pulse that peaks at 0.1 a.u. (configs[1])."""
    assert [W.get_config(i).nproj for i in range(5)] == [8, 32, 240, 240, 810]
    assert [W.get_config(i).electrons_per_domain for i in range(5)] == [16, 128, 352, 352, 1188]
    A = W.laser_samples(W.get_config(1))
    assert A.shape == (100, 1, 3) and abs(np.abs(A[:, 0, 0]).max() - 0.1) < 2e-4 and not A[:, 0, 1:].any()
    assert not W.laser_samples(W.get_config(0)).any()
    c = W.get_config(0)
    d = W.generate(c)
    flat = d["psi"][0].astype(np.complex128).reshape(c.ngrid, c.norb)
    assert np.abs(c.dv * flat.conj().T @ flat - np.eye(c.norb)).max() < 1e-6
    assert np.allclose(c.dv * (d["beta"][0].astype(np.float64) ** 2).sum(axis=0), 1.0, atol=1e-6)
