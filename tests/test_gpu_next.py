"""GPU parity of the SURVEY.md 8(f) rows finished in round 2, against the FP64 oracle on the same seeded inputs and
through the C ABI:
  NEXT-2  mlmd_current_nl: the nonlocal (pseudopotential) part of the current, the term PAPER.md L201 says is
          GEMMified (three more projection GEMMs against caller-supplied (r - R_p)_d beta_p arrays; reading D31);
  NEXT-3  MLMD_OPT_FD_ORDER = 2: the paper's own 2nd-order / 7-point local discretisation in
          mlmd_propagate, mlmd_propagate_split and mlmd_current (radius-1 instantiation of the TMA stencil kernel).
Tolerances: the FP32-grade bars of north_star for the steps; for the current the scale of test_gpu_observables.py
(the nonlocal part is a sum of products of two projection coefficients: relative 1e-5 of the same sum taken with
absolute values, i.e. without cancellation).
"""
import numpy as np
import pytest

import workloads as W
from test_gpu_parity import TOL_1STEP, TOL_LAST, TOL_RHO, make_domain, orb_err, rho_err

pytestmark = pytest.mark.gpu


def position_weights(c, rng, nproj):
    """(r - R_p)_d on the grid for a random centre R_p per projector, minimum image: [3, ngrid, nproj]."""
    ax = [np.arange(n) * s for n, s in zip(c.grid, c.h)]
    X = np.stack(np.meshgrid(*ax, indexing="ij"), axis=0).reshape(3, -1)          # [3, ngrid]
    R = rng.uniform(0, 1, (3, nproj)) * np.array(c.box)[:, None]
    d = X[:, :, None] - R[:, None, :]
    L = np.array(c.box)[:, None, None]
    return d - L * np.round(d / L)


def nl_scale(psi, occ, beta, rbeta, D, dv):
    """sum_n f_n sum_p |D_p| |G_dpn| |C_pn| * 2 dv^2: the sum of current_nl without cancellation (FP64, numpy)."""
    ndom = psi.shape[0]
    out = np.zeros((ndom, 3))
    for k in range(ndom):
        x = psi[k].reshape(-1, psi.shape[-1]).astype(np.complex128)
        C = beta[k].astype(np.complex128).conj().T @ x
        for d in range(3):
            G = rbeta[d, k].astype(np.complex128).conj().T @ x
            out[k, d] = 2 * dv * dv * (np.abs(D[k])[:, None] * np.abs(G) * np.abs(C) * occ[k][None, :]).sum()
    return out


@pytest.mark.parametrize("cfg,ndom,cplx", [(1, 1, False), (0, 2, True), (2, 1, False)])
def test_nonlocal_current_against_the_oracle(cfg, ndom, cplx):
    """configs[1] (tensor-core projection, 32 projectors), configs[0] with complex projectors and two domains, and one
    PbTiO3-shaped configs[2] domain (240 projectors, 224 orbitals: the hot-path GEMM shape); the state is the GPU's own
    after two steps in the field, read back and handed to the oracle."""
    from oracle import ref
    c = W.get_config(cfg, ndom=ndom, nsteps=2)
    d = W.generate(c)
    rng = np.random.default_rng(31 + cfg)
    beta = d["beta"]
    if cplx:
        beta = (beta * np.exp(1j * rng.uniform(0, 6.28, (c.ndom, 1, c.nproj)))).astype(np.complex64)
        d = dict(d, beta=beta)
    w = position_weights(c, rng, c.nproj)
    rbeta = np.ascontiguousarray((w[:, None] * beta[None]).astype(beta.dtype))        # [3, ndom, ngrid, nproj]
    A = W.laser_samples(W.get_config(1), nsteps=2, t0=0.9) * 5.0
    dom = make_domain(c, d)
    dom.propagate(2, c.dt, A)
    psi = dom.get_orbitals()
    J = dom.current_nl(rbeta)
    J_ref = ref.current_nl(psi, d["occ"], beta, rbeta, d["D"], c.dv)
    scale = nl_scale(psi, d["occ"], beta, rbeta, d["D"], c.dv)
    print("J_nl", J, J_ref, "scaled err", np.abs(J - J_ref) / scale)
    assert (np.abs(J - J_ref) <= 1e-5 * scale).all()
    # device-resident rbeta and J give the same numbers; the step after it is unaffected by the scratch it used
    import torch
    Jd = torch.empty((c.ndom, 3), dtype=torch.float64, device="cuda")
    import paper_2509_00966_b200 as M
    M.mlmd_current_nl(dom.handle, torch.from_numpy(rbeta).cuda(), Jd)
    assert np.array_equal(Jd.cpu().numpy(), J)
    dom.propagate(1, c.dt, A[:1])
    other = make_domain(c, d)
    other.propagate(2, c.dt, A)
    other.propagate(1, c.dt, A[:1])
    assert np.array_equal(dom.get_orbitals(), other.get_orbitals())
    dom.close()
    other.close()


def test_nonlocal_current_without_projectors_is_zero():
    c = W.get_config(0)
    d = W.generate(c)
    dom = make_domain(c, dict(d, beta=None, D=None))
    assert np.array_equal(dom.current_nl(None), np.zeros((1, 3)))
    dom.close()


@pytest.mark.parametrize("stencil", [0, 1, 2])
def test_second_order_stencil_config1(stencil):
    """MLMD_OPT_FD_ORDER = 2 on configs[1] (laser on, projectors on), 10 steps: every stencil kernel variant (TMA
    radius-1 instantiation, register marching, one thread per output) against the oracle's ORDER2 flag."""
    import paper_2509_00966_b200 as M
    from oracle import ref
    c = W.get_config(1, nsteps=10)
    d = W.generate(c)
    A = W.laser_samples(c, nsteps=10, t0=0.9)
    dom = make_domain(c, d, options=[(M.OPT_FD_ORDER, 2), (M.OPT_STENCIL, stencil)])
    dom.propagate(1, c.dt, A[:1])
    r1, _ = ref.propagate(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], A[:1], c.dt, c.h, flags=ref.ORDER2)
    assert orb_err(dom.get_orbitals(), r1) <= TOL_1STEP
    dom.set_orbitals(d["psi"], d["occ"])
    dom.propagate(10, c.dt, A)
    r, rho_ref = ref.propagate(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], A, c.dt, c.h, flags=ref.ORDER2)
    e, er = orb_err(dom.get_orbitals(), r), rho_err(dom.density(), rho_ref)
    print("order 2, stencil variant", stencil, e, er)
    assert e <= TOL_LAST and er <= TOL_RHO
    # it is not the 4th-order result
    r4, _ = ref.propagate(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], A, c.dt, c.h)
    assert orb_err(dom.get_orbitals(), r4) > 1e-2
    # the local current follows the option
    J = dom.current(A[9])
    J_ref = ref.current(r, d["occ"], A[9], c.h, flags=ref.ORDER2)
    ne = float(d["occ"].sum())
    assert np.abs(J - J_ref).max() <= 1e-5 * ne / min(c.h)
    dom.close()


def test_second_order_stencil_plane_waves_and_field_components():
    """Closed form on the GPU itself: e^{ik.r} is multiplied by P4(-i dt eps)^n with the 2nd-order symbol
    eps = sum_d [(1 - cos p_d)/h_d^2 + A_d sin(p_d)/h_d] + |A|^2/2; anisotropic grid, A with y and z components."""
    import paper_2509_00966_b200 as M
    grid, h, dt, nsteps = (10, 16, 32), (0.5, 0.45, 0.4), 0.02, 5
    A = np.array([0.07, -0.04, 0.11])
    box = [n * s for n, s in zip(grid, h)]
    ax = [np.arange(n) * s for n, s in zip(grid, h)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    ms = [(0, 0, 0), (1, 0, 0), (0, -2, 0), (0, 0, 3), (2, -1, 4), (-3, 3, -7), (3, 4, 7), (3, 3, 3)]
    psi = np.zeros((1, *grid, len(ms)), dtype=np.complex128)
    eps = []
    for n, m in enumerate(ms):
        k = [2 * np.pi * mi / b for mi, b in zip(m, box)]
        psi[0, ..., n] = np.exp(1j * (k[0] * X + k[1] * Y + k[2] * Z))
        eps.append(sum((1 - np.cos(k[d] * h[d])) / h[d] ** 2 + A[d] * np.sin(k[d] * h[d]) / h[d] for d in range(3)) + 0.5 * A @ A)
    psi32 = psi.astype(np.complex64)
    dom = M.Domain(1, grid, h, len(ms), 0)
    dom.set_option(M.OPT_FD_ORDER, 2)
    dom.set_vloc(np.zeros((1, *grid), dtype=np.float32))
    dom.set_orbitals(psi32, np.ones((1, len(ms))))
    dom.propagate(nsteps, dt, np.tile(A, (nsteps, 1, 1)))
    out = dom.get_orbitals().astype(np.complex128)
    z = lambda e: 1 + (-1j * dt * e) + (-1j * dt * e) ** 2 / 2 + (-1j * dt * e) ** 3 / 6 + (-1j * dt * e) ** 4 / 24
    for n, e in enumerate(eps):
        expect = z(e) ** nsteps * psi32[0, ..., n].astype(np.complex128)
        assert np.linalg.norm(out[0, ..., n] - expect) / np.linalg.norm(expect) < 1e-5
    with pytest.raises(M.MlmdError):
        dom.set_option(M.OPT_FD_ORDER, 3)
    dom.close()


def test_second_order_stencil_perovskite_domain_and_split_step():
    """One configs[2] domain (48^3: the TMA kernel's radius-1 instantiation with the tcgen05 GEMMs), Taylor and the
    literal Eq. (2) split step (through its nproj = 0 limit, where it is the Taylor step, and with projectors against the
    oracle's order switch)."""
    import paper_2509_00966_b200 as M
    from oracle import ref
    c = W.get_config(2, ndom=1, nsteps=3)
    d = W.generate(c)
    A = W.laser_samples(c, nsteps=3, t0=0.9)
    dom = make_domain(c, d, options=[(M.OPT_FD_ORDER, 2)])
    assert dom.gemm_path() == "tcgen05"
    dom.propagate(3, c.dt, A)
    r, rho_ref = ref.propagate(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], A, c.dt, c.h, flags=ref.ORDER2)
    e, er = orb_err(dom.get_orbitals(), r), rho_err(dom.density(), rho_ref)
    print("order 2 perovskite", e, er)
    assert e <= TOL_LAST and er <= TOL_RHO
    dom.close()
    nop = make_domain(c, dict(d, beta=None, D=None), options=[(M.OPT_FD_ORDER, 2)])
    nop.propagate_split(3, c.dt, A)
    r0, _ = ref.propagate(d["psi"], d["occ"], d["vloc"], None, None, A, c.dt, c.h, flags=ref.ORDER2)
    assert orb_err(nop.get_orbitals(), r0) <= TOL_LAST
    nop.close()
    # the Eq. (2) step with projectors on the 7-point operator against the oracle's own order switch (pin O2f)
    sp = make_domain(c, d, options=[(M.OPT_FD_ORDER, 2)])
    sp.propagate_split(3, c.dt, A)
    rs, rho_s = ref.propagate_split(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], A, c.dt, c.h, order=2)
    assert orb_err(sp.get_orbitals(), rs) <= TOL_LAST and rho_err(sp.density(), rho_s) <= TOL_RHO
    sp.close()
