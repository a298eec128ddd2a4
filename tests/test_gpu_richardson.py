"""GPU parity of the paper's own local solver inside the Eq. (2) step (MLMD_OPT_LOCAL_SOLVER = 1: block-diagonal
split-operator on 2nd-order differences, PAPER.md L147 / L283; reading D33) against the
FP64 oracle's mlmd_ref_propagate_split(local="richardson") on the same seeded inputs, through the C ABI.
Tolerances are the hot path's (BASELINE.json north_star): per-orbital rel L2 <= 1e-5 after one step, <= 1e-4 after the
last, density <= 1e-4, Gram <= 1e-5.
"""
import numpy as np
import pytest

import workloads as W
from test_gpu_parity import TOL_1STEP, TOL_LAST, TOL_RHO, TOL_GRAM, make_domain, orb_err, rho_err

pytestmark = pytest.mark.gpu


def run(c, d, nsteps, A=None, graph=None):
    import paper_2509_00966_b200 as M
    from oracle import ref
    A = d["A"] if A is None else A
    dom = make_domain(c, d)
    dom.set_option(M.OPT_LOCAL_SOLVER, 1)
    if graph is not None:
        dom.set_option(M.OPT_GRAPH, graph)
    dom.propagate_split(1, c.dt, A[:1])
    r1, _ = ref.propagate_split(d["psi"], d["occ"], d["vloc"], d.get("beta"), d.get("D"), A[:1], c.dt, c.h, local="richardson")
    out = {"err1": orb_err(dom.get_orbitals(), r1)}
    dom.set_orbitals(d["psi"], d["occ"])
    dom.propagate_split(nsteps, c.dt, A[:nsteps])
    g, rho, G = dom.get_orbitals(), dom.density(), dom.overlap(0)
    r, rho_ref = ref.propagate_split(d["psi"], d["occ"], d["vloc"], d.get("beta"), d.get("D"), A[:nsteps], c.dt, c.h,
                                     local="richardson")
    out.update(err=orb_err(g, r), rho=rho_err(rho, rho_ref), gram=float(np.abs(G - ref.overlap(r, r, c.dv)).max()))
    dom.close()
    print(out)
    assert out["err1"] <= TOL_1STEP and out["err"] <= TOL_LAST and out["rho"] <= TOL_RHO and out["gram"] <= TOL_GRAM
    return g


def test_richardson_config0_graph_and_eager_agree():
    """configs[0] (launch-bound: the 10-step call replays a CUDA graph of the step): parity, and the replayed steps are
    bit-identical to eager launches."""
    c = W.get_config(0)
    d = W.generate(c)
    a = run(c, d, c.nsteps)
    b = run(c, d, c.nsteps, graph=0)
    assert np.array_equal(a, b)


def test_richardson_config1_laser_100_steps():
    c = W.get_config(1)
    run(c, W.generate(c), c.nsteps)


def test_richardson_one_perovskite_domain():
    """One configs[2]-shaped domain (48^3 x 224 orbitals x 240 projectors): the tensor-core kicks around the local solver."""
    c = W.get_config(2, ndom=1, nsteps=3)
    d = W.generate(c)
    run(c, d, 3, A=W.laser_samples(c, nsteps=3, t0=0.9))


@pytest.mark.parametrize("grid,norb,cplx", [((6, 8, 10), 3, True), ((8, 16, 8), 5, False), ((16, 6, 32), 12, True)])
def test_richardson_anisotropic_grids_complex_projectors_per_domain_field(grid, norb, cplx):
    import paper_2509_00966_b200 as M
    from oracle import ref
    rng = np.random.default_rng(11 + norb)
    ndom, nproj, h, dt, nsteps = 3, 4, (0.5, 0.45, 0.4), 0.02, 3
    ngrid = int(np.prod(grid))
    psi = (rng.standard_normal((ndom, *grid, norb)) + 1j * rng.standard_normal((ndom, *grid, norb))).astype(np.complex64)
    psi /= np.sqrt((np.abs(psi) ** 2).sum(axis=(1, 2, 3), keepdims=True) * np.prod(h))
    occ = rng.uniform(0, 2, (ndom, norb))
    vloc = rng.uniform(-1, 0.5, (ndom, *grid)).astype(np.float32)
    beta = rng.standard_normal((ndom, ngrid, nproj)) + (1j * rng.standard_normal((ndom, ngrid, nproj)) if cplx else 0)
    beta = (beta * 0.5).astype(np.complex64 if cplx else np.float32)
    D = rng.uniform(-2, 2, (ndom, nproj))
    A = rng.uniform(-0.2, 0.2, (nsteps, ndom, 3))
    dom = M.Domain(ndom, grid, h, norb, nproj * (2 if cplx else 1))
    dom.set_option(M.OPT_LOCAL_SOLVER, 1)
    dom.set_vloc(vloc)
    dom.set_orbitals(psi, occ)
    dom.set_projectors(beta, D)
    dom.propagate_split(nsteps, dt, A)
    r, rho_ref = ref.propagate_split(psi, occ, vloc, beta, D, A, dt, h, local="richardson")
    assert orb_err(dom.get_orbitals(), r) <= TOL_LAST
    assert rho_err(dom.density(), rho_ref) <= TOL_RHO
    dom.close()


def test_richardson_is_unitary_for_a_time_step_the_taylor_sum_cannot_take():
    """No projectors, dt = 0.5 (dt |h_loc| ~ 15: Taylor-4 is unstable beyond 2.83): the Gram matrix of white-noise orbitals
    stays where it was through 20 steps, and the result still follows the oracle."""
    import paper_2509_00966_b200 as M
    from oracle import ref
    c = W.get_config(0)
    d = W.generate(c)
    d = dict(d, beta=None, D=None)
    dom = make_domain(c, d)
    dom.set_option(M.OPT_LOCAL_SOLVER, 1)
    g0 = dom.overlap(0).copy()
    A = np.zeros((20, 1, 3))
    A[:, 0, 0] = 0.1
    assert dom.propagate_split(20, 0.5, A) == M.OK          # no stability warning: the solver has no bound
    assert np.abs(dom.overlap(0) - g0).max() <= 1e-5
    r, _ = ref.propagate_split(d["psi"], d["occ"], d["vloc"], None, None, A, 0.5, c.h, local="richardson")
    assert orb_err(dom.get_orbitals(), r) <= TOL_LAST
    dom.close()


def test_richardson_rejects_an_odd_axis_and_leaves_the_taylor_path_alone():
    import paper_2509_00966_b200 as M
    rng = np.random.default_rng(3)
    grid, h, norb = (6, 5, 8), (0.5, 0.5, 0.5), 2
    psi = (rng.standard_normal((1, *grid, norb)) + 1j * rng.standard_normal((1, *grid, norb))).astype(np.complex64)
    dom = M.Domain(1, grid, h, norb, 0)
    dom.set_vloc(np.zeros((1, *grid), dtype=np.float32))
    dom.set_orbitals(psi, np.full((1, norb), 2.0))
    dom.set_projectors(None, None)
    dom.set_option(M.OPT_LOCAL_SOLVER, 1)
    with pytest.raises(M.MlmdError) as e:
        dom.propagate_split(1, 0.02, np.zeros((1, 1, 3)))
    assert e.value.code == M.api.ERR_SHAPE
    assert dom.propagate(1, 0.02, np.zeros((1, 1, 3))) == M.OK      # mlmd_propagate ignores the option
    dom.set_option(M.OPT_LOCAL_SOLVER, 0)
    assert dom.propagate_split(1, 0.02, np.zeros((1, 1, 3))) == M.OK
    dom.close()


@pytest.mark.parametrize("kick_norm,lowp", [(1, False), (0, True)])
def test_richardson_other_norm_path_and_low_precision_mode(kick_norm, lowp):
    """MLMD_OPT_KICK_NORM = 1 (every norm by a pass over psi: the path shapes without a usable projector Gram matrix take) and
    the opt-in low-precision GEMM mode (1e-3) around the same local solver,
    on one configs[2] domain (tcgen05 kicks); the occupations afterwards follow the oracle's overlap."""
    import paper_2509_00966_b200 as M
    from oracle import ref
    from test_gpu_parity import TOL_LOWP
    c = W.get_config(2, ndom=1, nsteps=3)
    d = W.generate(c)
    A = W.laser_samples(c, nsteps=3, t0=0.9)
    dom = make_domain(c, d, flags=M.KEEP_PSI0, mode=M.GEMM_LOWP_BF16 if lowp else None)
    dom.set_option(M.OPT_LOCAL_SOLVER, 1)
    dom.set_option(M.OPT_KICK_NORM, kick_norm)
    dom.propagate_split(3, c.dt, A)
    r, rho_ref = ref.propagate_split(d["psi"], d["occ"], d["vloc"], d["beta"], d["D"], A, c.dt, c.h, local="richardson")
    tol_psi, tol_rho = (TOL_LOWP, TOL_LOWP) if lowp else (TOL_LAST, TOL_RHO)
    assert orb_err(dom.get_orbitals(), r) <= tol_psi
    assert rho_err(dom.density(), rho_ref) <= tol_rho
    f, nexc = dom.occupations()
    f_ref, _ = ref.occupations(ref.overlap(d["psi"], r, c.dv), d["occ"])
    assert np.abs(f - f_ref).max() <= (1e-3 if lowp else 1e-5) * d["occ"].max()
    dom.close()
