"""GPU parity of the opt-in stage-adaptive GEMM mode (MLMD_GEMM_FP32GRADE_STAGED) against the
FP64 oracle, at the FP32-grade tolerances of BASELINE.json north_star (not the low-precision 1e-3):
  per-orbital relative L2 error <= 1e-5 after 1 step, <= 1e-4 after 100 steps; density <= 1e-4; Gram <= 1e-5.
The mode keeps 3xTF32 in the outermost Horner stage of mlmd_propagate and takes one product of nearest-rounded TF32
operands in the projection / two in the back-application of the three inner stages (weights dt^4/24, dt^3/6, dt^2/2).
"""
import numpy as np
import pytest

import workloads as W
from test_gpu_parity import check, make_domain, orb_err, run_both

pytestmark = pytest.mark.gpu


def test_staged_config1_100_steps_close_to_pure_3xtf32():
    import paper_2509_00966_b200 as M
    c = W.get_config(1)
    d = W.generate(c)
    pure = run_both(c, d, c.nsteps, mode=M.GEMM_FP32GRADE)
    staged = run_both(c, d, c.nsteps, mode=M.GEMM_FP32GRADE_STAGED)
    check(pure)
    check(staged)
    # the inner-stage rounding must stay at the level of the FP32 storage error of psi itself
    assert staged["err1"] <= pure["err1"] + 2e-7
    assert staged["err"] <= pure["err"] + 5e-6


def test_staged_perovskite_domain_on_tensor_cores():
    """One configs[2] domain (48^3, 224 orbitals, 240 projectors: the tcgen05 kernels with their full tiles),
    1 and 3 steps at the pulse maximum."""
    import paper_2509_00966_b200 as M
    c = W.get_config(2, ndom=1, nsteps=3)
    d = W.generate(c)
    A = W.laser_samples(c, nsteps=3, t0=0.9)
    dom = make_domain(c, d, mode=M.GEMM_FP32GRADE_STAGED)
    assert dom.gemm_path() == "tcgen05"
    dom.close()
    res = run_both(c, d, 3, A=A, mode=M.GEMM_FP32GRADE_STAGED)
    check(res)
    assert res["err1"] <= 1e-6 and res["err"] <= 3e-6   # two orders inside the FP32-grade bar


def test_staged_only_changes_the_taylor_step():
    """Every other call behaves as mode 0: the split step, the nonlocal energy and the overlap are bit-equal."""
    import paper_2509_00966_b200 as M
    c = W.get_config(2, ndom=1, nsteps=2)
    d = W.generate(c)
    A = W.laser_samples(c, nsteps=2, t0=0.9)
    out = []
    for mode in (M.GEMM_FP32GRADE, M.GEMM_FP32GRADE_STAGED):
        dom = make_domain(c, d, mode=mode)
        dom.propagate_split(2, c.dt, A)
        out.append((dom.get_orbitals(), dom.density(), dom.energy_nl()))
        dom.close()
    for a, b in zip(*out):
        assert np.array_equal(a, b)


def test_staged_differs_from_pure_but_barely():
    """The mode is really on (results differ from mode 0) and the difference is at the FP32 rounding level."""
    import paper_2509_00966_b200 as M
    c = W.get_config(2, ndom=1, nsteps=1)
    d = W.generate(c)
    A = W.laser_samples(c, nsteps=1, t0=0.9)
    psi = []
    for mode in (M.GEMM_FP32GRADE, M.GEMM_FP32GRADE_STAGED):
        dom = make_domain(c, d, mode=mode)
        dom.propagate(1, c.dt, A)
        psi.append(dom.get_orbitals())
        dom.close()
    assert not np.array_equal(psi[0], psi[1])
    assert orb_err(psi[1], psi[0].astype(np.complex128)) <= 5e-7


@pytest.mark.parametrize("grid,norb,cplx", [((6, 5, 7), 3, True), ((16, 8, 16), 12, True), ((16, 8, 16), 40, False)])
def test_staged_ragged_and_complex_projectors(grid, norb, cplx):
    """Shapes off the tensor-core tiling run the CUDA-core FP32 GEMMs in every stage (bit-equal to mode 0); a
    tileable grid with padded orbital counts and complex projectors (2 nproj real rows) runs the staged tcgen05
    stages and meets the FP32-grade bars against the oracle; per-domain field with y / z components."""
    from oracle import ref
    import paper_2509_00966_b200 as M
    from test_gpu_parity import rho_err
    rng = np.random.default_rng(11)
    ndom, nproj, h, dt, nsteps = 2, 5, (0.41, 0.37, 0.45), 0.02, 4
    ngrid = grid[0] * grid[1] * grid[2]
    dv = h[0] * h[1] * h[2]
    psi = (rng.standard_normal((ndom, *grid, norb)) + 1j * rng.standard_normal((ndom, *grid, norb))).astype(np.complex64)
    psi /= np.sqrt(dv * ngrid)
    beta = rng.standard_normal((ndom, ngrid, nproj)) + (1j * rng.standard_normal((ndom, ngrid, nproj)) if cplx else 0)
    beta /= np.sqrt(dv * (np.abs(beta) ** 2).sum(axis=1, keepdims=True))
    beta = beta.astype(np.complex64 if cplx else np.float32)
    D = rng.uniform(-1, 1, (ndom, nproj))
    vloc = (0.3 * rng.standard_normal((ndom, *grid))).astype(np.float32)
    occ = rng.uniform(0, 2, (ndom, norb))
    A = 0.1 * rng.standard_normal((nsteps, ndom, 3))
    out = {}
    for mode in (M.GEMM_FP32GRADE, M.GEMM_FP32GRADE_STAGED):
        dom = M.Domain(ndom, grid, h, norb, nproj * (2 if cplx else 1))
        dom.set_gemm_mode(mode)
        dom.set_vloc(vloc)
        dom.set_orbitals(psi, occ)
        dom.set_projectors(beta, D)
        dom.propagate(nsteps, dt, A)
        out[mode] = (dom.get_orbitals(), dom.density(), dom.gemm_path())
        dom.close()
    g, rho, path = out[M.GEMM_FP32GRADE_STAGED]
    assert path == ("tcgen05" if ngrid % 128 == 0 else "simt")
    if path == "simt":
        assert np.array_equal(g, out[M.GEMM_FP32GRADE][0]) and np.array_equal(rho, out[M.GEMM_FP32GRADE][1])
    r, rho_ref = ref.propagate(psi, occ, vloc, beta, D, A, dt, h)
    assert orb_err(g, r) <= 1e-5
    assert rho_err(rho, rho_ref) <= 1e-4


def test_staged_cuda_graph_equals_eager_and_mode_switch_drops_the_graph():
    """Small batches replay a captured step: in the staged mode the graph holds the staged launches (same bits as the
    eager launches), and switching the mode on a live handle re-captures (results equal a fresh handle's)."""
    import paper_2509_00966_b200 as M
    c = W.get_config(1, nsteps=9)
    d = W.generate(c)
    A = d["A"][:9]
    outs = {}
    for flag in ("1", "0"):
        dom = make_domain(c, d, mode=M.GEMM_FP32GRADE_STAGED, options=[(M.OPT_GRAPH, int(flag))])
        dom.propagate(9, c.dt, A)
        outs[flag] = (dom.get_orbitals(), dom.density())
        dom.close()
    assert np.array_equal(outs["1"][0], outs["0"][0]) and np.array_equal(outs["1"][1], outs["0"][1])
    dom = make_domain(c, d, mode=M.GEMM_FP32GRADE)
    dom.propagate(9, c.dt, A)                       # captures the default-mode step
    pure = dom.get_orbitals()
    dom.set_gemm_mode(M.GEMM_FP32GRADE_STAGED)
    dom.set_orbitals(d["psi"], d["occ"])
    dom.propagate(9, c.dt, A)                       # must not replay the default-mode graph
    assert np.array_equal(dom.get_orbitals(), outs["1"][0])
    assert not np.array_equal(pure, outs["1"][0])
    dom.close()


def test_staged_density_rides_on_the_one_product_projection():
    """In the staged mode the step's first projection takes one product of rounded operands; it carries the density of the
    previous step like the default mode's three-product projection does: random occupations, one call and step by step,
    against the oracle and bit for bit against each other; the rho formed inside the projection through the test hook."""
    import ctypes
    import torch
    import paper_2509_00966_b200 as M
    from oracle import ref
    from test_gpu_parity import TOL_LAST, TOL_RHO, make_domain, orb_err, rho_err
    c = W.get_config(1, nsteps=6)
    d = W.generate(c)
    occ = np.random.default_rng(6).uniform(0, 2, d["occ"].shape)
    A = W.laser_samples(c, nsteps=6, t0=0.9)
    r, rho_ref = ref.propagate(d["psi"], occ, d["vloc"], d["beta"], d["D"], A, c.dt, c.h)
    outs = []
    for graph, chunks in ((0, [6]), (1, [6]), (0, [1, 2, 3])):
        dom = make_domain(c, dict(d, occ=occ), mode=M.GEMM_FP32GRADE_STAGED, options=[(M.OPT_GRAPH, graph)])
        done = 0
        for n in chunks:
            dom.propagate(n, c.dt, A[done:done + n])
            done += n
        outs.append((dom.get_orbitals(), dom.density()))
        dom.close()
        assert rho_err(outs[-1][1], rho_ref) <= TOL_RHO and orb_err(outs[-1][0], r) <= TOL_LAST
    for o in outs[1:]:
        assert np.array_equal(o[0], outs[0][0]) and np.array_equal(o[1], outs[0][1])
    hook = ctypes.CDLL(M.api.TEST_LIB_PATH).mlmd_debug_fused_density_np
    hook.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
    dom = make_domain(c, dict(d, occ=occ), mode=M.GEMM_FP32GRADE_STAGED)
    dom.propagate(2, c.dt, A[:2])
    rho_fused = torch.empty((c.ndom, *c.grid), dtype=torch.float32, device="cuda")
    assert hook(dom.handle, rho_fused.data_ptr(), 4) == 0
    _, rho2 = ref.propagate(d["psi"], occ, d["vloc"], d["beta"], d["D"], A[:2], c.dt, c.h)
    assert rho_err(rho_fused.cpu().numpy(), rho2) <= TOL_RHO and rho_err(dom.density(), rho2) <= TOL_RHO
    dom.close()


def test_low_precision_mode_density_rides_on_the_bf16_projection():
    """The same for MLMD_GEMM_LOWP_BF16: the BF16 projection kernel sums the density from the FP32 values it packs."""
    import ctypes
    import torch
    import paper_2509_00966_b200 as M
    from oracle import ref
    from test_gpu_parity import TOL_LOWP, make_domain, orb_err, rho_err
    c = W.get_config(1, nsteps=6)
    d = W.generate(c)
    occ = np.random.default_rng(7).uniform(0, 2, d["occ"].shape)
    A = W.laser_samples(c, nsteps=6, t0=0.9)
    r, rho_ref = ref.propagate(d["psi"], occ, d["vloc"], d["beta"], d["D"], A, c.dt, c.h)
    outs = []
    for graph, chunks in ((0, [6]), (1, [6]), (0, [1, 2, 3])):
        dom = make_domain(c, dict(d, occ=occ), mode=M.GEMM_LOWP_BF16, options=[(M.OPT_GRAPH, graph)])
        done = 0
        for n in chunks:
            dom.propagate(n, c.dt, A[done:done + n])
            done += n
        outs.append((dom.get_orbitals(), dom.density()))
        dom.close()
        assert rho_err(outs[-1][1], rho_ref) <= TOL_LOWP and orb_err(outs[-1][0], r) <= TOL_LOWP
    for o in outs[1:]:
        assert np.array_equal(o[0], outs[0][0]) and np.array_equal(o[1], outs[0][1])
    hook = ctypes.CDLL(M.api.TEST_LIB_PATH).mlmd_debug_fused_density_np
    hook.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
    dom = make_domain(c, dict(d, occ=occ), mode=M.GEMM_LOWP_BF16)
    dom.propagate(2, c.dt, A[:2])
    rho_fused = torch.empty((c.ndom, *c.grid), dtype=torch.float32, device="cuda")
    assert hook(dom.handle, rho_fused.data_ptr(), 0) == 0
    rho_pass = dom.density()
    _, rho2 = ref.propagate(d["psi"], occ, d["vloc"], d["beta"], d["D"], A[:2], c.dt, c.h)
    assert rho_err(rho_fused.cpu().numpy(), rho2) <= TOL_LOWP
    # the riding sum and the separate pass see the same FP32 state: they agree to FP32 summation order
    assert rho_err(rho_fused.cpu().numpy(), rho_pass.astype(np.float64)) <= 1e-5
    dom.close()
