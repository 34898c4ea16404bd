"""-m gpu: a warm-started sequence of pressure steps with a moving body (SURVEY.md S8(f) N1 + N4;
PAPER.md:33 "swimming jellyfish", Table 1; PAPER.md:51 predictor/corrector solves): per step
gmg_set_coeffs -> gmg_divergence -> gmg_solve (p kept from the step before) -> gmg_project,
against the same loop run with the FP64 oracle on the same FP32 inputs."""
import numpy as np
import pytest

import oracle
from paper_2607_07687_b200 import gmg
from paper_2607_07687_b200 import workloads as W
from paper_2607_07687_b200.pressure_step import PressureStepper
from gpu_util import TOL_P, dev, host, rel_l2_demeaned, rel_linf

pytestmark = pytest.mark.gpu

OSOLVER = {gmg.GMG_RBGS: oracle.GMG_RBGS, gmg.GMG_PCG: oracle.GMG_PCG, gmg.GMG_CGS: oracle.GMG_CGS}


def _oracle_steps(p_exp, nsteps, solver, tol, maxiter):
    """The same loop with the oracle; a fresh hierarchy per step = gmg_set_coeffs (omega reset)."""
    nx = 2 ** (p_exp + 1)
    n, bc = (nx, nx, nx // 2), W.JELLYFISH_BC
    p = np.zeros((n[2], n[1], n[0]))
    out = []
    for L32, u32 in W.jellyfish_steps(p_exp, nsteps):
        H = oracle.Hierarchy(n, bc, L32)
        z = oracle.divergence(u32, bc)
        r = H.solve(solver, z, p0=p, tol=tol, maxiter=maxiter)
        p = r["p"]
        u = oracle.project(L32, bc, p, u32)
        out.append(dict(iterations=r["iterations"], status=r["status"], p=p.copy(), u=u, z=z, L=L32,
                        history=r["history"]))
    return out


@pytest.mark.parametrize("solver", [gmg.GMG_RBGS, gmg.GMG_PCG, gmg.GMG_CGS])
def test_fixed_cycle_steps_match_the_oracle(solver):
    """tol = 0, two iterations per step: both sides do the same work, so the warm-started
    iterates can be compared step by step."""
    p_exp, nsteps = 4, 5
    ref = _oracle_steps(p_exp, nsteps, OSOLVER[solver], 0.0, 2)
    nx = 2 ** (p_exp + 1)
    n, bc = (nx, nx, nx // 2), W.JELLYFISH_BC
    ps = PressureStepper(n, bc, solver=solver, tol=0.0, maxiter=2)
    try:
        for k, (L32, u32) in enumerate(W.jellyfish_steps(p_exp, nsteps)):
            ud = dev(u32)
            rc, st = ps.step(dev(L32), ud)
            assert rc == gmg.NOT_CONVERGED and st["iterations"] == 2
            act = W.active_mask(L32, bc)
            assert rel_l2_demeaned(host(ps.p), ref[k]["p"], act) <= TOL_P, k
            assert rel_linf(host(ud), ref[k]["u"]) <= 1e-4, k
    finally:
        ps.close()


@pytest.mark.parametrize("solver", [gmg.GMG_RBGS, gmg.GMG_CGS])
def test_warm_started_steps_converge_in_fewer_cycles_like_the_oracle(solver):
    p_exp, nsteps = 5, 6
    ref = _oracle_steps(p_exp, nsteps, OSOLVER[solver], 1e-4, 50)
    nx = 2 ** (p_exp + 1)
    n, bc = (nx, nx, nx // 2), W.JELLYFISH_BC
    ps = PressureStepper(n, bc, solver=solver, tol=1e-4, maxiter=50)
    its = []
    try:
        for k, (L32, u32) in enumerate(W.jellyfish_steps(p_exp, nsteps)):
            ud = dev(u32)
            rc, st = ps.step(dev(L32), ud)
            assert rc == gmg.OK and ref[k]["status"] == 0
            its.append(st["iterations"])
            assert abs(st["iterations"] - ref[k]["iterations"]) <= 1, (k, its, [r["iterations"] for r in ref])
            # what is left of the divergence is the solve's residual (FP64 check of the GPU's field)
            zn = oracle.divergence(host(ud), bc)
            zref = np.linalg.norm(np.where(W.active_mask(L32, bc), ref[k]["z"], 0.0))
            assert np.linalg.norm(zn) <= 1.05e-4 * zref, k
        # the warm start pays: later steps need fewer cycles than the cold first one
        assert max(its[1:]) < its[0], its
    finally:
        ps.close()


def test_rewriting_the_coefficients_in_place_reuses_the_graph_and_changes_nothing():
    """A moving body rewrites ONE coefficient array; gmg_set_coeffs with the same pointer keeps the
    captured solve graph.  Results must equal, bit for bit, those of fresh arrays every step."""
    import torch
    p_exp, nsteps = 4, 4
    nx = 2 ** (p_exp + 1)
    n, bc = (nx, nx, nx // 2), W.JELLYFISH_BC
    a = PressureStepper(n, bc, solver=gmg.GMG_RBGS, tol=1e-4, maxiter=50)
    b = PressureStepper(n, bc, solver=gmg.GMG_RBGS, tol=1e-4, maxiter=50)
    try:
        Lcur = torch.empty((3, n[2], n[1], n[0]), dtype=torch.float32, device="cuda")
        for L32, u32 in W.jellyfish_steps(p_exp, nsteps):
            ua, ub = dev(u32), dev(u32)
            Lcur.copy_(dev(L32))
            rca, sta = a.step(Lcur, ua)
            rcb, stb = b.step(dev(L32), ub)
            assert rca == rcb == gmg.OK and sta["iterations"] == stb["iterations"]
            assert torch.equal(a.p, b.p) and torch.equal(ua, ub)
    finally:
        a.close()
        b.close()


def test_one_call_pressure_step_equals_the_four_calls_and_rejects_bad_coefficients():
    import torch
    p_exp, nsteps = 4, 3
    nx = 2 ** (p_exp + 1)
    n, bc = (nx, nx, nx // 2), W.JELLYFISH_BC
    a = PressureStepper(n, bc, fused=True)
    b = PressureStepper(n, bc, fused=False)
    try:
        for L32, u32 in W.jellyfish_steps(p_exp, nsteps):
            ua, ub = dev(u32), dev(u32)
            rca, sta = a.step(dev(L32), ua)
            rcb, stb = b.step(dev(L32), ub)
            torch.cuda.synchronize()
            assert rca == rcb == gmg.OK and sta["iterations"] == stb["iterations"]
            assert torch.equal(a.p, b.p) and torch.equal(ua, ub)
        bad = dev(L32)
        bad[1, 3, 4, 5] = -0.25
        with pytest.raises(gmg.GMGError):
            a.step(bad, dev(u32))
        # and the context recovers with valid coefficients
        rc, _ = a.step(dev(L32), dev(u32))
        assert rc == gmg.OK
    finally:
        a.close()
        b.close()
