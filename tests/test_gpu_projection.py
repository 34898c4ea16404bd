"""-m gpu: the steps either side of the solve ("predictor +
corrector steps"): divergence of a staggered velocity field -> Poisson solve -> projection.
Operator parity vs the FP64 oracle (rel-L-inf <= 1e-5) and the end-to-end property that the
projected field's divergence is the solve's residual (<= tol * ||z||)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_07687_b200 import gmg
from paper_2607_07687_b200 import workloads as W
from gpu_util import TOL_OP, dev, host, make_gpu, random_workload, rel_linf

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n,bc", [((24, 16, 12), (0, 0, 0)), ((20, 24, 10), (1, 0, 1)),
                                  ((15, 9, 7), (1, 1, 1)), ((128, 20, 12), (1, 0, 0))])
def test_divergence_and_projection_match_oracle(n, bc):
    wl = random_workload(n, bc, seed=31)
    rng = np.random.default_rng(32)
    u = rng.standard_normal((3, n[2], n[1], n[0])).astype(np.float32)
    p = rng.standard_normal((n[2], n[1], n[0])).astype(np.float32)
    wall = (0.25, -0.5, 0.75)
    g = make_gpu(wl)
    try:
        z = host(g.divergence(dev(u), wall))
        zo = oracle.divergence(u, bc, wall)
        assert rel_linf(z, zo) <= TOL_OP
        un = host(g.project(dev(u), dev(p)))
        uo = oracle.project(wl.L, bc, p, u)
        assert rel_linf(un, uo) <= TOL_OP
        # wall faces of Neumann axes are untouched, bit for bit
        for d in range(3):
            if bc[d] == 1:
                sl = [slice(None)] * 3
                sl[2 - d] = 0
                assert np.array_equal(un[d][tuple(sl)].astype(np.float32), u[d][tuple(sl)])
    finally:
        g.close()


@pytest.mark.parametrize("name", ["c2_small", "c3p5"])
def test_pressure_step_makes_the_field_divergence_free(name):
    """div(u*) -> solve -> u = u* - L grad p: the remaining divergence IS the solve's residual."""
    wl = W.config2(D=4) if name == "c2_small" else W.config3(5)
    n, bc = wl.n, wl.bc
    rng = np.random.default_rng(33)
    Le = W.effective_L(wl.L, bc)
    u = (rng.standard_normal((3, n[2], n[1], n[0])) * Le).astype(np.float32)   # no flow through solids / walls
    g = make_gpu(wl)
    try:
        ud = dev(u)
        z = g.divergence(ud)
        # compatible by construction: wall faces carry 0, periodic axes telescope
        assert abs(float(z.double().sum().item())) <= 1e-3 * float(z.double().abs().sum().item())
        p = torch.zeros_like(z)
        rc = g.solve(p, z, tol=1e-4, maxiter=100, solver=gmg.GMG_RBGS)
        st = g.stats()
        assert rc == gmg.OK
        g.project(ud, p)
        div_after = g.divergence(ud)
        zn = float(torch.linalg.vector_norm(z.double()).item())
        dn = float(torch.linalg.vector_norm(div_after.double()).item())
        assert dn <= 1.05 * 1e-4 * zn + 1e-6 * zn, (dn / zn, st)
        # and it equals the residual field z - A p (identity div(u - L grad p) = div u - A p)
        r = g.op_residual(0, p, z)
        act = torch.from_numpy(W.active_mask(wl.L, bc)).cuda()
        diff = float(((div_after - r) * act).abs().max().item())
        assert diff <= 1e-4 * float(z.abs().max().item())
    finally:
        g.close()
