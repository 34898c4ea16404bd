"""-m gpu: the fused_norm path of gmg_solve (include/gmg.h): the first pre-smoothing sweep of cycle
k+1, run out of place by the TMA-fed kernel, also accumulates ||z - A p_k||^2 (and ||z||^2 over the
active cells), so the 20 B/cell stopping-test pass after every V-cycle disappears.  It must change
nothing: same sweep result bit for bit, the oracle's norms, the same iterates, counts and omega
sequence -- including when the speculated relaxation factor turns out wrong and the sweep is re-run."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_07687_b200 import gmg
from paper_2607_07687_b200 import workloads as W
from gpu_util import TOL_OP, TOL_P, dev, host, make_gpu, make_oracle, random_workload, rel_l2_demeaned, rel_linf

pytestmark = pytest.mark.gpu


# (128, 534, 16): 42 tile rows, as many as make the PLAIN sweep take the row-copy instantiation --
# the norm-carrying one keeps the EDGE body at any size, here with interior, FIRST and ragged FINAL
# tile rows like the 1024^3 level 0; (128, 12, 16): a single periodic tile row, the one shape on
# which the norm-carrying sweep runs the non-EDGE instantiation (row copies everywhere)
@pytest.mark.parametrize("n,bc", [((128, 40, 16), (0, 0, 0)), ((256, 20, 12), (1, 0, 1)),
                                  ((128, 27, 70), (1, 1, 1)), ((384, 16, 8), (0, 1, 0)),
                                  ((128, 534, 16), (0, 0, 0)), ((128, 12, 16), (0, 0, 0))])
@pytest.mark.parametrize("first_colour", [0, 1])
def test_sweep_with_norm_matches_oracle_and_the_plain_sweep(n, bc, first_colour):
    wl = random_workload(n, bc, seed=sum(n) + first_colour)
    g = make_gpu(wl, tma_min_cells=0)
    h = make_oracle(wl)
    rng = np.random.default_rng(4)
    try:
        src = rng.standard_normal((n[2], n[1], n[0])).astype(np.float32)
        b = rng.standard_normal((n[2], n[1], n[0])).astype(np.float32)
        dst, rr, bb = g.op_sweep_with_norm(0, dev(src), dev(b), omega=0.875, first_colour=first_colour)
        ref = h.level_sweeps(0, src, b, omega=0.875, count=1, first_colour=first_colour)
        assert rel_linf(host(dst), ref) <= TOL_OP
        # bit-identical to one sweep of the generic half-sweep kernels
        plain = g.op_smooth(0, dev(src), dev(b), omega=0.875, nsweeps=1, first_colour=first_colour)
        assert torch.equal(dst, plain)
        r = h.level_residual(0, src, b)
        act = W.active_mask(wl.L, wl.bc)
        assert abs(rr - float((r * r).sum())) <= 2e-6 * float((r * r).sum())
        bref = float((np.where(act, b.astype(np.float64), 0.0) ** 2).sum())
        assert abs(bb - bref) <= 2e-6 * bref
    finally:
        g.close()


def test_levels_the_tma_kernel_cannot_take_are_refused():
    wl = random_workload((40, 24, 8), (0, 1, 0), seed=2)
    g = make_gpu(wl, tma_min_cells=0)
    try:
        x = dev(wl.z)
        with pytest.raises(gmg.GMGError):
            g.op_sweep_with_norm(0, x, x.clone())
    finally:
        g.close()


def _solve(wl, **prm):
    g = make_gpu(wl, **prm)
    try:
        p = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
        rc = g.solve(p, dev(wl.z), tol=prm.pop("_tol", wl.tol), maxiter=wl.maxiter, solver=gmg.GMG_RBGS)
        return rc, p.cpu().numpy().copy(), g.stats(), np.array(g.history()), np.array(g.omega_history())
    finally:
        g.close()


@pytest.mark.parametrize("name", ["c4_128", "c1"])
@pytest.mark.parametrize("use_graph", [1, 0])
def test_fused_norm_changes_nothing_but_the_time(name, use_graph):
    wl = W.by_name(name)
    a = _solve(wl, tma_min_cells=0, cluster_tail=1, fused_norm=1, use_graph=use_graph)
    b = _solve(wl, tma_min_cells=0, cluster_tail=1, fused_norm=0, use_graph=use_graph)
    assert a[0] == b[0] == gmg.OK
    assert a[2]["iterations"] == b[2]["iterations"]
    assert np.array_equal(a[1], b[1])                          # the iterate: bit for bit
    assert np.allclose(a[3], b[3], rtol=1e-5, atol=0)          # the norms: another summation order
    assert np.array_equal(a[4], b[4])
    # and against the oracle
    h = make_oracle(wl)
    ref = h.solve(oracle.GMG_RBGS, wl.z, tol=wl.tol, maxiter=wl.maxiter)
    assert ref["iterations"] == a[2]["iterations"]
    assert np.all(np.abs(a[3] - ref["history"]) <= 0.05 * ref["history"] + 1e-7)
    assert rel_l2_demeaned(a[1], ref["p"], W.active_mask(wl.L, wl.bc)) <= TOL_P


def test_wrong_speculation_of_omega_reruns_the_sweep():
    """An under-smoothed V(2,0) case whose first cycle GROWS the residual: omega drops to 7/8, the
    sweep that already ran with the decay-branch omega (1) is run again.  The omega sequence and the
    residual history must be the oracle's, and equal to the unfused path's."""
    wl = random_workload((128, 16, 16), (1, 1, 1), seed=3, zero_frac=0.5)
    prm = dict(nu_pre=2, nu_post=0, nu_coarse=2, tma_min_cells=0, cluster_tail=0)
    outs = []
    for fused in (1, 0):
        g = make_gpu(wl, fused_norm=fused, **prm)
        try:
            assert "fused-rb-sweep(TMA" in g.describe_plan().split("\n")[0]
            p = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
            rc = g.solve(p, dev(wl.z), tol=0.0, maxiter=8, solver=gmg.GMG_RBGS)
            assert rc == gmg.NOT_CONVERGED
            outs.append((p.cpu().numpy().copy(), np.array(g.history()), np.array(g.omega_history()), g.stats()))
        finally:
            g.close()
    h = make_oracle(wl, nu1=2, nu2=0, nuc=2)
    ref = h.solve(oracle.GMG_RBGS, wl.z, tol=0.0, maxiter=8)
    assert np.any(np.diff(ref["history"]) > 0) and ref["omegas"][1] == 0.875
    for p, hist, om, st in outs:
        assert np.array_equal(om, ref["omegas"])
        assert np.all(np.abs(hist - ref["history"]) <= 0.05 * ref["history"])
        assert st["omega_final"] == h.omega
    assert np.array_equal(outs[0][0], outs[1][0])


@pytest.mark.parametrize("tol,maxiter", [(1e-4, 50), (0.0, 1), (0.0, 4), (1e-3, 50), (3e-6, 50)])
def test_last_cycle_prediction_changes_nothing(tol, maxiter):
    """The cycle expected to be the last (rate-based, or the maxiter-th) is followed by the plain
    norm pass instead of the next cycle's norm-carrying sweep; when the prediction fails that sweep
    runs at the start of the next cycle.  Whatever the tolerance makes of the prediction (hit, miss,
    never made), iterates and counts equal the unfused loop's."""
    wl = W.by_name("c4_128")
    outs = []
    for fused in (1, 0):
        g = make_gpu(wl, tma_min_cells=0, fused_norm=fused)
        try:
            p = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
            rc = g.solve(p, dev(wl.z), tol=tol, maxiter=maxiter, solver=gmg.GMG_RBGS)
            outs.append((rc, p.cpu().numpy().copy(), g.stats()["iterations"], np.array(g.history())))
        finally:
            g.close()
    a, b = outs
    assert a[0] == b[0] and a[2] == b[2]
    assert np.array_equal(a[1], b[1])
    assert np.allclose(a[3], b[3], rtol=1e-5, atol=0)
