"""-m gpu: the paper's own "GMG-PCG" -- the V-cycle with a Jacobi-PCG smoother (SURVEY.md S8(f) N2,
PAPER.md:43 S3.1 / Table 1 at PAPER.md:37, reading O12) -- against the FP64 oracle.

Bars: the smoother alone (a handful of operator applications and two inner products per iteration)
rel-L_inf <= 1e-5 for one iteration, 3e-5 for up to three; one cycle 1e-4; solves as in
test_gpu_solvers.py (cycle counts +-1, pressure rel-L2 <= 1e-4 at equal count, residual below tol)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_07687_b200 import gmg
from paper_2607_07687_b200 import workloads as W
from gpu_util import TOL_OP, TOL_P, dev, host, make_gpu, make_oracle, random_workload, rel_l2_demeaned, rel_linf

pytestmark = pytest.mark.gpu

SHAPES = [((32, 24, 16), (0, 0, 0), {}), ((40, 24, 8), (1, 0, 1), {}), ((13, 7, 6), (1, 1, 1), {}),
          ((30, 10, 12), (0, 1, 0), {}), ((256, 20, 12), (1, 0, 1), {"tma_min_cells": 0}),
          ((128, 40, 16), (0, 0, 0), {"tma_min_cells": 0}), ((64, 64, 64), (0, 0, 0), {})]


@pytest.mark.parametrize("n,bc,prm", SHAPES)
@pytest.mark.parametrize("m", [1, 2, 3])
def test_cg_smoother_parity_every_level(n, bc, prm, m):
    wl = random_workload(n, bc, seed=11 * m + sum(n))
    g = make_gpu(wl, **prm)
    h = make_oracle(wl)
    rng = np.random.default_rng(5)
    try:
        assert g.num_levels() == h.nlev
        for lev in range(h.nlev):
            (nx, ny, nz), _ = h.shape(lev)
            x0 = rng.standard_normal((nz, ny, nx)).astype(np.float32)
            b = rng.standard_normal((nz, ny, nx)).astype(np.float32)
            ref = h.level_cg_smooth(lev, x0, b, m)
            out = host(g.op_cg_smooth(lev, dev(x0), dev(b), m))
            tol = TOL_OP if m == 1 else 3 * TOL_OP
            assert rel_linf(out, ref) <= tol, (n, lev, m, rel_linf(out, ref))
    finally:
        g.close()


def test_cg_smoother_zero_count_and_zero_residual_leave_x_alone():
    wl = random_workload((16, 12, 8), (0, 1, 0), seed=3)
    g = make_gpu(wl)
    try:
        x0 = np.random.default_rng(1).standard_normal((8, 12, 16)).astype(np.float32)
        z = np.zeros_like(x0)
        assert np.array_equal(host(g.op_cg_smooth(0, dev(x0), dev(wl.z), 0)), x0.astype(np.float64))
        # b = A x0 exactly representable case: x0 constant -> A x0 = 0 = b: residual 0, rho not < 0
        c = np.full_like(x0, 2.5)
        assert np.array_equal(host(g.op_cg_smooth(0, dev(c), dev(z), 4)), c.astype(np.float64))
    finally:
        g.close()


@pytest.mark.parametrize("name,mk", [("c0", lambda: W.config0()), ("c3p5", lambda: W.config3(5)),
                                     ("rand", lambda: random_workload((48, 32, 16), (1, 0, 1), seed=9))])
def test_cgs_cycle_parity(name, mk):
    wl = mk()
    g = make_gpu(wl)
    h = make_oracle(wl)
    try:
        x0 = np.zeros(wl.z.shape, dtype=np.float32)
        ref = h.vcycle_cgs(x0, wl.z)
        out = host(g.op_vcycle_cgs(dev(x0), dev(wl.z)))
        assert rel_linf(out - out.mean(), ref - ref.mean()) <= 1e-4, rel_linf(out, ref)
    finally:
        g.close()


CONFIGS = {"c0": lambda: W.config0(), "c1": lambda: W.config1(), "c2": lambda: W.config2(),
           "c3p5": lambda: W.config3(5), "c3p6": lambda: W.config3(6), "c4_128": lambda: W.by_name("c4_128")}


@pytest.mark.parametrize("name", sorted(CONFIGS))
def test_cgs_solver_parity(name):
    wl = CONFIGS[name]()
    act = W.active_mask(wl.L, wl.bc)
    g = make_gpu(wl)
    h = make_oracle(wl)
    try:
        g.set_omega(0.75)                      # the relaxation factor must come back untouched
        p = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
        rc = g.solve(p, dev(wl.z), tol=wl.tol, maxiter=wl.maxiter, solver=gmg.GMG_CGS)
        st, hist = g.stats(), g.history()
        ref = h.solve(oracle.GMG_CGS, wl.z, tol=wl.tol, maxiter=wl.maxiter)
        assert rc == gmg.OK and ref["status"] == 0, (name, st, ref["iterations"])
        assert st["omega_final"] == 0.75
        k, ko = st["iterations"], ref["iterations"]
        assert abs(k - ko) <= 1, (name, k, ko)
        assert st["resid_final_rel"] <= wl.tol * (1.0 + 1e-6)
        assert len(hist) == k + 1
        if ko != k:
            ref = h.solve(oracle.GMG_CGS, wl.z, tol=0.0, maxiter=k)
        err = rel_l2_demeaned(host(p), ref["p"], act)
        assert err <= TOL_P, (name, err)
        m = min(k, ko)
        ho, hg = ref["history"][: m + 1], np.array(hist[: m + 1])
        assert np.all(np.abs(hg - ho) <= 0.05 * ho + 1e-7), (name, hg, ho)
        r = oracle.residual(W.effective_L(wl.L, wl.bc), wl.bc, host(p), wl.z)
        assert oracle.norm2(r) / ref["r_ref"] <= wl.tol * 1.02
    finally:
        g.close()


def test_cgs_graph_equals_plain_launches_and_is_reproducible():
    wl = W.config3(5)
    outs = []
    for use_graph in (1, 1, 0):
        g = make_gpu(wl, use_graph=use_graph)
        try:
            p = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
            rc = g.solve(p, dev(wl.z), tol=wl.tol, maxiter=wl.maxiter, solver=gmg.GMG_CGS)
            assert rc == gmg.OK
            outs.append((p.cpu().numpy().copy(), g.stats()["iterations"], tuple(g.history())))
        finally:
            g.close()
    for o in outs[1:]:
        assert o[1] == outs[0][1] and o[2] == outs[0][2] and np.array_equal(o[0], outs[0][0])


def test_cgs_survives_an_incompatible_right_hand_side():
    """A right-hand side with a mean (outside the range of the singular operator) made the first
    version of this smoother blow up in the oracle (d.q -> 0 along the null vector); with the
    mean-free restart both sides stay finite and agree."""
    wl = W.config0()
    z = (wl.z.astype(np.float64) + 1e-3).astype(np.float32)
    act = W.active_mask(wl.L, wl.bc)
    g = make_gpu(wl)
    h = make_oracle(wl)
    try:
        p = torch.zeros(z.shape, dtype=torch.float32, device="cuda")
        rc = g.solve(p, dev(z), tol=0.0, maxiter=6, solver=gmg.GMG_CGS)
        ref = h.solve(oracle.GMG_CGS, z, tol=0.0, maxiter=6)
        assert rc == gmg.NOT_CONVERGED and ref["status"] == 1
        out = host(p)
        assert np.all(np.isfinite(out)) and np.abs(out).max() < 1e3
        assert rel_l2_demeaned(out, ref["p"], act) <= TOL_P
    finally:
        g.close()


@pytest.mark.parametrize("n,bc", [((32, 32, 16), (0, 0, 0)), ((16, 16, 16), (1, 0, 1)), ((64, 64, 32), (1, 1, 1)),
                                  ((40, 24, 8), (1, 0, 1)), ((128, 128, 64), (1, 1, 1))])
def test_single_cta_smoothing_gives_the_bits_of_the_multi_launch_path(n, bc):
    """`small_cg` (include/gmg.h): on levels of at most 4096 cells a whole smoothing is ONE kernel that
    keeps the multi-launch kernels' expressions and summation order.  Every level and iteration count
    through the hook, one whole cycle, and a solve: identical bits with the switch on and off."""
    wl = random_workload(n, bc, seed=sum(n))
    on, off = make_gpu(wl, small_cg=1), make_gpu(wl, small_cg=0)
    rng = np.random.default_rng(9)
    try:
        small = 0
        for lev in range(on.num_levels()):
            (nx, ny, nz), _ = on.level_shape(lev)
            small += int(nx * ny * nz <= 4096 and nx % 4 == 0)
            x0 = dev(rng.standard_normal((nz, ny, nx)))
            b = dev(rng.standard_normal((nz, ny, nx)))
            for m in (1, 2, 5, 32):
                a = on.op_cg_smooth(lev, x0.clone(), b, m)
                c = off.op_cg_smooth(lev, x0.clone(), b, m)
                assert torch.equal(a, c), (n, lev, m, float((a - c).abs().max()))
        assert small >= 1, "the case must reach a level the single-CTA kernel takes"
        p, z = dev(rng.standard_normal(wl.z.shape)), dev(wl.z)
        assert torch.equal(on.op_vcycle_cgs(p.clone(), z), off.op_vcycle_cgs(p.clone(), z))
        out = []
        for g in (on, off):
            x = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
            rc = g.solve(x, z, tol=1e-5, maxiter=60, solver=gmg.GMG_CGS)
            out.append((rc, g.stats()["iterations"], x, g.stats()["kernel_launches"]))
        assert out[0][:2] == out[1][:2] and torch.equal(out[0][2], out[1][2])
        assert out[0][3] < out[1][3]          # fewer launches
    finally:
        on.close()
        off.close()
