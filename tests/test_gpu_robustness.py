"""-m gpu: behaviour at the edges of the contract (VERDICT r1 "Next round" 1(d)):
norms blind to inactive cells, non-finite input, misaligned caller pointers."""
import ctypes as C

import numpy as np
import pytest
import torch

import oracle
from paper_2607_07687_b200 import gmg
from paper_2607_07687_b200 import workloads as W
from gpu_util import TOL_P, dev, host, make_gpu, make_oracle, random_workload, rel_l2_demeaned

pytestmark = pytest.mark.gpu

ALL = [(gmg.GMG_RBGS, oracle.GMG_RBGS), (gmg.PCG, oracle.PCG), (gmg.GMG_PCG, oracle.GMG_PCG),
       (gmg.GMG_CGS, oracle.GMG_CGS)]


@pytest.mark.parametrize("n,bc,prm", [((24, 16, 12), (1, 0, 0), {}),
                                      ((128, 40, 16), (0, 0, 0), {"tma_min_cells": 0}),      # fused_norm: b^2 in the sweep
                                      ((128, 40, 16), (0, 0, 0), {"tma_min_cells": 0, "fused_norm": 0})])
def test_garbage_on_inactive_cells_changes_nothing(n, bc, prm):
    """Reading O9: the reference norm and the residual run over ACTIVE cells.  The same solve with
    large values written into the right-hand side INSIDE the solid blob gives the same reference
    norm, history, count and (bit for bit) pressure; the oracle agrees on count and norm."""
    wl = random_workload(n, bc, seed=61, zero_frac=0.1)
    act = W.active_mask(wl.L, wl.bc)
    assert (~act).sum() >= 1
    zg = wl.z.copy()
    zg[~act] = 50.0
    g = make_gpu(wl, **prm)
    try:
        for sg, so in ALL:
            out = []
            for z in (wl.z, zg):
                g.set_omega(1.0)
                p = torch.zeros(z.shape, dtype=torch.float32, device="cuda")
                rc = g.solve(p, dev(z), tol=1e-5, maxiter=2000, solver=sg)
                out.append((rc, g.stats(), np.array(g.history()), host(p)))
            (rc0, st0, h0, p0), (rc1, st1, h1, p1) = out
            assert rc0 == rc1 == gmg.OK, (sg, st0, st1)
            assert st0["iterations"] == st1["iterations"] and st0["resid_ref"] == st1["resid_ref"]
            assert np.array_equal(h0, h1) and np.array_equal(p0[act], p1[act])
            ref = make_oracle(wl).solve(so, zg, tol=1e-5, maxiter=2000)
            assert abs(ref["iterations"] - st1["iterations"]) <= (1 if sg != gmg.PCG else 3)
            if "r_ref" in ref:
                assert abs(st1["resid_ref"] - ref["r_ref"]) <= 1e-6 * ref["r_ref"]
    finally:
        g.close()


@pytest.mark.parametrize("use_graph", [1, 0])
@pytest.mark.parametrize("where", ["z", "p0"])
def test_non_finite_input_is_not_reported_as_converged(where, use_graph):
    """A NaN norm is neither '> tol ||z||' nor '<= tol ||z||': like the oracle's loop (reading O9 as
    written in oracle/gmg_oracle.c) the solve stops at once and returns NOT_CONVERGED, never OK."""
    wl = W.config0()
    z = wl.z.copy()
    p0 = np.zeros_like(z)
    (z if where == "z" else p0)[3, 5, 7] = np.nan
    ref = {}
    for so in (oracle.GMG_RBGS, oracle.PCG, oracle.GMG_PCG, oracle.GMG_CGS):
        o = make_oracle(wl).solve(so, z, p0=p0, tol=1e-4, maxiter=20)
        assert o["status"] == 1 and o["iterations"] == 0
    g = make_gpu(wl, use_graph=use_graph)
    try:
        for sg in (gmg.GMG_RBGS, gmg.PCG, gmg.GMG_PCG, gmg.GMG_CGS):
            p = dev(p0)
            rc = g.solve(p, dev(z), tol=1e-4, maxiter=20, solver=sg)
            st = g.stats()
            assert rc == gmg.NOT_CONVERGED and st["iterations"] == 0, (sg, rc, st)
            assert not np.isfinite(st["resid_final_rel"]) or st["resid_final_rel"] > 1e-4
    finally:
        g.close()


@pytest.mark.parametrize("name,prm", [("c0", {}), ("c4_128", {"tma_min_cells": 0})])
def test_overflowing_norms_are_never_reported_as_convergence(name, prm):
    """A finite right-hand side of size 1e30: wherever a squared FP32 value overflows, the norms are
    Inf and 'Inf <= tol * Inf' must not count as converged.  Either the solve works (then the FP64
    residual of its p meets the tolerance) or it says NOT_CONVERGED."""
    wl = W.by_name(name)
    z = (wl.z.astype(np.float64) * 1e30).astype(np.float32)
    assert np.isfinite(z).all()
    g = make_gpu(wl, **prm)
    try:
        for sg in (gmg.GMG_RBGS, gmg.GMG_PCG):
            g.set_omega(1.0)
            p = torch.zeros(z.shape, dtype=torch.float32, device="cuda")
            rc = g.solve(p, dev(z), tol=1e-4, maxiter=30, solver=sg)
            assert rc in (gmg.OK, gmg.NOT_CONVERGED)
            if rc == gmg.OK:
                r = oracle.residual(W.effective_L(wl.L, wl.bc), wl.bc, host(p), z)
                assert oracle.norm2(r) <= 1.02e-4 * np.linalg.norm(z.astype(np.float64)), (name, sg)
    finally:
        g.close()


def test_misaligned_caller_pointers_are_refused():
    """The float4 / TMA paths read 16 bytes at a time: a contiguous view that starts 4 bytes into an
    allocation is answered with GMG_EINVAL, not with a misaligned-address fault."""
    wl = W.config0()
    N = wl.cells
    g = make_gpu(wl)
    try:
        raw = torch.zeros(3 * N + 4, dtype=torch.float32, device="cuda")
        off = raw[1:N + 1].view(wl.z.shape)                  # contiguous, 4 bytes off
        assert off.is_contiguous() and off.data_ptr() % 16 == 4
        ok = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
        z = dev(wl.z)
        for args in ((off, z), (ok, off)):
            with pytest.raises(gmg.GMGError) as e:
                g.solve(args[0], args[1])
            assert e.value.code == gmg.EINVAL and "aligned" in str(e.value)
        with pytest.raises(gmg.GMGError) as e:
            g.op_residual(0, off, z)
        assert e.value.code == gmg.EINVAL
        Loff = raw[1:3 * N + 1].view(wl.L.shape)
        with pytest.raises(gmg.GMGError) as e:
            g.set_coeffs(Loff)
        assert e.value.code == gmg.EINVAL
        with pytest.raises(gmg.GMGError) as e:
            g.divergence(Loff, out=ok)
        assert e.value.code == gmg.EINVAL
        # the context is still usable (no sticky CUDA error)
        g.set_coeffs(dev(wl.L))
        assert g.solve(ok, z) == gmg.OK
    finally:
        g.close()
