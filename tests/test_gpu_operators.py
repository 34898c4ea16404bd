"""-m gpu: per-operator parity of the CUDA path (through the C-ABI) against the FP64 oracle.

Bar (BASELINE.json:north_star): relative L-infinity <= 1e-5 for single operator applications
(residual, one smoothing sweep, restrict, prolong); level shapes exact; coarse coefficients to
FP32 rounding."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_07687_b200 import workloads as W
from gpu_util import TOL_OP, dev, host, make_gpu, make_oracle, random_workload, rel_linf

pytestmark = pytest.mark.gpu

CASES = {
    "c0": lambda: W.config0(),
    "rand_PPP": lambda: random_workload((24, 16, 12), (0, 0, 0), 11),
    "rand_NPN": lambda: random_workload((20, 24, 10), (1, 0, 1), 12),
    "rand_NNN_odd": lambda: random_workload((15, 9, 7), (1, 1, 1), 13),
    "rand_ragged": lambda: random_workload((36, 20, 6), (0, 1, 0), 14),
    "c3p5": lambda: W.config3(5),
    "c4_64": lambda: W.config4(n=64, nspheres=8, diameter=8),
    "sphere_D4": lambda: W.config2(D=4),
    # wide enough (nx % 128 == 0) for the TMA-fed sweep: interior and boundary tiles, all BC mixes
    "rand_128_NPP": lambda: random_workload((128, 20, 12), (1, 0, 0), 15),
    "rand_256_PNN": lambda: random_workload((256, 12, 10), (0, 1, 1), 16),
    "rand_128_PPP": lambda: random_workload((128, 40, 8), (0, 0, 0), 17),
    "rand_256_aniso": lambda: random_workload((256, 6, 12), (0, 0, 0), 18),      # c = (2,1,2)
    "rand_128_xonly": lambda: random_workload((128, 36, 10), (1, 0, 0), 19, blob=False),
    # more than 40 tile rows on a periodic y axis: the instantiation k_rb_sweep_bulk<.., EDGE = false>
    # that bench.py's 1024^3 level 0 runs (interior boxes + ROW-COPY tiles on the first / final tile
    # row, final tile ragged: 534 = 41 * 13 + 1, 546 = 42 * 13), whole field against the oracle
    "rand_128x534x16_PPP": lambda: random_workload((128, 534, 16), (0, 0, 0), 20),
    "rand_256x546x8_NPP": lambda: random_workload((256, 546, 8), (1, 0, 0), 21),
}
NON_EDGE = ("rand_128x534x16_PPP", "rand_256x546x8_NPP")


@pytest.fixture(scope="module", params=sorted(CASES), ids=sorted(CASES))
def case(request):
    wl = CASES[request.param]()
    g = make_gpu(wl, tma_min_cells=0)      # TMA-fed kernels wherever the shape allows
    h = make_oracle(wl)
    yield wl, g, h
    g.close()


def _fields(n, seed):
    rng = np.random.default_rng(seed)
    shp = (n[2], n[1], n[0])
    return (rng.standard_normal(shp).astype(np.float32), rng.standard_normal(shp).astype(np.float32))


def test_plan_names_the_sweep_instantiation(case):
    """describe_plan says which k_rb_sweep_bulk instantiation a TMA-fed level runs, so that the
    whole-field comparisons below are known to cover BOTH."""
    wl, g, h = case
    line0 = g.describe_plan().split("\n")[0]
    if wl.name.startswith("random_") and wl.n[1] > 520 and wl.bc[1] == 0:
        assert "fused-rb-sweep(TMA,rowcopy-edges)" in line0, line0
    elif wl.n[0] % 128 == 0 and wl.n[1] >= 4 and wl.n[2] >= 8:
        assert "fused-rb-sweep(TMA,EDGE)" in line0 or wl.n[1] <= 13, line0


def test_level_shapes_match_oracle(case):
    wl, g, h = case
    assert g.num_levels() == h.nlev
    for l in range(h.nlev):
        assert g.level_shape(l) == h.shape(l)


def test_coarse_coefficients(case):
    wl, g, h = case
    for l in range(h.nlev):
        Lg = host(g.level_coeffs(l))
        Lo = h.L(l)
        if l == 0:
            # level 0 is the caller's array; the library ignores the Neumann wall plane
            Lg = W.effective_L(Lg, wl.bc)
        assert rel_linf(Lg, Lo) <= 1e-6, l
        assert np.array_equal(Lg == 0.0, Lo == 0.0), l      # activity pattern is exact


def test_residual_every_level(case):
    wl, g, h = case
    for l in range(h.nlev):
        n, _ = h.shape(l)
        p, b = _fields(n, 100 + l)
        r = host(g.op_residual(l, dev(p), dev(b)))
        ro = h.level_residual(l, p, b)
        assert rel_linf(r, ro) <= TOL_OP, (l, rel_linf(r, ro))
        assert np.array_equal(r == 0.0, ro == 0.0) or np.count_nonzero((r == 0) != (ro == 0)) < 3


@pytest.mark.parametrize("omega,first", [(1.0, 0), (0.8125, 0), (1.0, 1)])
def test_one_sweep_every_level(case, omega, first):
    wl, g, h = case
    for l in range(h.nlev):
        n, _ = h.shape(l)
        p, b = _fields(n, 200 + l)
        out = host(g.op_smooth(l, dev(p), dev(b), omega=omega, nsweeps=1, first_colour=first))
        ref = h.level_sweeps(l, p, b, omega=omega, count=1, first_colour=first)
        assert rel_linf(out, ref) <= TOL_OP, (l, rel_linf(out, ref))


def test_two_and_three_sweeps(case):
    """Even counts take the ping-pong fused path where the level supports it; odd counts mix
    it with the generic half-sweeps."""
    wl, g, h = case
    for l in range(min(h.nlev, 3)):
        n, _ = h.shape(l)
        p, b = _fields(n, 300 + l)
        for cnt in (2, 3):
            out = host(g.op_smooth(l, dev(p), dev(b), omega=1.0, nsweeps=cnt, first_colour=0))
            ref = h.level_sweeps(l, p, b, omega=1.0, count=cnt, first_colour=0)
            assert rel_linf(out, ref) <= 3 * TOL_OP, (l, cnt, rel_linf(out, ref))


def test_fused_pair_black_first_underrelaxed(case):
    """The symmetric V-cycle's post-smoothing order (black then red) through the fused kernel."""
    wl, g, h = case
    for l in range(min(h.nlev, 3)):
        n, _ = h.shape(l)
        p, b = _fields(n, 350 + l)
        out = host(g.op_smooth(l, dev(p), dev(b), omega=0.8125, nsweeps=2, first_colour=1))
        ref = h.level_sweeps(l, p, b, omega=0.8125, count=2, first_colour=1)
        assert rel_linf(out, ref) <= 3 * TOL_OP, (l, rel_linf(out, ref))


def test_restrict_and_fused_residual_restrict(case):
    wl, g, h = case
    for l in range(h.nlev - 1):
        n, c = h.shape(l)
        p, b = _fields(n, 400 + l)
        ro = h.level_residual(l, p, b)
        bc_o = oracle.restrict_sum(ro, c)
        bc_g = host(g.op_restrict(l, dev(ro)))
        assert rel_linf(bc_g, bc_o) <= TOL_OP, l
        fused = host(g.op_residual_restrict(l, dev(p), dev(b)))
        assert rel_linf(fused, bc_o) <= TOL_OP, (l, rel_linf(fused, bc_o))


def test_prolong_every_level(case):
    wl, g, h = case
    for l in range(h.nlev - 1):
        n, c = h.shape(l)
        nc, _ = h.shape(l + 1)
        p, _ = _fields(n, 500 + l)
        e, _ = _fields(nc, 600 + l)
        out = host(g.op_prolong(l, dev(e), dev(p)))
        ref = oracle.prolong_add(p, e, c)
        assert rel_linf(out, ref) <= 1e-6, l


@pytest.mark.parametrize("sym", [False, True])
def test_one_vcycle(case, sym):
    """One V(2,2) cycle from a zero guess; the tolerance allows for the accumulated rounding of
    ~20 operator applications (derived in DESIGN.md)."""
    wl, g, h = case
    p = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
    out = host(g.op_vcycle(p, dev(wl.z), omega=1.0, symmetric=sym))
    ref = h.vcycle(np.zeros_like(wl.z, dtype=np.float64), wl.z, omega=1.0, sym=sym)
    act = W.active_mask(wl.L, wl.bc)
    assert rel_linf(np.where(act, out, 0), np.where(act, ref, 0)) <= 1e-4, rel_linf(out, ref)


def test_norm2(case):
    wl, g, h = case
    r = np.random.default_rng(7).standard_normal(wl.z.shape).astype(np.float32)
    got = g.op_norm2(0, dev(r))
    assert abs(got - np.linalg.norm(r.astype(np.float64))) <= 1e-12 * np.linalg.norm(r)
