"""-m gpu: the float4 streaming passes around the solve (
kernels_setup.cu): coefficient validation + coarsening, divergence, projection.

They restate the one-value-per-thread kernels with the same operations in the same order, so the
two paths must agree bit for bit (fast_path=1 vs fast_path=0); parity of either with the FP64
oracle is in test_gpu_operators.py / test_gpu_projection.py.  Also: every invalid coefficient is
counted exactly once by the fused validation, wherever it sits in the brick a thread reads."""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_07687_b200 import gmg
from paper_2607_07687_b200 import workloads as W
from gpu_util import dev, host, make_gpu, make_oracle, random_workload, rel_linf

pytestmark = pytest.mark.gpu

SHAPES = [
    ((64, 32, 16), (0, 0, 0)),      # c = (2,2,2) all the way
    ((64, 32, 16), (1, 1, 1)),
    ((256, 6, 12), (0, 1, 0)),      # c = (2,1,2): y cannot coarsen
    ((128, 36, 10), (1, 0, 0)),     # c = (2,2,1) then (2,1,1)
    ((8, 64, 64), (1, 0, 1)),       # x stops first: c = (1,2,2) on the second level
    ((48, 20, 12), (0, 1, 1)),      # nx % 8 == 0 but the next level (24) is taken too, then 12 -> generic
    ((36, 20, 6), (0, 1, 0)),       # nx % 8 != 0: generic kernel on the finest level
]


@pytest.mark.parametrize("n,bc", SHAPES)
def test_float4_passes_are_bit_identical_to_the_generic_kernels(n, bc):
    wl = random_workload(n, bc, seed=41)
    rng = np.random.default_rng(42)
    u = rng.standard_normal((3, n[2], n[1], n[0])).astype(np.float32)
    p = rng.standard_normal((n[2], n[1], n[0])).astype(np.float32)
    wall = (0.5, -1.25, 2.0)
    fast = make_gpu(wl, fast_path=1)
    slow = make_gpu(wl, fast_path=0)
    try:
        assert fast.num_levels() == slow.num_levels()
        for l in range(1, fast.num_levels()):
            assert torch.equal(fast.level_coeffs(l), slow.level_coeffs(l)), l
        assert torch.equal(fast.divergence(dev(u), wall), slow.divergence(dev(u), wall))
        assert torch.equal(fast.project(dev(u), dev(p)), slow.project(dev(u), dev(p)))
    finally:
        fast.close()
        slow.close()


@pytest.mark.parametrize("n,bc", SHAPES[:5])
def test_float4_coarsening_matches_oracle(n, bc):
    wl = random_workload(n, bc, seed=43)
    g = make_gpu(wl)
    h = make_oracle(wl)
    try:
        assert g.num_levels() == h.nlev
        for l in range(1, h.nlev):
            Lg, Lo = host(g.level_coeffs(l)), h.L(l)
            assert rel_linf(Lg, Lo) <= 1e-6, l
            assert np.array_equal(Lg == 0.0, Lo == 0.0), l
    finally:
        g.close()


def test_fused_validation_counts_every_bad_value_once():
    n, bc = (64, 16, 8), (0, 0, 0)
    wl = random_workload(n, bc, seed=44)
    g = gmg.GMG(n, bc)
    try:
        rng = np.random.default_rng(45)
        # every position of the 8 x 2 x 2 brick one thread reads, in each of the three arrays
        for d in range(3):
            for (k, j, i) in [(0, 0, 0), (1, 0, 3), (0, 1, 4), (1, 1, 7), (5, 9, 62), (7, 15, 63)]:
                for v in (-1e-3, np.nan, np.inf):
                    bad = wl.L.copy()
                    bad[d, k, j, i] = v
                    with pytest.raises(gmg.GMGError) as e:
                        g.set_coeffs(dev(bad))
                    assert e.value.code == gmg.EINVAL
                    assert " 1 coefficient" in str(e.value), str(e.value)
        bad = wl.L.copy()
        idx = rng.choice(bad.size, size=37, replace=False)
        bad.reshape(-1)[idx] = -1.0
        with pytest.raises(gmg.GMGError) as e:
            g.set_coeffs(dev(bad))
        assert " 37 coefficient" in str(e.value), str(e.value)
        g.set_coeffs(dev(wl.L))                      # and a valid set is accepted afterwards
        p = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
        assert g.solve(p, dev(wl.z)) == gmg.OK
    finally:
        g.close()
