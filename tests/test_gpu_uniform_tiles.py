"""-m gpu: the lean path of the TMA-fed kernels (include/gmg.h `uniform_tiles`, csrc/uniform.cuh).
Where every face coefficient in a CTA's footprint equals the level's constant (1 on the finest
level away from bodies), the kernels do not load the coefficient streams at all.
allows this as "a lossless 'tile is all L=1' flag ... honest only if reported as such": LOSSLESS is
what these tests pin -- every operator and every solve gives the SAME BITS with the flag on and
off -- and REPORTED is gmg_stats.uniform_fraction / bytes_as_run.  Parity with the oracle of the
configurations that take the lean path (c1, c4_*) is in the other test files, which run with the
default uniform_tiles = 1."""
import numpy as np
import pytest
import torch

from paper_2607_07687_b200 import gmg
from paper_2607_07687_b200 import workloads as W
from gpu_util import dev, make_gpu

pytestmark = pytest.mark.gpu


def _ones_with_bodies(n, bc, seed, nblobs=2, scale=1.0):
    """L == 1 except inside a few small boxes (random values incl. zeros) -- the structure of an
    immersed-boundary coefficient field; compatible random right-hand side."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = n
    L = np.full((3, nz, ny, nx), scale, dtype=np.float64)
    for _ in range(nblobs):
        i0, j0, k0 = (int(rng.integers(0, max(1, m - 6))) for m in (nx, ny, nz))
        blk = rng.uniform(0.0, 1.0, (3, 5, 5, 5))
        blk[rng.uniform(size=blk.shape) < 0.3] = 0.0
        L[:, k0:k0 + 5, j0:j0 + 5, i0:i0 + 5] = blk[:, :min(5, nz - k0), :min(5, ny - j0), :min(5, nx - i0)]
    L32 = L.astype(np.float32)
    act = W.active_mask(L32, bc)
    z = W.project_compatible(rng.standard_normal((nz, ny, nx)), act)
    return W.Workload(f"ones_{nx}x{ny}x{nz}", tuple(n), tuple(bc), L32, z.astype(np.float32), seed=seed)


CASES = {
    "c4_128": lambda: W.by_name("c4_128"),                                   # EDGE kernel, 10 tile rows
    "c1": lambda: W.config1(),                                              # L == 1 everywhere
    "ones_256x64x32_PPP": lambda: _ones_with_bodies((256, 64, 32), (0, 0, 0), 1),
    "ones_128x534x16_PPP": lambda: _ones_with_bodies((128, 534, 16), (0, 0, 0), 2),   # non-EDGE kernel
    "ones_256x40x24_NPN": lambda: _ones_with_bodies((256, 40, 24), (1, 0, 1), 3),     # walls: x tiles all refuse
    "ones_384x64x64_PNP": lambda: _ones_with_bodies((384, 64, 64), (0, 1, 0), 4, nblobs=1),   # walls in y: EDGE, YMODE 0
    "ones_128x64x64_none": lambda: _ones_with_bodies((128, 64, 64), (0, 0, 0), 5, nblobs=0),
    # one small body in a big box: most tiles lean, some not -- both halves of the folded prolongation
    "ones_256x128x64_one": lambda: _ones_with_bodies((256, 128, 64), (0, 0, 0), 6, nblobs=1),
}


@pytest.fixture(scope="module", params=sorted(CASES), ids=sorted(CASES))
def pair(request):
    wl = CASES[request.param]()
    on = make_gpu(wl, tma_min_cells=0, uniform_tiles=1)
    off = make_gpu(wl, tma_min_cells=0, uniform_tiles=0)
    yield wl, on, off
    on.close()
    off.close()


def _fields(wl, seed):
    rng = np.random.default_rng(seed)
    shp = wl.z.shape
    return dev(rng.standard_normal(shp)), dev(rng.standard_normal(shp))


def test_lean_path_is_taken_and_reported(pair):
    wl, on, off = pair
    p = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
    on.solve(p, dev(wl.z), tol=0.0, maxiter=1)
    off.solve(p.zero_(), dev(wl.z), tol=0.0, maxiter=1)
    s_on, s_off = on.stats(), off.stats()
    assert s_off["uniform_fraction"] == 0.0 and s_off["bytes_as_run"] == s_off["bytes_algorithmic"]
    if wl.name.startswith("ones_256x40x24"):
        # two x tiles, both next to an x wall: no CTA may take the lean path
        assert s_on["uniform_fraction"] == 0.0
    else:
        assert s_on["uniform_fraction"] > (0.99 if wl.name in ("config1_tgv", "ones_128x64x64") else 0.1), s_on
        assert s_on["bytes_as_run"] < s_on["bytes_algorithmic"]
    assert s_on["bytes_algorithmic"] == s_off["bytes_algorithmic"]       # the 24-B reference line stays


@pytest.mark.parametrize("omega,first,count", [(1.0, 0, 1), (0.8125, 1, 2), (1.0, 0, 2), (0.9375, 0, 3)])
def test_sweeps_bit_identical(pair, omega, first, count):
    wl, on, off = pair
    p, b = _fields(wl, 10 * count + first)
    a = on.op_smooth(0, p.clone(), b, omega=omega, nsweeps=count, first_colour=first)
    c = off.op_smooth(0, p.clone(), b, omega=omega, nsweeps=count, first_colour=first)
    assert torch.equal(a, c)


def test_sweep_with_norm_bit_identical(pair):
    wl, on, off = pair
    p, b = _fields(wl, 33)
    for first in (0, 1):
        d1, rr1, bb1 = on.op_sweep_with_norm(0, p, b, omega=0.875, first_colour=first)
        d0, rr0, bb0 = off.op_sweep_with_norm(0, p, b, omega=0.875, first_colour=first)
        assert torch.equal(d1, d0)
        assert rr1 == rr0 and bb1 == bb0          # same per-thread sums in the same order


def test_residual_restrict_and_vcycle_bit_identical(pair):
    wl, on, off = pair
    p, b = _fields(wl, 44)
    if on.num_levels() > 1:
        assert torch.equal(on.op_residual_restrict(0, p, b), off.op_residual_restrict(0, p, b))
    for sym in (False, True):
        assert torch.equal(on.op_vcycle(p.clone(), b, omega=0.9375, symmetric=sym),
                           off.op_vcycle(p.clone(), b, omega=0.9375, symmetric=sym))


def test_prolongation_folded_into_the_sweep_is_bit_identical_every_time(pair):
    """With uniform bricks marked, the first post-smoothing sweep of a TMA-fed 2x2x2 level takes the
    prolongation + correction along (lean tiles: parents added where source values enter registers;
    other tiles: a corrected copy of their footprints) instead of running k_prolong_add4 first.  The
    lean kernel stores corrected values into planes its neighbours read, so a missing barrier shows
    as a run-to-run difference: every one of 25 cycles must give the bits of the separate pass."""
    wl, on, off = pair
    p0 = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
    on.solve(p0, dev(wl.z), tol=0.0, maxiter=1)
    share = on.stats()["uniform_fraction"]
    plan = on.describe_plan().split("\n")[0]
    folded = "prolong=in-sweep" in plan
    # folded where at least half of the level's tiles are lean (a remaining tile's corrected copy
    # costs more than the separate pass)
    if share > 0.6 and on.level_shape(0)[1] == (2, 2, 2):      # (the folded kernels assume 2x2x2 coarsening)
        assert folded, (share, plan)
    if share < 0.4:
        assert not folded, (share, plan)
    if wl.name == "ones_256x128x64":
        assert folded and 0.5 < share < 1.0, (share, plan)
    assert "prolong=pass" in off.describe_plan().split("\n")[0]
    p, b = _fields(wl, 55)
    for sym in (False, True):
        ref = off.op_vcycle(p.clone(), b, omega=0.875, symmetric=sym)
        for _ in range(25 if folded else 2):
            assert torch.equal(on.op_vcycle(p.clone(), b, omega=0.875, symmetric=sym), ref)


@pytest.mark.parametrize("solver", [gmg.GMG_RBGS, gmg.GMG_PCG, gmg.PCG, gmg.GMG_CGS])
def test_solves_bit_identical(pair, solver):
    wl, on, off = pair
    out = []
    for g in (on, off):
        g.set_omega(1.0)
        p = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
        rc = g.solve(p, dev(wl.z), tol=1e-5, maxiter=60 if solver != gmg.PCG else 3000, solver=solver)
        out.append((rc, g.stats()["iterations"], p, np.array(g.history())))
    assert out[0][0] == out[1][0] and out[0][1] == out[1][1]
    assert torch.equal(out[0][2], out[1][2])
    assert np.array_equal(out[0][3], out[1][3])


def test_coarse_level_constants_and_a_moving_body():
    """Level 1 of a 256^3-class grid is TMA-fed too; its constant is 2 = (2*2)/2 (reading O5 applied
    to ones).  Rewriting the coefficients (a body that moved) re-marks the bricks."""
    wl = _ones_with_bodies((256, 128, 64), (0, 0, 0), 7)
    on = make_gpu(wl, tma_min_cells=0, uniform_tiles=1)
    off = make_gpu(wl, tma_min_cells=0, uniform_tiles=0)
    try:
        L1 = on.level_coeffs(1)
        vals, counts = torch.unique(L1, return_counts=True)
        assert float(vals[counts.argmax()]) == 2.0
        n1, _ = on.level_shape(1)
        rng = np.random.default_rng(8)
        p1 = dev(rng.standard_normal((n1[2], n1[1], n1[0])))
        b1 = dev(rng.standard_normal((n1[2], n1[1], n1[0])))
        assert torch.equal(on.op_smooth(1, p1.clone(), b1, omega=0.875, nsweeps=2),
                           off.op_smooth(1, p1.clone(), b1, omega=0.875, nsweeps=2))
        assert torch.equal(on.op_residual_restrict(1, p1, b1), off.op_residual_restrict(1, p1, b1))
        # the body moves: same array rewritten in place, bricks re-marked by gmg_set_coeffs
        Ldev_on, Ldev_off = dev(wl.L), dev(wl.L)
        on.set_coeffs(Ldev_on)
        off.set_coeffs(Ldev_off)
        wl2 = _ones_with_bodies((256, 128, 64), (0, 0, 0), 9)
        for Ld, g in ((Ldev_on, on), (Ldev_off, off)):
            Ld.copy_(dev(wl2.L))
            g.set_coeffs(Ld)
        res = []
        for g in (on, off):
            p = torch.zeros(wl2.z.shape, dtype=torch.float32, device="cuda")
            rc = g.solve(p, dev(wl2.z), tol=1e-5, maxiter=50)
            res.append((rc, g.stats()["iterations"], p))
        assert res[0][0] == res[1][0] == gmg.OK and res[0][1] == res[1][1]
        assert torch.equal(res[0][2], res[1][2])
    finally:
        on.close()
        off.close()


def test_pressure_steps_with_a_moving_body_bit_identical():
    """gmg_pressure_step does not read the tile counts back between the coefficient update and the
    solve: the kernels of the remaining tiles (k_rb_sweep_bulk, k_prolong_tiles) launch the whole grid
    and bound themselves by the device-side list length, and the fold hint is the one of the last
    count.  Four steps with a body that moves, warm-started: u, p and the cycle counts of every step
    are those of the run without uniform tiles."""
    n, bc = (256, 128, 64), (0, 0, 0)
    fields = [_ones_with_bodies(n, bc, 20 + s, nblobs=1) for s in range(4)]
    rng = np.random.default_rng(21)
    u0 = rng.standard_normal((3, n[2], n[1], n[0])).astype(np.float32)
    runs = []
    for uni in (1, 0):
        g = gmg.GMG(n, bc, tma_min_cells=0, uniform_tiles=uni)
        try:
            p = torch.zeros((n[2], n[1], n[0]), dtype=torch.float32, device="cuda")
            L = dev(fields[0].L)
            out = []
            for s, wl in enumerate(fields):
                L.copy_(dev(wl.L))              # the body moves: the same array, rewritten in place
                u = dev(u0 * (1.0 + 0.1 * s))
                rc = g.pressure_step(L, u, p, tol=1e-5, maxiter=60)
                torch.cuda.synchronize()
                st = g.stats()
                out.append((rc, st["iterations"], u.clone(), p.clone(), st["uniform_fraction"]))
            if uni:
                assert out[-1][4] > 0.5, out[-1][4]
                assert "prolong=in-sweep" in g.describe_plan().split("\n")[0]
            runs.append(out)
        finally:
            g.close()
    for a, b in zip(*runs):
        assert a[:2] == b[:2] and a[0] == gmg.OK
        assert torch.equal(a[2], b[2]) and torch.equal(a[3], b[3])


@pytest.mark.parametrize("nu_pre,nu_post", [(1, 3), (3, 2), (2, 1), (4, 4), (0, 2)])
def test_other_sweep_counts_bit_identical(nu_pre, nu_post):
    """Odd and larger sweep counts take other routes through smooth(): pairs of fused sweeps, a last
    sweep as two half-sweeps, the prolongation folded in only where a pair follows it."""
    wl = _ones_with_bodies((256, 128, 64), (0, 0, 0), 6, nblobs=1)
    on = make_gpu(wl, tma_min_cells=0, uniform_tiles=1, nu_pre=nu_pre, nu_post=nu_post)
    off = make_gpu(wl, tma_min_cells=0, uniform_tiles=0, nu_pre=nu_pre, nu_post=nu_post)
    try:
        p, b = _fields(wl, 66)
        for sym in (False, True):
            assert torch.equal(on.op_vcycle(p.clone(), b, omega=0.9375, symmetric=sym),
                               off.op_vcycle(p.clone(), b, omega=0.9375, symmetric=sym))
        out = []
        for g in (on, off):
            x = torch.zeros(wl.z.shape, dtype=torch.float32, device="cuda")
            rc = g.solve(x, dev(wl.z), tol=1e-5, maxiter=80)
            out.append((rc, g.stats()["iterations"], x))
        assert out[0][:2] == out[1][:2] and torch.equal(out[0][2], out[1][2])
    finally:
        on.close()
        off.close()
