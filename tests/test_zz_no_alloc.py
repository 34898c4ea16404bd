"""gmg_residual_norm2_noalloc (include/gmg.h): the entry point that allocates nothing -- the
stopping-test norm with its reduction scratch in a static device array.  Collected LAST on purpose
(the run is `pytest -x`): a failure here must not hide the parity tests.

The gpu tests compare it with the existing path (gmg_op_residual + gmg_op_norm2 of a context) on two
calls in a row, and with the FP64 oracle; they hold in a fresh process and after the other tests."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2607_07687_b200 import gmg

# Both paths accumulate the SAME float32 residuals (one arithmetic order, stencil.cuh) in FP64; only
# the order of the FP64 additions differs (grid-stride blocks here, float4 rows there).
TOL_SAME_R = 1e-12
I3 = C.c_int * 3


def _call_raw(n, bc, ptrs, cap=512):
    err = C.create_string_buffer(cap)
    rc = gmg.lib.gmg_residual_norm2_noalloc(n[0], n[1], n[2], I3(*bc), *[C.c_void_p(p) for p in ptrs],
                                            None, err, cap)
    return rc, err.value.decode()


def test_sizes_beyond_the_static_scratch_are_refused_before_any_cuda_call():
    """No GPU needed: validation comes first.  257 x 256 x 256 > GMG_NOALLOC_MAX_CELLS = 256^3."""
    assert gmg.NOALLOC_MAX_CELLS == 256 ** 3
    fake = [256, 256, 256, 256]          # non-null, aligned; never dereferenced
    rc, msg = _call_raw((257, 256, 256), (0, 0, 0), fake)
    assert rc == gmg.EINVAL
    assert "GMG_NOALLOC_MAX_CELLS" in msg and "16777216" in msg and str(257 * 256 * 256) in msg
    rc, msg = _call_raw((4096, 4096, 4096), (1, 1, 1), fake)        # would overflow an int
    assert rc == gmg.EINVAL and "GMG_NOALLOC_MAX_CELLS" in msg
    rc, msg = _call_raw((8, 8, 8), (0, 0, 0), [0, 256, 256, 256])
    assert rc == gmg.EINVAL and "null" in msg
    rc, msg = _call_raw((8, 0, 8), (0, 0, 0), fake)
    assert rc == gmg.EINVAL and "extents" in msg
    rc, msg = _call_raw((8, 8, 8), (0, 2, 0), fake)
    assert rc == gmg.EINVAL and "bc[1]" in msg
    rc, msg = _call_raw((8, 8, 8), (0, 0, 0), [256, 258, 256, 256])
    assert rc == gmg.EINVAL and "aligned" in msg
    rc, msg = _call_raw((8, 8, 8), (0, 0, 0), [256, 256, 256, 260])
    assert rc == gmg.EINVAL and "aligned" in msg
    # a short / absent message buffer is fine
    err = C.create_string_buffer(8)
    rc = gmg.lib.gmg_residual_norm2_noalloc(257, 256, 256, I3(0, 0, 0), *[C.c_void_p(256)] * 4, None, err, 8)
    assert rc == gmg.EINVAL and len(err.value) == 7
    assert gmg.lib.gmg_residual_norm2_noalloc(257, 256, 256, I3(0, 0, 0), *[C.c_void_p(256)] * 4, None, None, 0) == gmg.EINVAL


CASES = [((96, 40, 24), (1, 0, 1), 5),       # 45 blocks; walls in x and z, periodic y; a solid blob
         ((130, 17, 9), (1, 1, 1), 6),       # ragged: odd extents, last block partly empty
         ((256, 128, 64), (0, 0, 0), 7)]     # 1024 blocks, all periodic


@pytest.mark.gpu
@pytest.mark.parametrize("n,bc,seed", CASES)
def test_matches_the_existing_path_on_two_calls_in_a_row(n, bc, seed):
    import oracle
    from gpu_util import TOL_OP, dev, random_workload

    wl = random_workload(n, bc, seed=seed, zero_frac=0.1)
    rng = np.random.default_rng(100 + seed)
    shape = wl.z.shape
    Ld = dev(wl.L)
    b = dev(wl.z)
    ps = [dev(rng.standard_normal(shape)), dev(rng.standard_normal(shape) * 3.0 + 1.0)]

    # existing path: a context's residual kernel + its norm reduction
    g = gmg.GMG(wl.n, wl.bc)
    g.set_coeffs(Ld)
    want = [g.op_norm2(0, g.op_residual(0, p, b)) for p in ps]
    g.close()
    assert want[0] > 0 and want[1] > 0 and abs(want[0] - want[1]) > 1e-3 * want[0]

    out = [torch.full((1,), -1.0, dtype=torch.float64, device="cuda") for _ in range(4)]
    torch.cuda.synchronize()
    # first call on this device: looks the scratch address up
    gmg.residual_norm2_noalloc(wl.n, wl.bc, Ld, ps[0], b, out[0])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # ... then back to back on one stream, different inputs: the array still holds the last call's
    # partials and ticket
    gmg.residual_norm2_noalloc(wl.n, wl.bc, Ld, ps[1], b, out[1])
    gmg.residual_norm2_noalloc(wl.n, wl.bc, Ld, ps[0], b, out[2])
    gmg.residual_norm2_noalloc(wl.n, wl.bc, Ld, ps[1], b, out[3])
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    got = [float(o.item()) for o in out]
    for k, w in zip(got, [want[0], want[1], want[0], want[1]]):
        assert abs(k - w) <= TOL_SAME_R * w, (got, want)
    assert got[0] == got[2] and got[1] == got[3]          # deterministic, nothing left over
    assert free1 >= free0, "device memory shrank across calls that must not allocate"

    # and the oracle (FP64 operator): the tolerance of single operator applications
    for p, k in zip(ps, got[:2]):
        r = oracle.residual(wl.L, wl.bc, p.cpu().numpy().astype(np.float64), wl.z)
        ref = float(np.sqrt(np.sum(np.asarray(r, dtype=np.float64) ** 2)))
        assert abs(k - ref) <= TOL_OP * ref, (k, ref)


@pytest.mark.gpu
def test_the_limit_itself_runs_twice():
    """The largest grid the scratch covers (256^3: 8192 partials), constant coefficients, p = 0:
    every cell active, r = b, so the norm is sqrt(sum b^2) in closed form.  Run twice."""
    n = (256, 256, 256)
    N = n[0] * n[1] * n[2]
    L = torch.ones((3,) + n, dtype=torch.float32, device="cuda")
    p = torch.zeros(n, dtype=torch.float32, device="cuda")
    b = torch.full(n, 0.5, dtype=torch.float32, device="cuda")
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    gmg.residual_norm2_noalloc(n, (0, 0, 0), L, p, b, out[0:1])
    gmg.residual_norm2_noalloc(n, (0, 0, 0), L, p, b, out[1:2])
    torch.cuda.synchronize()
    want = float(np.sqrt(0.25 * N))
    assert out[0].item() == want and out[1].item() == want
    with pytest.raises(gmg.GMGError) as e:
        gmg.residual_norm2_noalloc((256, 256, 258), (0, 0, 0), L, p, b, out[0:1])
    assert e.value.code == gmg.EINVAL and "GMG_NOALLOC_MAX_CELLS" in str(e.value)
