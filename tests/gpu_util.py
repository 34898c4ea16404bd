"""Helpers shared by the -m gpu parity tests: build a GMG context from a Workload, move
arrays, compare with the FP64 oracle.  Test infrastructure only."""
import numpy as np
import torch

import oracle
from paper_2607_07687_b200 import workloads as W

# Tolerances (BASELINE.json:north_star).
TOL_OP = 1e-5      # relative L-infinity, single operator applications
TOL_P = 1e-4       # final pressure, relative L2 (mean over active cells removed)


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def host(t):
    return t.detach().cpu().numpy().astype(np.float64)


def rel_linf(a, b):
    """max|a-b| / max|b| over the whole array."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = np.max(np.abs(b))
    if den == 0.0:
        return float(np.max(np.abs(a)))
    return float(np.max(np.abs(a - b)) / den)


def rel_l2_demeaned(a, b, act):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    a = np.where(act, a - a[act].mean(), 0.0)
    b = np.where(act, b - b[act].mean(), 0.0)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def make_gpu(wl, **params):
    from paper_2607_07687_b200 import gmg
    g = gmg.GMG(wl.n, wl.bc, **params)
    g.set_coeffs(dev(wl.L))
    return g


def make_oracle(wl, **kw):
    n_min = kw.pop("n_min", 4)
    iso = kw.pop("iso", False)
    h = oracle.Hierarchy(wl.n, wl.bc, wl.L, n_min=n_min, iso=iso)
    if kw:
        h.set_params(**kw)
    return h


def random_workload(n, bc, seed, zero_frac=0.15, blob=True):
    """Random coefficients in [0,1) with exact zeros (isolated faces and one solid blob of
    fully inactive cells), random RHS made compatible.  Input conditioning only."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = n
    L = rng.uniform(0.0, 1.0, (3, nz, ny, nx))
    L[rng.uniform(size=L.shape) < zero_frac] = 0.0
    if blob and min(n) >= 6:
        k0, j0, i0 = nz // 3, ny // 3, nx // 3
        L[:, k0:k0 + 3, j0:j0 + 3, i0:i0 + 3] = 0.0     # interior cells of the blob are inactive
    L32 = L.astype(np.float32)
    act = W.active_mask(L32, bc)
    z = W.project_compatible(rng.standard_normal((nz, ny, nx)), act)
    return W.Workload(f"random_{nx}x{ny}x{nz}_{''.join(map(str, bc))}", tuple(n), tuple(bc), L32,
                      z.astype(np.float32), seed=seed)
