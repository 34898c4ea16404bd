"""Pins of the FP64 oracle against things OTHER than itself.

Each pin is chosen so that a plausible mistake in oracle/gmg_oracle.c (dropped term, wrong
sign or index, transposed operand, wrong face) fails at least one of them.
"""
import itertools
import os

import numpy as np
import pytest

import oracle
from paper_2607_07687_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
BCS = [(0, 0, 0), (1, 0, 0), (1, 1, 1), (1, 0, 1), (0, 1, 0)]


# --------------------------------------------------------------------------------------
# independent restatement: FACE-by-FACE scatter assembly of the dense matrix (the oracle
# gathers per cell).  A face between cells a and b with coefficient L contributes
# +L to A[a,b], A[b,a] and -L to A[a,a], A[b,b]  (flux form of div(L grad)).
# --------------------------------------------------------------------------------------
def dense_by_faces(n, bc, L):
    nx, ny, nz = n
    N = nx * ny * nz
    A = np.zeros((N, N))
    idx = lambda i, j, k: i + nx * (j + ny * k)
    for k, j, i in itertools.product(range(nz), range(ny), range(nx)):
        I = (i, j, k)
        for d in range(3):
            if I[d] == 0 and bc[d] == 1:
                continue                      # wall face: no flux, stored value ignored
            J = list(I)
            J[d] = (I[d] - 1) % n[d]
            a, b = idx(*I), idx(*J)
            if a == b:
                continue
            c = L[d, k, j, i]
            A[a, b] += c
            A[b, a] += c
            A[a, a] -= c
            A[b, b] -= c
    return A


def rand_L(rng, n, zero_frac=0.0):
    L = rng.uniform(0.0, 1.0, (3, n[2], n[1], n[0]))
    if zero_frac:
        L[rng.uniform(size=L.shape) < zero_frac] = 0.0
    return L


@pytest.mark.parametrize("bc", BCS)
def test_operator_matches_face_assembly(bc):
    rng = np.random.default_rng(1)
    n = (4, 6, 4)
    L = rand_L(rng, n, 0.2)
    A = dense_by_faces(n, bc, L)
    p = rng.standard_normal((n[2], n[1], n[0]))
    assert np.allclose(oracle.apply_A(L, bc, p).ravel(), A @ p.ravel(), rtol=0, atol=1e-13)
    assert np.allclose(oracle.diag(L, bc).ravel(), np.diag(A), rtol=0, atol=1e-14)
    # residual: b - A p on active cells, 0 where the row is empty
    L[:, 1:3, 2:4, 1:3] = 0.0
    L[0, 1:3, 2:4, 3] = 0.0; L[1, 1:3, 4, 1:3] = 0.0; L[2, 3, 2:4, 1:3] = 0.0
    A = dense_by_faces(n, bc, L)
    b = rng.standard_normal(p.shape)
    r = oracle.residual(L, bc, p, b).ravel()
    ref = np.where(np.diag(A) != 0.0, b.ravel() - A @ p.ravel(), 0.0)
    assert (np.diag(A) == 0).sum() >= 1
    assert np.allclose(r, ref, rtol=0, atol=1e-13)


def test_fourier_eigenmode_closed_form():
    vals = {}
    for line in open(os.path.join(GOLD, "eigenmode.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        vals[t[0]] = [float(x) for x in t[1:]]
    n = tuple(int(v) for v in vals["n"]); m = vals["m"]; lam_gold = vals["lambda"][0]
    th = [2 * np.pi * m[d] / n[d] for d in range(3)]
    lam = sum(2 * np.cos(t) - 2 for t in th)
    assert abs(lam - lam_gold) < 1e-10
    k, j, i = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    p = np.sin(th[0] * i + th[1] * j + th[2] * k + 0.3)
    L = np.ones((3, n[2], n[1], n[0]))
    Ap = oracle.apply_A(L, (0, 0, 0), p)
    assert np.max(np.abs(Ap - lam * p)) < 1e-12


def test_level_shapes_table():
    for line in open(os.path.join(GOLD, "level_shapes.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, bc, shapes = [s.strip() for s in line.split("|")]
        bc = tuple(int(x) for x in bc.split())
        shapes = [tuple(int(x) for x in s.split("x")) for s in shapes.split()]
        assert oracle.level_shapes(shapes[0], bc) == shapes, name
    # isotropic mode stops when the smallest direction stops
    assert oracle.level_shapes((32, 32, 16), (0, 0, 0), iso=True) == [(32, 32, 16), (16, 16, 8), (8, 8, 4)]
    # odd periodic half-extent is never produced; Neumann may go odd
    assert oracle.level_shapes((20, 20, 20), (0, 0, 0)) == [(20, 20, 20), (10, 10, 10)]
    assert oracle.level_shapes((20, 20, 20), (1, 1, 1)) == [(20, 20, 20), (10, 10, 10), (5, 5, 5)]
    assert oracle.level_shapes((20, 20, 20), (1, 0, 0)) == [(20, 20, 20), (10, 10, 10), (5, 10, 10)]


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 0, 0), (1, 1, 1)])
def test_symmetry_rowsum_definiteness_every_level(bc):
    rng = np.random.default_rng(2)
    n = (16, 8, 8)
    L32 = rand_L(rng, n, 0.1).astype(np.float32)
    H = oracle.Hierarchy(n, bc, L32)
    assert H.nlev >= 2
    for lev in range(H.nlev):
        nl, _ = H.shape(lev)
        Ll = H.L(lev)
        a = rng.standard_normal((nl[2], nl[1], nl[0])); b = rng.standard_normal(a.shape)
        Aa, Ab = oracle.apply_A(Ll, bc, a), oracle.apply_A(Ll, bc, b)
        assert abs((a * Ab).sum() - (b * Aa).sum()) < 1e-10
        assert np.max(np.abs(oracle.apply_A(Ll, bc, np.ones_like(a)))) == 0.0
        assert (a * Aa).sum() <= 0.0
        # Neumann wall planes stay zero after coarsening
        for d in range(3):
            if bc[d] == 1:
                sl = [slice(None)] * 3; sl[2 - d] = 0
                assert np.all(Ll[d][tuple(sl)] == 0.0)


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 0, 1)])
def test_half_sweep_zeroes_own_colour_and_decreases_energy(bc):
    rng = np.random.default_rng(3)
    n = (6, 4, 4)
    L = rand_L(rng, n, 0.15)
    A = dense_by_faces(n, bc, L)
    xs = rng.standard_normal(A.shape[0]); xs[np.diag(A) == 0] = 0
    b = (A @ xs).reshape(n[2], n[1], n[0])          # compatible rhs with known solution
    k, j, i = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    col = (i + j + k) % 2
    p = rng.standard_normal(b.shape)
    for colour in (0, 1):
        q = oracle.half_sweep(L, bc, p, b, 1.0, colour)
        r = oracle.residual(L, bc, q, b)
        assert np.max(np.abs(r[col == colour])) < 1e-13
        assert np.max(np.abs(r[col != colour])) > 1e-3
        assert np.array_equal(q[col != colour], p[col != colour])
    energy = lambda e: -(e.ravel() @ (A @ e.ravel()))
    for omega in (0.7, 1.0, 1.5):
        q = p.copy(); e0 = energy(q - xs.reshape(q.shape))
        for s in range(6):
            q = oracle.half_sweep(L, bc, q, b, omega, s % 2)
            e1 = energy(q - xs.reshape(q.shape))
            assert e1 <= e0 * (1 + 1e-12)
            e0 = e1
    # omega scales the update linearly
    q1 = oracle.half_sweep(L, bc, p, b, 1.0, 0); qh = oracle.half_sweep(L, bc, p, b, 0.5, 0)
    assert np.allclose(qh - p, 0.5 * (q1 - p), atol=1e-14)


@pytest.mark.parametrize("c", [(2, 2, 2), (2, 1, 1), (2, 2, 1), (1, 2, 2), (1, 1, 2)])
def test_transfer_adjoint_and_sum(c):
    rng = np.random.default_rng(4)
    nf = (8, 4, 6)
    nc = tuple(a // b for a, b in zip(nf, c))
    r = rng.standard_normal((nf[2], nf[1], nf[0])); e = rng.standard_normal((nc[2], nc[1], nc[0]))
    Rr = oracle.restrict_sum(r, c)
    Pe = oracle.prolong_add(np.zeros_like(r), e, c)
    assert abs((Rr * e).sum() - (r * Pe).sum()) < 1e-12
    assert abs(Rr.sum() - r.sum()) < 1e-12
    # brute force: parent index by integer division
    k, j, i = np.meshgrid(np.arange(nf[2]), np.arange(nf[1]), np.arange(nf[0]), indexing="ij")
    assert np.array_equal(Pe, e[k // c[2], j // c[1], i // c[0]])
    ref = np.zeros_like(e); np.add.at(ref, (k // c[2], j // c[1], i // c[0]), r)
    assert np.allclose(Rr, ref, atol=1e-13)


def test_coarse_coeffs_closed_form_uniform():
    n, bc = (32, 16, 8), (0, 0, 0)
    H = oracle.Hierarchy(n, bc, np.ones((3, 8, 16, 32), np.float32))
    C = [1, 1, 1]
    for lev in range(H.nlev):
        Ll = H.L(lev)
        for d in range(3):
            e1, e2 = (d + 1) % 3, (d + 2) % 3
            assert np.all(Ll[d] == C[e1] * C[e2] / C[d]), (lev, d)
        _, c = H.shape(lev)
        C = [a * b for a, b in zip(C, c)]
    assert H.shape(H.nlev - 1)[0] == (4, 4, 4) and tuple(H.L(3)[:, 0, 0, 0]) == (1.0, 4.0, 16.0)


@pytest.mark.parametrize("c", [(2, 2, 2), (2, 1, 1), (2, 2, 1), (1, 2, 2), (1, 1, 2)])
def test_coarse_operator_consistent_on_quadratics(c):
    """A^{l+1} q_c = R (A^l q_f) in the interior for a quadratic q sampled at cell centres."""
    nf = (8, 8, 8); bc = (1, 1, 1)
    nc = tuple(a // b for a, b in zip(nf, c))
    Lf = np.ones((3,) + nf[::-1])
    Lc = oracle.coarsen_coeffs(Lf, c)
    quad = lambda x, y, z: 0.3 * x * x - 0.7 * y * y + 0.2 * z * z + 0.5 * x * y - 0.1 * y * z + x - 2 * z
    k, j, i = np.meshgrid(*[np.arange(m) for m in nf[::-1]], indexing="ij")
    qf = quad(i + 0.5, j + 0.5, k + 0.5)
    K, J, I = np.meshgrid(*[np.arange(m) for m in nc[::-1]], indexing="ij")
    qc = quad((I + 0.5) * c[0], (J + 0.5) * c[1], (K + 0.5) * c[2])
    lhs = oracle.apply_A(Lc, bc, qc)
    rhs = oracle.restrict_sum(oracle.apply_A(Lf, bc, qf), c)
    assert np.max(np.abs((lhs - rhs)[1:-1, 1:-1, 1:-1])) < 1e-11


def _dense_solution(n, bc, L, z):
    A = dense_by_faces(n, bc, L)
    x, *_ = np.linalg.lstsq(A, z.ravel(), rcond=None)
    return x.reshape(z.shape), A


def _demean(p, act):
    return np.where(act, p - p[act].mean(), 0.0)


@pytest.mark.parametrize("solver", [oracle.GMG_RBGS, oracle.PCG, oracle.GMG_PCG, oracle.GMG_CGS])
def test_solvers_reach_dense_solution_8cubed(solver):
    rng = np.random.default_rng(5)
    n, bc = (8, 8, 8), (1, 0, 1)
    L32 = rng.uniform(0, 1, (3, 8, 8, 8)).astype(np.float32)
    Le = W.effective_L(L32, bc)
    act = W.active_mask(L32, bc)
    z = W.project_compatible(rng.standard_normal((8, 8, 8)), act)
    xs, A = _dense_solution(n, bc, Le, z)
    assert np.linalg.norm(A @ xs.ravel() - z.ravel()) < 1e-10
    H = oracle.Hierarchy(n, bc, L32)
    out = H.solve(solver, z, tol=1e-10, maxiter=400)
    assert out["status"] == 0
    err = np.linalg.norm(_demean(out["p"], act) - _demean(xs, act)) / np.linalg.norm(_demean(xs, act))
    assert err < 1e-8, err
    assert out["true_res"] <= 1.001e-10 or solver != oracle.GMG_RBGS
    assert np.all(np.diff(out["history"]) < 0) or solver != oracle.GMG_RBGS


def test_invariants_and_config0_history():
    w = W.config0()
    H = oracle.Hierarchy(w.n, w.bc, w.L)
    z = w.z.astype(np.float64)
    out = H.solve(oracle.GMG_RBGS, z, tol=w.tol, maxiter=w.maxiter)
    # textbook cell-centred V(2,2) on L=1 periodic: fast, omega stays 1 (3 cycles)
    assert out["iterations"] == 3 and out["status"] == 0
    assert np.all(out["omegas"] == 1.0) and H.omega == 1.0
    h = out["history"]
    assert abs(h[0] - 1.0) < 1e-12 and 5e-3 < h[1] < 5e-2 and h[3] < 1e-4
    # sum(r_k) = sum(z) for every iterate (column sums of A vanish)
    r = oracle.residual(w.L, w.bc, out["p"], z)
    assert abs(r.sum() - z.sum()) < 1e-9
    # k-cycle prefix property: maxiter=k, tol=0 gives the same iterate sequence
    H2 = oracle.Hierarchy(w.n, w.bc, w.L)
    o2 = H2.solve(oracle.GMG_RBGS, z, tol=0.0, maxiter=2)
    assert o2["iterations"] == 2 and o2["status"] == 1
    assert np.allclose(o2["history"], h[:3], rtol=1e-12)
    # zero rhs: 0 iterations, p untouched
    o3 = H2.solve(oracle.GMG_RBGS, np.zeros_like(z), p0=np.ones_like(z))
    assert o3["iterations"] == 0 and np.all(o3["p"] == 1.0)


def test_adaptive_omega_follows_dyadic_rule():
    """O8 on an under-smoothed V(1,0) jellyfish case (p=4) that grows AND decays:
    growth -> -1/8 (floor 1/2), decay -> +1/32 (cap 1); no rollback of the iterate."""
    w = W.config3(4)
    H = oracle.Hierarchy(w.n, w.bc, w.L)
    H.set_params(nu1=1, nu2=0)
    out = H.solve(oracle.GMG_RBGS, w.z.astype(np.float64), tol=0.0, maxiter=8)
    h, om = out["history"], out["omegas"]
    assert out["iterations"] == 8 and out["status"] == 1
    d = np.diff(h)
    assert np.any(d > 0) and np.any(d <= 0), "this case must exercise both branches"
    w_ = 1.0                                            # the rule restated, fed by the history
    for k in range(out["iterations"]):
        assert om[k] == w_
        w_ = max(0.5, w_ - 0.125) if h[k + 1] > h[k] else min(1.0, w_ + 0.03125)
    assert H.omega == w_ == 0.5
    # adaptive off: omega never moves
    H2 = oracle.Hierarchy(w.n, w.bc, w.L)
    H2.set_params(nu1=1, nu2=0, adaptive=False)
    o2 = H2.solve(oracle.GMG_RBGS, w.z.astype(np.float64), tol=0.0, maxiter=3)
    assert np.all(o2["omegas"] == 1.0) and H2.omega == 1.0


def test_pcg_properties_and_ordering():
    w = W.config0()
    H = oracle.Hierarchy(w.n, w.bc, w.L)
    z = w.z.astype(np.float64)
    pcg = H.solve(oracle.PCG, z, tol=1e-4, maxiter=500)
    mg = H.solve(oracle.GMG_PCG, z, tol=1e-4, maxiter=50)
    assert pcg["status"] == 0 and mg["status"] == 0
    assert mg["iterations"] <= 4 < 20 < pcg["iterations"] < 120
    assert abs(pcg["true_res"] - pcg["history"][-1]) < 1e-8


# --------------------------------------------------------------------------------------
# N2: the paper's own "GMG-PCG" = GMG with a Jacobi-PCG smoother (reading O12)
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(1, 0, 1), (0, 0, 0), (1, 1, 1)])
@pytest.mark.parametrize("m", [1, 2, 4])
def test_cg_smoother_is_the_krylov_energy_minimiser(bc, m):
    """m preconditioned CG iterations from x0 give THE minimiser of the energy
    phi(x) = 1/2 x'(-A)x + x'b over x0 + span{v, Tv, .., T^(m-1)v}, v = M^-1 r0, T = M^-1 A
    (the textbook characterisation of PCG), computed here densely from the face-assembled A."""
    rng = np.random.default_rng(100 + m)
    n = (8, 6, 4)
    L32 = rand_L(rng, n, zero_frac=0.15).astype(np.float32)
    L32[:, 1:3, 2:4, 3:5] = 0.0                       # a solid block: inactive cells
    Le = W.effective_L(L32, bc)
    act = W.active_mask(L32, bc)
    assert not act.all()
    A = dense_by_faces(n, bc, Le)
    Dg = np.diag(A).copy()
    Minv = np.where(Dg != 0.0, 1.0 / np.where(Dg != 0.0, Dg, 1.0), 0.0)
    b = W.project_compatible(rng.standard_normal((n[2], n[1], n[0])), act)
    x0 = rng.standard_normal(b.shape)
    r0 = np.where(act.ravel(), b.ravel() - A @ x0.ravel(), 0.0)
    v = Minv * r0
    K = [v]
    for _ in range(m - 1):
        K.append(Minv * (A @ K[-1]))
    K = np.stack(K, axis=1)
    y = np.linalg.solve(K.T @ A @ K, K.T @ r0)
    x_ref = x0.ravel() + K @ y
    H = oracle.Hierarchy(n, bc, L32, n_min=64)        # one level
    assert H.nlev == 1
    x = H.level_cg_smooth(0, x0, b, m)
    scale = np.abs(x_ref - x0.ravel()).max()
    assert np.abs(x.ravel() - x_ref).max() < 1e-9 * max(scale, 1.0)
    assert np.array_equal(x[~act], x0[~act])          # inactive cells untouched
    # energy of the error never increases with more iterations
    xs, _ = _dense_solution(n, bc, Le, b)
    def energy(xx):
        e = (xx - xs).ravel()
        return float(-(e @ (A @ e)))
    e_prev = energy(x0)
    for mm in range(1, m + 1):
        e_now = energy(H.level_cg_smooth(0, x0, b, mm))
        assert e_now <= e_prev * (1 + 1e-12)
        e_prev = e_now


def test_cg_smoother_guards():
    """Zero residual, zero count, and a long run on a singular 4^3 level stay put / finite."""
    rng = np.random.default_rng(7)
    n, bc = (4, 4, 4), (0, 0, 0)
    L32 = np.ones((3, 4, 4, 4), dtype=np.float32)
    H = oracle.Hierarchy(n, bc, L32)
    assert H.nlev == 1
    x0 = rng.standard_normal((4, 4, 4))
    b = oracle.apply_A(L32, bc, x0)
    assert np.array_equal(H.level_cg_smooth(0, x0, b, 5), x0)        # r0 = 0: nothing moves
    b2 = rng.standard_normal((4, 4, 4))
    b2 -= b2.mean()
    assert np.array_equal(H.level_cg_smooth(0, x0, b2, 0), x0)       # m = 0
    x = H.level_cg_smooth(0, np.zeros_like(b2), b2, 500)             # far past convergence
    assert np.all(np.isfinite(x))
    r = oracle.residual(L32, bc, x, b2)
    assert np.linalg.norm(r) < 1e-4 * np.linalg.norm(b2)
    # an inconsistent right-hand side (non-zero mean on a singular level) must not blow up either
    x = H.level_cg_smooth(0, np.zeros_like(b2), b2 + 1e-7, 500)
    assert np.all(np.isfinite(x)) and np.abs(x).max() < 1e3


def test_gmg_cgs_invariants_and_cycle_structure():
    w = W.config0()
    H = oracle.Hierarchy(w.n, w.bc, w.L)
    z = w.z.astype(np.float64)
    out = H.solve(oracle.GMG_CGS, z, tol=w.tol, maxiter=w.maxiter)
    assert out["status"] == 0 and 1 <= out["iterations"] <= 12
    h = out["history"]
    assert abs(h[0] - 1.0) < 1e-12 and h[-1] <= w.tol
    r = oracle.residual(w.L, w.bc, out["p"], z)
    assert abs(r.sum() - z.sum()) < 1e-9
    # prefix property and the cycle as a composition of its pinned parts (one 2-level case)
    o2 = oracle.Hierarchy(w.n, w.bc, w.L).solve(oracle.GMG_CGS, z, tol=0.0, maxiter=1)
    assert np.allclose(o2["history"], h[:2], rtol=1e-12)
    n, bc = (8, 8, 4), (1, 0, 1)
    rng = np.random.default_rng(3)
    L32 = rng.uniform(0, 1, (3, 4, 8, 8)).astype(np.float32)
    H2 = oracle.Hierarchy(n, bc, L32)
    assert H2.nlev == 2
    H2.set_params(nu1=2, nu2=3, nuc=5)
    b = W.project_compatible(rng.standard_normal((4, 8, 8)), W.active_mask(L32, bc))
    x0 = rng.standard_normal(b.shape)
    _, c0 = H2.shape(0)
    x = H2.level_cg_smooth(0, x0, b, 2)
    bc_ = oracle.restrict_sum(H2.level_residual(0, x, b), c0)
    e = H2.level_cg_smooth(1, np.zeros_like(bc_), bc_, 5)
    x = H2.level_cg_smooth(0, oracle.prolong_add(x, e, c0), b, 3)
    assert np.allclose(H2.vcycle_cgs(x0, b), x, rtol=0, atol=1e-13)
    # zero rhs: 0 iterations, p untouched
    o3 = H.solve(oracle.GMG_CGS, np.zeros_like(z), p0=np.ones_like(z))
    assert o3["iterations"] == 0 and np.all(o3["p"] == 1.0)


# --------------------------------------------------------------------------------------
# N1: divergence / projection either side of the solve
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", BCS)
def test_projection_identity_ties_to_the_pinned_operator(bc):
    """div(u - L grad p) = div(u) - A p for any u, p, L, boundary mix (A is pinned above)."""
    rng = np.random.default_rng(21)
    n = (6, 4, 8)
    L = rand_L(rng, n, 0.2)
    p = rng.standard_normal((n[2], n[1], n[0]))
    u = rng.standard_normal((3, n[2], n[1], n[0]))
    wall = (0.3, -0.7, 1.1)
    lhs = oracle.divergence(oracle.project(L, bc, p, u), bc, wall)
    rhs = oracle.divergence(u, bc, wall) - oracle.apply_A(L, bc, p)
    assert np.max(np.abs(lhs - rhs)) < 1e-13


def test_divergence_closed_forms():
    n = (5, 6, 4)
    bc = (1, 1, 1)
    # u_d = a_d * (lower-face coordinate): exact divergence a_x + a_y + a_z in every cell, the
    # upper wall carrying a_d * n_d
    a = (0.5, -1.25, 2.0)
    u = np.zeros((3, n[2], n[1], n[0]))
    u[0] += a[0] * np.arange(n[0])[None, None, :]
    u[1] += a[1] * np.arange(n[1])[None, :, None]
    u[2] += a[2] * np.arange(n[2])[:, None, None]
    z = oracle.divergence(u, bc, tuple(a[d] * n[d] for d in range(3)))
    assert np.allclose(z, sum(a), atol=1e-14)
    # discrete Gauss theorem: sum(z) = net outflow through the walls; periodic axes contribute 0
    rng = np.random.default_rng(2)
    u = rng.standard_normal((3, n[2], n[1], n[0]))
    wall = (0.2, 0.4, -0.1)
    for bcm in [(1, 1, 1), (0 if n[0] % 2 == 0 else 1, 1, 0)]:
        z = oracle.divergence(u, bcm, wall)
        flux = 0.0
        if bcm[0] == 1:
            flux += wall[0] * n[1] * n[2] - u[0][:, :, 0].sum()
        if bcm[1] == 1:
            flux += wall[1] * n[0] * n[2] - u[1][:, 0, :].sum()
        if bcm[2] == 1:
            flux += wall[2] * n[0] * n[1] - u[2][0, :, :].sum()
        assert abs(z.sum() - flux) < 1e-12


def test_projection_closed_form_and_wall_faces():
    n = (6, 4, 4)
    L = np.ones((3, n[2], n[1], n[0]))
    p = 0.75 * (np.arange(n[0]) + 0.5)[None, None, :] * np.ones((n[2], n[1], 1))   # slope 0.75 in x
    u = np.zeros((3, n[2], n[1], n[0]))
    out = oracle.project(L, (1, 0, 0), p, u)
    assert np.allclose(out[0][:, :, 1:], -0.75) and np.all(out[0][:, :, 0] == 0.0)   # wall untouched
    assert np.all(out[1] == 0.0) and np.all(out[2] == 0.0)
    out = oracle.project(L, (0, 0, 0), p, u)                                          # periodic seam
    assert np.allclose(out[0][:, :, 0], -(p[0, 0, 0] - p[0, 0, -1]))


def test_projected_field_is_divergence_free_after_an_exact_solve():
    rng = np.random.default_rng(8)
    n, bc = (8, 8, 8), (1, 0, 1)
    L = rand_L(rng, n, 0.1)
    u = rng.standard_normal((3, n[2], n[1], n[0])) * W.effective_L(L, bc)
    for d in range(3):
        if bc[d] == 1:
            sl = [slice(None)] * 3
            sl[2 - d] = 0
            u[d][tuple(sl)] = 0.0
    z = oracle.divergence(u, bc)
    A = dense_by_faces(n, bc, L)
    p = np.linalg.lstsq(A, z.ravel(), rcond=None)[0].reshape(z.shape)
    assert np.linalg.norm(A @ p.ravel() - z.ravel()) < 1e-9 * np.linalg.norm(z)      # z compatible
    div_after = oracle.divergence(oracle.project(L, bc, p, u), bc)
    assert np.max(np.abs(div_after)) < 1e-9


# --------------------------------------------------------------------------------------
# 2-D mode: an nx x ny x 1 grid with Neumann z (Fig. 2 left)
# --------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(1, 0, 1), (0, 0, 1), (1, 1, 1)])
def test_2d_grid_operator_is_the_five_point_face_assembly(bc):
    rng = np.random.default_rng(21)
    n = (8, 6, 1)
    L = rand_L(rng, n, zero_frac=0.2)
    A = dense_by_faces(n, bc, L)
    # the z coefficients must not matter at all: a five-point operator
    A2 = dense_by_faces(n, bc, np.stack([L[0], L[1], rng.uniform(0, 1, L[2].shape)]))
    assert np.array_equal(A, A2)
    assert np.max(np.count_nonzero(A, axis=1)) <= 5
    p = rng.standard_normal((1, 6, 8))
    assert np.allclose(oracle.apply_A(L, bc, p).ravel(), A @ p.ravel(), atol=1e-13)
    assert np.allclose(oracle.diag(L, bc).ravel(), np.diag(A), atol=1e-13)


def test_2d_level_shapes_and_dense_solution():
    assert oracle.level_shapes((64, 16, 1), (1, 0, 1)) == [(64, 16, 1), (32, 8, 1), (16, 4, 1), (8, 4, 1), (4, 4, 1)]
    # isotropic = both in-plane directions or stop; the extent-1 axis has nothing to coarsen
    assert oracle.level_shapes((64, 16, 1), (1, 0, 1), iso=True) == [(64, 16, 1), (32, 8, 1), (16, 4, 1)]
    rng = np.random.default_rng(22)
    n, bc = (16, 8, 1), (1, 0, 1)
    L32 = rng.uniform(0.1, 1, (3, 1, 8, 16)).astype(np.float32)
    Le = W.effective_L(L32, bc)
    act = W.active_mask(L32, bc)
    z = W.project_compatible(rng.standard_normal((1, 8, 16)), act)
    xs, A = _dense_solution(n, bc, Le, z)
    for solver in (oracle.GMG_RBGS, oracle.PCG, oracle.GMG_PCG, oracle.GMG_CGS):
        H = oracle.Hierarchy(n, bc, L32)
        assert H.nlev == 3
        out = H.solve(solver, z, tol=1e-10, maxiter=400)
        assert out["status"] == 0, solver
        err = np.linalg.norm(_demean(out["p"], act) - _demean(xs, act)) / np.linalg.norm(_demean(xs, act))
        assert err < 1e-8, (solver, err)


# --------------------------------------------------------------------------------------
# Round-2 pins: parts that mutation testing of a copy of gmg_oracle.c showed unpinned
# (VERDICT r1 "What's weak" 1).  Each names the mutation it turns red.
# --------------------------------------------------------------------------------------
def _compose_rbgs_cycle(H, x0, b, nu1, nu2, nuc, omega, sym):
    """Reading O7 / O11 written out from the single-operator calls that are pinned on their own
    (half_sweep <- own-colour residual 0; residual <- face assembly; restrict/prolong <- brute
    force), with every colour order spelt explicitly.  2-level hierarchies only."""
    assert H.nlev == 2
    (n0, c0), (n1, _) = H.shape(0), H.shape(1)
    L0, L1, bc = H.L(0), H.L(1), H.bc
    RED, BLACK = 0, 1

    def sweep(L, x, rhs, first):
        x = oracle.half_sweep(L, bc, x, rhs, omega, first)
        return oracle.half_sweep(L, bc, x, rhs, omega, 1 - first)

    x = x0
    for _ in range(nu1):                                   # pre-smoothing: red -> black
        x = sweep(L0, x, b, RED)
    bc1 = oracle.restrict_sum(oracle.residual(L0, bc, x, b), c0)
    e = np.zeros_like(bc1)                                 # coarse unknown starts at 0 (O6)
    if not sym:
        for _ in range(nuc):                               # coarsest: nu_c sweeps red -> black
            e = sweep(L1, e, bc1, RED)
    else:
        for _ in range(nuc // 2):                          # O11: nu_c/2 red -> black ...
            e = sweep(L1, e, bc1, RED)
        for _ in range(nuc // 2):                          # ... then nu_c/2 black -> red
            e = sweep(L1, e, bc1, BLACK)
    x = oracle.prolong_add(x, e, c0)
    for _ in range(nu2):                                   # post: red -> black (O7) / black -> red (O11)
        x = sweep(L0, x, b, BLACK if sym else RED)
    return x


@pytest.mark.parametrize("sym", [False, True])
@pytest.mark.parametrize("n,bc", [((8, 8, 4), (1, 0, 1)), ((8, 4, 8), (0, 0, 0))])
def test_rbgs_cycle_is_the_composition_of_its_pinned_parts(n, bc, sym):
    """Fails: nu_c replaced by a constant, nu1/nu2 off by one, a wrong colour order in the pre-,
    post- or coarsest sweeps of either variant (gmg_oracle.c vcycle_rec)."""
    rng = np.random.default_rng(31)
    L32 = rand_L(rng, n, 0.1).astype(np.float32)
    H = oracle.Hierarchy(n, bc, L32, n_min=4)
    assert H.nlev == 2
    nu1, nu2, nuc = 2, 3, (6 if sym else 5)
    H.set_params(nu1=nu1, nu2=nu2, nuc=nuc)
    b = rng.standard_normal((n[2], n[1], n[0]))
    x0 = rng.standard_normal(b.shape)
    for omega in (1.0, 0.75):
        ref = _compose_rbgs_cycle(H, x0, b, nu1, nu2, nuc, omega, sym)
        got = H.vcycle(x0, b, omega=omega, sym=sym)
        assert np.allclose(got, ref, rtol=0, atol=1e-12)
        # the test must be able to tell the variants apart
        other = _compose_rbgs_cycle(H, x0, b, nu1, nu2, nuc + (2 if sym else 1), omega, sym)
        assert np.abs(other - ref).max() > 1e-6
        flip = _compose_rbgs_cycle(H, x0, b, nu1, nu2, 6, omega, not sym)
        assert np.abs(flip - ref).max() > 1e-6


@pytest.mark.parametrize("bc", [(1, 0, 1), (0, 0, 0), (1, 1, 1)])
def test_symmetric_cycle_is_self_adjoint(bc):
    """O11 needs B (one symmetric cycle from a zero guess) self-adjoint: <a, B b> = <b, B a>.
    The plain cycle (post-sweeps red->black) is NOT, and neither is a symmetric cycle whose
    coarsest second half is not reversed (fails that mutation of gmg_oracle.c vcycle_rec)."""
    rng = np.random.default_rng(32)
    n = (8, 8, 8)
    L32 = rand_L(rng, n, 0.1).astype(np.float32)
    H = oracle.Hierarchy(n, bc, L32)
    assert H.nlev == 2
    H.set_params(nu1=2, nu2=2, nuc=2)
    # CG applies B to residuals, which are 0 on inactive cells (O9); the prolongation also
    # writes the (never read) unknowns of inactive cells, so B is self-adjoint on the active ones
    act = W.active_mask(L32, bc)
    a = rng.standard_normal((8, 8, 8)) * act; b = rng.standard_normal(a.shape) * act
    zero = np.zeros_like(a)
    Ba, Bb = H.vcycle(zero, a, sym=True), H.vcycle(zero, b, sym=True)
    scale = abs((a * Bb).sum())
    assert abs((a * Bb).sum() - (b * Ba).sum()) < 1e-12 * max(scale, 1.0)
    Na, Nb = H.vcycle(zero, a, sym=False), H.vcycle(zero, b, sym=False)
    assert abs((a * Nb).sum() - (b * Na).sum()) > 1e-6 * max(scale, 1.0)
    # three levels, default counts: still self-adjoint
    L3 = rand_L(rng, (16, 8, 8), 0.1).astype(np.float32)
    L3[:, 2:4, 2:4, 5:8] = 0.0                          # with a solid block
    H3 = oracle.Hierarchy((16, 8, 8), bc, L3)
    assert H3.nlev == 3
    act = W.active_mask(L3, bc)
    assert not act.all()
    a = rng.standard_normal((8, 8, 16)) * act; b = rng.standard_normal(a.shape) * act
    zero = np.zeros_like(a)
    Ba, Bb = H3.vcycle(zero, a, sym=True), H3.vcycle(zero, b, sym=True)
    assert abs((a * Bb).sum() - (b * Ba).sum()) < 1e-12 * max(abs((a * Bb).sum()), 1.0)


@pytest.mark.parametrize("c", [(2, 2, 2), (2, 1, 1), (2, 2, 1), (1, 2, 2), (1, 1, 2)])
@pytest.mark.parametrize("d", [0, 1, 2])
def test_coarse_coefficients_conserve_the_flux_of_linear_fields(c, d):
    """O5 on HETEROGENEOUS coefficients.  For q = x_d (linear) the fine operator gives the
    difference of the two d-face coefficients of a cell; summed over the children of a coarse
    cell the inner faces telescope and what is left is the sum over the fine faces tiling the
    coarse cell's two d-faces.  The coarse operator on the same field (coarse spacing c_d) gives
    c_d * (L^c_hi - L^c_lo).  Both agree for every random L iff L^c = (1/c_d) * sum over exactly
    the tiling fine faces.  With walls on every axis the wall faces carry 0 on both levels, so the
    identity holds in EVERY cell; with periodic axes away from the seam of q.  Fails: a fine
    face summed twice or missed, a wrong child plane, the 1/c_d factor dropped."""
    rng = np.random.default_rng(40 + d)
    nf = (8, 6, 8)
    nc = tuple(a // b for a, b in zip(nf, c))
    k, j, i = np.meshgrid(*[np.arange(m) for m in nf[::-1]], indexing="ij")
    K, J, I = np.meshgrid(*[np.arange(m) for m in nc[::-1]], indexing="ij")
    qf = (i, j, k)[d] + 0.5
    qc = ((I, J, K)[d] + 0.5) * c[d]
    for bc in [(1, 1, 1), (0, 0, 0)]:
        Lf = W.effective_L(rand_L(rng, nf, 0.2), bc)
        Lc = oracle.coarsen_coeffs(Lf, c)
        lhs = oracle.apply_A(Lc, bc, qc)
        rhs = oracle.restrict_sum(oracle.apply_A(Lf, bc, qf), c)
        sl = [slice(None)] * 3
        if bc[d] == 0:
            sl[2 - d] = slice(1, -1)          # the linear field jumps across the periodic seam
        assert np.max(np.abs((lhs - rhs)[tuple(sl)])) < 1e-12
        assert np.max(np.abs(lhs)) > 0.1
        # the coarse wall plane of a Neumann axis is the coarsened (zero) fine wall plane
        if bc[d] == 1:
            w = [slice(None)] * 3; w[2 - d] = 0
            assert np.all(Lc[d][tuple(w)] == 0.0)


@pytest.mark.parametrize("solver", [oracle.GMG_RBGS, oracle.PCG, oracle.GMG_PCG, oracle.GMG_CGS])
def test_norms_and_stopping_ignore_inactive_cells(solver):
    """O9: the reference norm and the residual are taken over ACTIVE cells.  Garbage in the
    right-hand side on inactive cells (inside a solid) must change nothing: r_ref equals the
    norm over the independently built activity mask, history, count and p are unchanged.
    Fails: active_norm summing over all cells."""
    rng = np.random.default_rng(33)
    n, bc = (8, 8, 8), (1, 0, 0)
    L32 = rng.uniform(0.2, 1, (3, 8, 8, 8)).astype(np.float32)
    L32[:, 2:5, 2:5, 2:5] = 0.0                        # a solid block: 2x2x2 cells have no face
    A = dense_by_faces(n, bc, W.effective_L(L32, bc))
    act = (np.diag(A) != 0.0).reshape(8, 8, 8)
    assert (~act).sum() == 8
    z = W.project_compatible(rng.standard_normal((8, 8, 8)), act)
    zg = z.copy()
    zg[~act] = 50.0 * rng.standard_normal((~act).sum())
    o1 = oracle.Hierarchy(n, bc, L32).solve(solver, z, tol=1e-6, maxiter=300)
    o2 = oracle.Hierarchy(n, bc, L32).solve(solver, zg, tol=1e-6, maxiter=300)
    assert o1["status"] == 0 and o2["status"] == 0
    assert o1["iterations"] == o2["iterations"] >= 2
    assert np.array_equal(o1["history"], o2["history"])
    assert np.array_equal(o1["p"], o2["p"]) and np.all(o2["p"][~act] == 0.0)
    if "r_ref" in o2:
        assert abs(o2["r_ref"] - np.linalg.norm(z[act])) < 1e-12
    # history[0] = ||z - A 0|| / ||z|| over active cells = 1 exactly with a zero guess
    assert abs(o2["history"][0] - 1.0) < 1e-12
    r = np.where(act.ravel(), zg.ravel() - A @ o2["p"].ravel(), 0.0)
    assert abs(np.linalg.norm(r) / np.linalg.norm(z[act]) - o2["true_res"]) < 1e-9


def _two_slab_level(sigma, seed=51):
    """One level, (4, 6, 8) periodic, cut into two x-slabs of width 2 by zero x-faces at i = 0
    and i = 2: two disconnected fluid regions, null space = constants per slab.  Coefficients
    1 + 0.01*noise (D = -5 up to 1 % in every cell); right-hand side +1 / -1 on the two slabs
    (zero global mean, incompatible per slab) plus sigma * compatible noise."""
    rng = np.random.default_rng(seed)
    n, bc = (4, 6, 8), (0, 0, 0)
    L = 1.0 + 0.01 * rng.uniform(-1, 1, (3, 8, 6, 4))
    L[0, :, :, 0] = 0.0
    L[0, :, :, 2] = 0.0
    L32 = L.astype(np.float32)
    b = np.zeros((8, 6, 4))
    b[:, :, :2] = 1.0
    b[:, :, 2:] = -1.0
    b += sigma * W.project_compatible(rng.standard_normal(b.shape), np.ones(b.shape, bool))
    return n, bc, L32, b


def _dense_first_cg_step(n, bc, L32, b):
    """alpha_1 and x_1 of Jacobi-PCG from x0 = 0, from the face-assembled matrix: x_1 is the
    energy minimiser along v = D^-1 r0 and alpha_1 = r0.(x_1 - x0) / (r0 . D^-1 r0)."""
    A = dense_by_faces(n, bc, L32.astype(np.float64))
    Dg = np.diag(A)
    r0 = b.ravel() - b.mean()
    v = r0 / Dg
    t = (v @ r0) / (v @ (A @ v))
    x1 = t * v
    return (r0 @ x1) / (r0 @ v), x1.reshape(b.shape)


def test_cg_smoother_step_length_cap():
    """O12's guard 'a step of length alpha > 16 n_max^2 is not taken' in a case where it fires in
    FP64: a right-hand side incompatible on each of two disconnected regions (only the global
    mean is removed at the restart), with nearly uniform coefficients so that the first search
    direction is nearly a null vector (the smaller the compatible part of the right-hand side,
    the longer the step).  alpha_1 is computed independently from the dense matrix;
    just below the cap the oracle takes the step (= the dense minimiser), just above it leaves x
    untouched for any iteration count.  Fails: cap removed, cap on another extent or constant,
    step applied before the test."""
    cap = 16.0 * 8 * 8
    lo, hi = 1e-3, 0.3                                  # alpha_1 falls as the noise sigma grows
    for _ in range(60):
        mid = np.sqrt(lo * hi)
        a, _ = _dense_first_cg_step(*_two_slab_level(mid))
        lo, hi = (mid, hi) if a > cap else (lo, mid)
    sigma_cap = hi
    below, above = None, None
    for sigma in (sigma_cap * 1.2, sigma_cap / 1.2):
        n, bc, L32, b = _two_slab_level(sigma)
        a1, x1 = _dense_first_cg_step(n, bc, L32, b)
        H = oracle.Hierarchy(n, bc, L32, n_min=64)
        assert H.nlev == 1
        x0 = np.zeros_like(b)
        if a1 <= cap:
            below = a1
            got = H.level_cg_smooth(0, x0, b, 1)
            assert np.abs(got - x1).max() < 1e-9 * np.abs(x1).max() and np.abs(x1).max() > 1.0
        else:
            above = a1
            for m in (1, 2, 7):
                assert np.array_equal(H.level_cg_smooth(0, x0, b, m), x0)
    assert below is not None and above is not None
    assert 0.5 * cap < below <= cap < above < 2.0 * cap


@pytest.mark.parametrize("solver", [oracle.GMG_RBGS, oracle.PCG, oracle.GMG_PCG, oracle.GMG_CGS])
def test_stopping_test_is_relative_to_the_right_hand_side_not_the_first_residual(solver):
    """O9: stop when ||z - A p|| <= tol ||z||, tested BEFORE the first cycle.  A warm start whose
    residual is already below tol ||z|| takes 0 iterations and leaves p alone; history[0] is the
    warm start's residual relative to ||z|| (recomputed here from the face-assembled matrix)."""
    rng = np.random.default_rng(34)
    n, bc = (8, 8, 8), (0, 1, 0)
    L32 = rng.uniform(0.2, 1, (3, 8, 8, 8)).astype(np.float32)
    A = dense_by_faces(n, bc, W.effective_L(L32, bc))
    z = W.project_compatible(rng.standard_normal((8, 8, 8)), np.ones((8, 8, 8), bool))
    good = oracle.Hierarchy(n, bc, L32).solve(oracle.GMG_RBGS, z, tol=1e-7, maxiter=100)["p"]
    rel0 = np.linalg.norm(z.ravel() - A @ good.ravel()) / np.linalg.norm(z)
    assert 1e-9 < rel0 <= 1e-7
    out = oracle.Hierarchy(n, bc, L32).solve(solver, z, p0=good, tol=1e-4, maxiter=50)
    assert out["iterations"] == 0 and out["status"] == 0 and np.array_equal(out["p"], good)
    assert abs(out["history"][0] - rel0) < 1e-12
    # a start WORSE than zero: history[0] > 1 is still relative to ||z||, and the solve goes on
    # until tol * ||z||, not merely tol * (first residual)
    poor = good + 10.0 * rng.standard_normal(good.shape)
    rel1 = np.linalg.norm(z.ravel() - A @ poor.ravel()) / np.linalg.norm(z)
    assert rel1 > 5.0
    out = oracle.Hierarchy(n, bc, L32).solve(solver, z, p0=poor, tol=1e-3, maxiter=300)
    assert abs(out["history"][0] - rel1) < 1e-12 * rel1 and out["iterations"] >= 1
    assert out["status"] == 0 and out["history"][-1] <= 1e-3 < out["history"][-2]


def test_relaxation_factor_persists_for_rbgs_and_never_enters_the_preconditioner():
    """O8: omega is carried from one GMG-RBGS solve to the next on the same hierarchy (time
    stepping).  O11: the preconditioning cycle runs at omega = 1 whatever that
    state is."""
    w = W.config0()
    z = w.z.astype(np.float64)
    H = oracle.Hierarchy(w.n, w.bc, w.L)
    H.omega = 0.625
    out = H.solve(oracle.GMG_RBGS, z, tol=0.0, maxiter=3)
    # started from the carried value; every cycle decays here, so +1/32 per cycle
    assert list(out["omegas"]) == [0.625, 0.65625, 0.6875] and H.omega == 0.71875
    fresh = oracle.Hierarchy(w.n, w.bc, w.L).solve(oracle.GMG_RBGS, z, tol=0.0, maxiter=3)
    assert not np.allclose(fresh["history"][1:], out["history"][1:], rtol=1e-3)
    H = oracle.Hierarchy(w.n, w.bc, w.L)
    H.omega = 0.625
    a = H.solve(oracle.GMG_PCG, z, tol=1e-6, maxiter=50)
    b = oracle.Hierarchy(w.n, w.bc, w.L).solve(oracle.GMG_PCG, z, tol=1e-6, maxiter=50)
    assert np.array_equal(a["history"], b["history"]) and H.omega == 0.625
