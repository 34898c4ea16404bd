"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is the ONLY code shared by the CUDA path (tests, bench.py) and the
oracle (tests): it builds input arrays and holds none of the solver's
arithmetic.  NumPy only; FP64 maths, one final cast to FP32, so that oracle and
GPU are fed the same FP32 bits (SURVEY.md §8(d) "Common generator conventions").

The paper measures on WaterLily simulations (TGV Re=1600, sphere Re_D=3700,
swimming jellyfish: §2/§3 Table 1).  Those cases are not
available; these generators are synthetic stand-ins with the paper's grid
shapes, boundary-condition types and coefficient structure (0 in solids, linear
BDIM-like ramp near bodies).  See DESIGN.md "Input recipe".

Conventions
-----------
* arrays are C-ordered ``[k][j][i]`` (x fastest); ``L`` has shape ``(3,nz,ny,nx)``
  with ``L[d]`` the coefficient on the LOWER face of each cell in direction d.
* cell centre ``(i+1/2, j+1/2, k+1/2)``; lower-d face centre = that minus e_d/2.
* ``bc[d]`` = 0 periodic, 1 homogeneous Neumann (the wall face carries 0).
* discrete divergence ``z_I = sum_d u_d(I+e_d) - u_d(I)``, ``u_d(I)`` on the lower
  face of I; periodic axes wrap, Neumann axes carry prescribed wall values.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

PERIODIC = 0
NEUMANN = 1


@dataclass
class Workload:
    name: str
    n: tuple            # (nx, ny, nz)
    bc: tuple           # per axis, PERIODIC / NEUMANN
    L: np.ndarray       # float32 (3, nz, ny, nx)
    z: np.ndarray       # float32 (nz, ny, nx)
    tol: float = 1e-4
    maxiter: int = 50
    seed: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def cells(self) -> int:
        return int(self.n[0]) * int(self.n[1]) * int(self.n[2])


# --------------------------------------------------------------------------
# helpers (input conditioning only)
# --------------------------------------------------------------------------
def ramp(d):
    """BDIM-like linear ramp over +-2 cells of signed distance (positive in fluid)."""
    return np.clip((d + 2.0) / 4.0, 0.0, 1.0)


def face_coords(n, d, dtype=np.float64):
    """Broadcastable (x, y, z) coordinates of the lower-d face centres, [k][j][i] order."""
    nx, ny, nz = n
    x = np.arange(nx, dtype=dtype) + 0.5
    y = np.arange(ny, dtype=dtype) + 0.5
    z = np.arange(nz, dtype=dtype) + 0.5
    if d == 0:
        x = x - 0.5
    elif d == 1:
        y = y - 0.5
    else:
        z = z - 0.5
    return x[None, None, :], y[None, :, None], z[:, None, None]


def _upper(a, axis_d, bc_d, wall_value=0.0):
    """Value on the UPPER d-face of every cell given lower-face array ``a``.

    axis_d: 0=x,1=y,2=z -> numpy axes 2,1,0.  Periodic: wrap.  Neumann: the upper
    wall face carries ``wall_value``.
    """
    ax = 2 - axis_d
    up = np.roll(a, -1, axis=ax)
    if bc_d == NEUMANN:
        sl = [slice(None)] * 3
        sl[ax] = -1
        up[tuple(sl)] = wall_value
    return up


def effective_L(L, bc):
    """Copy of L (float64) with the wall plane L_d(index 0) zeroed on Neumann axes."""
    Le = np.array(L, dtype=np.float64, copy=True)
    for d in range(3):
        if bc[d] == NEUMANN:
            sl = [slice(None)] * 3
            sl[2 - d] = 0
            Le[d][tuple(sl)] = 0.0
    return Le


def active_mask(L, bc):
    """Cells with at least one non-zero face coefficient (an exact test, L >= 0)."""
    Le = effective_L(L, bc)
    tot = np.zeros(Le.shape[1:], dtype=np.float64)
    for d in range(3):
        tot += Le[d] + _upper(Le[d], d, bc[d], 0.0)
    return tot != 0.0


def divergence(u, bc, wall_hi=(0.0, 0.0, 0.0)):
    """z_I = sum_d u_d(upper face) - u_d(lower face).  ``u``: (3,nz,ny,nx) float64.

    On a Neumann axis ``u[d][index 0]`` is the lower wall value and ``wall_hi[d]``
    (scalar or array broadcastable to the wall plane) the upper wall value.
    """
    z = np.zeros(u.shape[1:], dtype=np.float64)
    for d in range(3):
        z += _upper(u[d], d, bc[d], wall_hi[d]) - u[d]
    return z


def project_compatible(z, act):
    """Zero inactive cells and remove the FP64 mean over active cells."""
    z = np.where(act, z, 0.0)
    nact = int(act.sum())
    if nact:
        z = z - np.where(act, z.sum(dtype=np.float64) / nact, 0.0)
    return z


# --------------------------------------------------------------------------
# configs[0]: tiny anisotropic, triple periodic, L = 1
# --------------------------------------------------------------------------
def config0(seed=76870, n=(32, 32, 16)):
    rng = np.random.default_rng(seed)
    nx, ny, nz = n
    L = np.ones((3, nz, ny, nx), dtype=np.float32)
    z = rng.standard_normal((nz, ny, nx))
    z = z - z.mean(dtype=np.float64)
    return Workload("config0_tiny", tuple(n), (PERIODIC,) * 3, L, z.astype(np.float32),
                    tol=1e-4, maxiter=50, seed=seed)


# --------------------------------------------------------------------------
# configs[1]: TGV-shaped, 128^3, triple periodic, L = 1
# --------------------------------------------------------------------------
def config1(seed=76871, n=(128, 128, 128), sigma=0.01):
    rng = np.random.default_rng(seed)
    nx, ny, nz = n
    h = 2.0 * np.pi / nx
    bc = (PERIODIC,) * 3
    u = np.zeros((3, nz, ny, nx), dtype=np.float64)
    X, Y, Z = face_coords(n, 0)
    u[0] = np.sin(X * h) * np.cos(Y * h) * np.cos(Z * h)
    X, Y, Z = face_coords(n, 1)
    u[1] = -np.cos(X * h) * np.sin(Y * h) * np.cos(Z * h)
    for d in range(3):                      # drawn x, y, z, full arrays
        u[d] += sigma * rng.standard_normal((nz, ny, nx))
    z = divergence(u, bc)
    z = z - z.mean(dtype=np.float64)
    L = np.ones((3, nz, ny, nx), dtype=np.float32)
    return Workload("config1_tgv", tuple(n), bc, L, z.astype(np.float32),
                    tol=1e-4, maxiter=50, seed=seed)


# --------------------------------------------------------------------------
# configs[2]: sphere in a channel, (16x6x6)D, x Neumann, y/z periodic
# --------------------------------------------------------------------------
def config2(seed=76872, D=16, sigma=0.05):
    rng = np.random.default_rng(seed)
    n = (16 * D, 6 * D, 6 * D)
    nx, ny, nz = n
    bc = (NEUMANN, PERIODIC, PERIODIC)
    c = (4.0 * D, 3.0 * D, 3.0 * D)
    R = 0.5 * D
    L = np.empty((3, nz, ny, nx), dtype=np.float64)
    for d in range(3):
        X, Y, Z = face_coords(n, d)
        L[d] = ramp(np.sqrt((X - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2) - R)
    L32 = L.astype(np.float32)
    Lq = L32.astype(np.float64)
    xi = [rng.standard_normal((nz, ny, nx)) for _ in range(3)]     # drawn x, y, z
    u = np.empty_like(Lq)
    u[0] = Lq[0] * (1.0 + sigma * xi[0])
    u[1] = Lq[1] * (sigma * xi[1])
    u[2] = Lq[2] * (sigma * xi[2])
    u[0][:, :, 0] = 1.0                      # inflow face (lower face of i = 0)
    z = divergence(u, bc, wall_hi=(1.0, 0.0, 0.0))   # outflow face carries 1.0
    act = active_mask(L32, bc)
    z = project_compatible(z, act)
    return Workload("config2_sphere", n, bc, L32, z.astype(np.float32),
                    tol=1e-4, maxiter=50, seed=seed,
                    meta={"active_fraction": float(act.mean())})


# --------------------------------------------------------------------------
# configs[3]: jellyfish-like hemispherical shell, 4 x 2^(3p) cells, all Neumann
# --------------------------------------------------------------------------
def _shell_distance(X, Y, Z, c, R):
    """Distance to the mid-surface of the upper (+z) hemisphere of radius R incl. its rim."""
    h = Z - c[2]
    rho = np.hypot(X - c[0], Y - c[1])
    r = np.hypot(rho, h)
    return np.where(h >= 0.0, np.abs(r - R), np.hypot(rho - R, h))


def config3(p=5, seed=None):
    if seed is None:
        seed = {5: 76873, 6: 76875}.get(p, 76873 + 2 * (p - 5))
    rng = np.random.default_rng(seed)
    nx = 2 ** (p + 1)
    n = (nx, nx, nx // 2)
    nx, ny, nz = n
    bc = (NEUMANN,) * 3
    c = (nx / 2.0, ny / 2.0, nz / 2.0)
    R = 0.25 * nx
    L = np.empty((3, nz, ny, nx), dtype=np.float64)
    S = []
    for d in range(3):
        X, Y, Z = face_coords(n, d)
        s = _shell_distance(X, Y, Z, c, R)
        S.append(s)
        L[d] = np.clip((s - 1.5) / 4.0, 0.0, 1.0)
    L32 = L.astype(np.float32)
    Lq = L32.astype(np.float64)
    u = np.empty_like(Lq)
    for d in range(3):
        X, Y, Z = face_coords(n, d)
        coords = (X, Y, Z)
        uF = np.zeros((nz, ny, nx), dtype=np.float64)
        for _t in range(8):
            k = rng.integers(0, 5, 3)
            phi = rng.uniform(0.0, 2.0 * np.pi, 3)
            a = rng.standard_normal()
            term = a
            for q in range(3):
                term = term * np.cos(2.0 * np.pi * k[q] * coords[q] / n[q] + phi[q])
            uF += term
        uF *= 0.125
        rel = (X - c[0], Y - c[1], Z - c[2])
        dist = np.sqrt(rel[0] ** 2 + rel[1] ** 2 + rel[2] ** 2)
        dist = np.where(dist == 0.0, 1.0, dist)
        uC = -0.5 * np.exp(-(S[d] / 3.0) ** 2) * rel[d] / dist
        u[d] = Lq[d] * (uF + uC)
    for d in range(3):                       # all wall faces carry 0
        sl = [slice(None)] * 3
        sl[2 - d] = 0
        u[d][tuple(sl)] = 0.0
    z = divergence(u, bc)
    act = active_mask(L32, bc)
    z = project_compatible(z, act)
    return Workload(f"config3_jellyfish_p{p}", n, bc, L32, z.astype(np.float32),
                    tol=1e-4, maxiter=50, seed=seed,
                    meta={"active_fraction": float(act.mean()), "p": p})


def jellyfish_steps(p=5, nsteps=8, period=64, seed=None):
    """A swimming-jellyfish-SHAPED sequence of pressure steps ("simplified swimming
    jellyfish", Table 1; warm starts and a coefficient update every step).
    The shell of configs[3] heaves along z, c_z(k) = nz/2 + 2 sin(2 pi k / period) cells, and its
    contraction velocity swings with it, amplitude 0.5 cos(2 pi k / period); the random-Fourier
    background flow is drawn once and kept.  Yields per step (L32, ustar32): the face
    coefficients [3][nz][ny][nx] and the predicted velocity u* = L (u_F + u_C) on the lower faces
    (all wall faces 0, so div u* sums to zero).  A synthetic stand-in: no Navier-Stokes step is
    taken, the steps are linked only through the warm start of p.  Input conditioning only."""
    if seed is None:
        seed = 76880 + p
    rng = np.random.default_rng(seed)
    nx = 2 ** (p + 1)
    n = (nx, nx, nx // 2)
    nx, ny, nz = n
    R = 0.25 * nx
    coords = [face_coords(n, d) for d in range(3)]
    uF = []
    for d in range(3):
        f = np.zeros((nz, ny, nx), dtype=np.float64)
        for _t in range(8):
            kk = rng.integers(0, 5, 3)
            phi = rng.uniform(0.0, 2.0 * np.pi, 3)
            a = rng.standard_normal()
            term = a
            for q in range(3):
                term = term * np.cos(2.0 * np.pi * kk[q] * coords[d][q] / n[q] + phi[q])
            f += term
        uF.append(0.125 * f)
    for k in range(nsteps):
        th = 2.0 * np.pi * k / period
        c = (nx / 2.0, ny / 2.0, nz / 2.0 + 2.0 * np.sin(th))
        amp = 0.5 * np.cos(th)
        L = np.empty((3, nz, ny, nx), dtype=np.float64)
        u = np.empty_like(L)
        for d in range(3):
            X, Y, Z = coords[d]
            sd = _shell_distance(X, Y, Z, c, R)
            L[d] = np.clip((sd - 1.5) / 4.0, 0.0, 1.0)
            rel = (X - c[0], Y - c[1], Z - c[2])
            dist = np.sqrt(rel[0] ** 2 + rel[1] ** 2 + rel[2] ** 2)
            dist = np.where(dist == 0.0, 1.0, dist)
            uC = -amp * np.exp(-(sd / 3.0) ** 2) * rel[d] / dist
            u[d] = L[d].astype(np.float32).astype(np.float64) * (uF[d] + uC)
            sl = [slice(None)] * 3
            sl[2 - d] = 0
            u[d][tuple(sl)] = 0.0                      # wall faces carry 0
        yield L.astype(np.float32), u.astype(np.float32)


JELLYFISH_BC = (NEUMANN,) * 3


# --------------------------------------------------------------------------
# configs[4]: billion-cell stress: periodic cube, seeded random solid spheres
# --------------------------------------------------------------------------
def config4(n=1024, nspheres=64, diameter=32, seed=76874):
    """1024^3 by default; ``n``/``nspheres``/``diameter`` shrink it for parity tests.

    L starts from ones and only each sphere's bounding box is rewritten (minimum
    over spheres of the ramp, minimum-image distance).  z plane k comes from
    ``default_rng([seed, k])`` so it can be regenerated plane by plane.
    """
    rng = np.random.default_rng(seed)
    bc = (PERIODIC,) * 3
    centres = rng.uniform(0.0, float(n), (nspheres, 3))
    R = 0.5 * diameter
    hw = int(np.ceil(R)) + 3
    L = np.ones((3, n, n, n), dtype=np.float32)
    act = np.ones((n, n, n), dtype=bool) if n <= 256 else None
    inactive_boxes = []
    for s in range(nspheres):
        cx, cy, cz = centres[s]
        ii = (np.arange(int(np.floor(cx)) - hw, int(np.floor(cx)) + hw + 2)) % n
        jj = (np.arange(int(np.floor(cy)) - hw, int(np.floor(cy)) + hw + 2)) % n
        kk = (np.arange(int(np.floor(cz)) - hw, int(np.floor(cz)) + hw + 2)) % n
        for d in range(3):
            off = [0.5, 0.5, 0.5]
            off[d] = 0.0
            dx = ii + off[0] - cx
            dy = jj + off[1] - cy
            dz = kk + off[2] - cz
            dx = dx - n * np.round(dx / n)         # minimum image
            dy = dy - n * np.round(dy / n)
            dz = dz - n * np.round(dz / n)
            dist = np.sqrt(dx[None, None, :] ** 2 + dy[None, :, None] ** 2 + dz[:, None, None] ** 2)
            val = ramp(dist - R).astype(np.float32)
            idx = np.ix_(kk, jj, ii)
            L[d][idx] = np.minimum(L[d][idx], val)
        inactive_boxes.append((kk, jj, ii))
    # z: plane by plane
    z = np.empty((n, n, n), dtype=np.float32)
    for k in range(n):
        z[k] = np.random.default_rng([seed, k]).standard_normal((n, n), dtype=np.float32)
    # inactive cells only occur inside the sphere boxes: evaluate the mask there
    n_inactive = 0
    for (kk, jj, ii) in inactive_boxes:
        kk2 = np.concatenate([kk, [(kk[-1] + 1) % n]])
        jj2 = np.concatenate([jj, [(jj[-1] + 1) % n]])
        ii2 = np.concatenate([ii, [(ii[-1] + 1) % n]])
        sub = L[np.ix_([0, 1, 2], kk2, jj2, ii2)].astype(np.float64)
        tot = (sub[0][:-1, :-1, :-1] + sub[0][:-1, :-1, 1:]
               + sub[1][:-1, :-1, :-1] + sub[1][:-1, 1:, :-1]
               + sub[2][:-1, :-1, :-1] + sub[2][1:, :-1, :-1])
        dead = tot == 0.0
        idx = np.ix_(kk, jj, ii)
        blk = z[idx]
        n_inactive += int(np.count_nonzero(dead & (blk != 0.0)))
        blk[dead] = 0.0
        z[idx] = blk
    total = 0.0
    for k in range(n):
        total += float(z[k].sum(dtype=np.float64))
    nact = n ** 3 - n_inactive
    mean = np.float32(total / nact)
    for k in range(n):
        zk = z[k]
        nz_mask = zk != 0.0            # inactive cells hold exact zeros (N(0,1) never is)
        zk[nz_mask] -= mean
    del act
    return Workload(f"config4_spheres_{n}", (n, n, n), bc, L, z,
                    tol=1e-4, maxiter=50, seed=seed,
                    meta={"active_fraction": nact / float(n ** 3), "nspheres": nspheres,
                          "diameter": diameter})


# --------------------------------------------------------------------------
# Aspect-ratio study (Fig. 2 right): impulsive start of a uniform flow past a
# sphere in an (N b) x b x b box -- x Neumann (inflow / outflow faces carry the free stream),
# y/z periodic.  Synthetic stand-in for the paper's case: same structure, our own sizes.
# --------------------------------------------------------------------------
def impulsive_sphere(N=4, base=32, D=None):
    D = base / 4.0 if D is None else float(D)
    n = (int(N) * base, base, base)
    nx, ny, nz = n
    bc = (NEUMANN, PERIODIC, PERIODIC)
    c = (min(1.0, 0.5 * N) * base, 0.5 * base, 0.5 * base)
    L = np.empty((3, nz, ny, nx), dtype=np.float64)
    for d in range(3):
        X, Y, Z = face_coords(n, d)
        L[d] = ramp(np.sqrt((X - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2) - 0.5 * D)
    L32 = L.astype(np.float32)
    Lq = L32.astype(np.float64)
    u = np.zeros_like(Lq)
    u[0] = Lq[0]                             # u* = the free stream (1, 0, 0), masked by the body
    u[0][:, :, 0] = 1.0                      # inflow face
    z = divergence(u, bc, wall_hi=(1.0, 0.0, 0.0))
    act = active_mask(L32, bc)
    z = project_compatible(z, act)
    return Workload(f"impulsive_sphere_N{N}", n, bc, L32, z.astype(np.float32),
                    tol=1e-4, maxiter=200, seed=0,
                    meta={"active_fraction": float(act.mean()), "aspect": int(N)})


def impulsive_cylinder_2d(N=4, base=32, D=None):
    """2-D counterpart of impulsive_sphere (Fig. 2 left "2D flow around a circular
    cylinder"): an (N b) x b x 1 grid, x Neumann with the free stream on the in/outflow faces, y
    periodic, the single z layer between two walls (its coefficients are ignored)."""
    D = base / 4.0 if D is None else float(D)
    n = (int(N) * base, base, 1)
    nx, ny, nz = n
    bc = (NEUMANN, PERIODIC, NEUMANN)
    c = (min(1.0, 0.5 * N) * base, 0.5 * base)
    L = np.empty((3, nz, ny, nx), dtype=np.float64)
    for d in range(3):
        X, Y, Z = face_coords(n, d)
        L[d] = ramp(np.sqrt((X - c[0]) ** 2 + (Y - c[1]) ** 2) - 0.5 * D)
    L32 = L.astype(np.float32)
    Lq = L32.astype(np.float64)
    u = np.zeros_like(Lq)
    u[0] = Lq[0]
    u[0][:, :, 0] = 1.0
    z = divergence(u, bc, wall_hi=(1.0, 0.0, 0.0))
    act = active_mask(L32, bc)
    z = project_compatible(z, act)
    return Workload(f"impulsive_cylinder2d_N{N}", n, bc, L32, z.astype(np.float32),
                    tol=1e-4, maxiter=200, seed=0,
                    meta={"active_fraction": float(act.mean()), "aspect": int(N)})


def by_name(name: str) -> Workload:
    """configs by short name: c0, c1, c2, c3p5, c3p6, c4 (1024^3), c4_128, c4_256, c4_512."""
    if name == "c0":
        return config0()
    if name == "c1":
        return config1()
    if name == "c2":
        return config2()
    if name == "c3p5":
        return config3(5)
    if name == "c3p6":
        return config3(6)
    if name == "c4":
        return config4()
    if name == "c4_128":
        return config4(n=128, nspheres=16, diameter=8)
    if name == "c4_256":
        return config4(n=256, nspheres=64, diameter=8)
    if name == "c4_512":
        return config4(n=512, nspheres=64, diameter=16)
    raise KeyError(name)
