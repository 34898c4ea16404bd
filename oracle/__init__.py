"""ctypes front-end of the FP64 CPU oracle (oracle/gmg_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  The product package
(paper_2607_07687_b200) never imports this module and this module never imports it.

Arrays: numpy float64, C-ordered [k][j][i]; L float64 (3,nz,ny,nx) for the single-operator
calls, float32 for Hierarchy (the same FP32 bits the GPU gets).  Readings O1..O12 are
documented in gmg_oracle.c and DESIGN.md.
"""
import ctypes as C
import os

import numpy as np

from .build import build as _build

_lib = C.CDLL(_build())

_I3 = C.c_int * 3
_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_fp = np.ctypeslib.ndpointer(dtype=np.float32, flags="C_CONTIGUOUS")


def _sig(name, res, *args):
    f = getattr(_lib, name)
    f.restype = res
    f.argtypes = list(args)
    return f


_apply = _sig("gmgo_apply", None, _I3, _I3, _dp, _dp, _dp)
_diag = _sig("gmgo_diag", None, _I3, _I3, _dp, _dp)
_residual = _sig("gmgo_residual", None, _I3, _I3, _dp, _dp, _dp, _dp)
_norm2 = _sig("gmgo_norm2", C.c_double, _I3, _dp)
_half = _sig("gmgo_half_sweep", None, _I3, _I3, _dp, _dp, _dp, C.c_double, C.c_int)
_rule = _sig("gmgo_coarsen_rule", C.c_int, _I3, _I3, C.c_int, C.c_int, _I3)
_ccoef = _sig("gmgo_coarsen_coeffs", None, _I3, _I3, _dp, _dp)
_rsum = _sig("gmgo_restrict_sum", None, _I3, _I3, _dp, _dp)
_padd = _sig("gmgo_prolong_add", None, _I3, _I3, _dp, _dp)
_div = _sig("gmgo_divergence", None, _I3, _I3, _dp, C.c_double * 3, _dp)
_proj = _sig("gmgo_project", None, _I3, _I3, _dp, _dp, _dp)
_hcreate = _sig("gmgo_hier_create", C.c_void_p, _I3, _I3, _fp, C.c_int, C.c_int)
_hdestroy = _sig("gmgo_hier_destroy", None, C.c_void_p)
_hnlev = _sig("gmgo_hier_nlev", C.c_int, C.c_void_p)
_hshape = _sig("gmgo_hier_shape", None, C.c_void_p, C.c_int, _I3, _I3)
_hL = _sig("gmgo_hier_L", C.POINTER(C.c_double), C.c_void_p, C.c_int)
_hparams = _sig("gmgo_hier_set_params", None, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double,
                C.c_double, C.c_double, C.c_double, C.c_int)
_homega = _sig("gmgo_hier_omega", C.c_double, C.c_void_p)
_hsetomega = _sig("gmgo_hier_set_omega", None, C.c_void_p, C.c_double)
_vcycle = _sig("gmgo_vcycle", None, C.c_void_p, _dp, _dp, C.c_double, C.c_int)
_lres = _sig("gmgo_level_residual", None, C.c_void_p, C.c_int, _dp, _dp, _dp)
_lsweeps = _sig("gmgo_level_sweeps", None, C.c_void_p, C.c_int, _dp, _dp, C.c_double, C.c_int, C.c_int)
_solve_rbgs = _sig("gmgo_solve_gmg_rbgs", C.c_int, C.c_void_p, _dp, _dp, C.c_double, C.c_int, _dp, _dp,
                   C.POINTER(C.c_int), C.POINTER(C.c_double))
_solve_pcg = _sig("gmgo_solve_pcg", C.c_int, C.c_void_p, C.c_int, _dp, _dp, C.c_double, C.c_int, _dp,
                  C.POINTER(C.c_int), C.POINTER(C.c_double))

_cgsmooth = _sig("gmgo_level_cg_smooth", None, C.c_void_p, C.c_int, _dp, _dp, C.c_int)
_vcycle_cgs = _sig("gmgo_vcycle_cgs", None, C.c_void_p, _dp, _dp)
_solve_cgs = _sig("gmgo_solve_gmg_cgs", C.c_int, C.c_void_p, _dp, _dp, C.c_double, C.c_int, _dp,
                  C.POINTER(C.c_int), C.POINTER(C.c_double))

# GMG_CGS = the paper's own "GMG-PCG": GMG whose smoother is Jacobi-PCG (reading O12)
PCG, GMG_PCG, GMG_RBGS, GMG_CGS = 0, 1, 2, 3


def _n_of(a):
    nz, ny, nx = a.shape[-3:]
    return _I3(nx, ny, nz), (nx, ny, nz)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def apply_A(L, bc, p):
    n3, _ = _n_of(p)
    out = np.empty_like(_f64(p))
    _apply(n3, _I3(*bc), _f64(L), _f64(p), out)
    return out


def diag(L, bc):
    L = _f64(L)
    n3, _ = _n_of(L)
    out = np.empty(L.shape[1:], dtype=np.float64)
    _diag(n3, _I3(*bc), L, out)
    return out


def residual(L, bc, p, b):
    n3, _ = _n_of(p)
    out = np.empty_like(_f64(p))
    _residual(n3, _I3(*bc), _f64(L), _f64(p), _f64(b), out)
    return out


def norm2(r):
    n3, _ = _n_of(r)
    return float(_norm2(n3, _f64(r)))


def half_sweep(L, bc, p, b, omega, colour):
    """Returns a new array: p after one colour half-sweep (0 = red)."""
    q = _f64(p).copy()
    n3, _ = _n_of(q)
    _half(n3, _I3(*bc), _f64(L), q, _f64(b), float(omega), int(colour))
    return q


def coarsen_rule(n, bc, n_min=4, iso=False):
    c = _I3()
    any_ = _rule(_I3(*n), _I3(*bc), int(n_min), int(bool(iso)), c)
    return bool(any_), tuple(c)


def level_shapes(n, bc, n_min=4, iso=False):
    shapes = [tuple(n)]
    while True:
        any_, c = coarsen_rule(shapes[-1], bc, n_min, iso)
        if not any_:
            return shapes
        shapes.append(tuple(s // f for s, f in zip(shapes[-1], c)))


def coarsen_coeffs(Lf, c):
    Lf = _f64(Lf)
    n3, n = _n_of(Lf)
    nc = tuple(s // f for s, f in zip(n, c))
    Lc = np.empty((3, nc[2], nc[1], nc[0]), dtype=np.float64)
    _ccoef(n3, _I3(*c), Lf, Lc)
    return Lc


def restrict_sum(rf, c):
    rf = _f64(rf)
    n3, n = _n_of(rf)
    nc = tuple(s // f for s, f in zip(n, c))
    out = np.empty((nc[2], nc[1], nc[0]), dtype=np.float64)
    _rsum(n3, _I3(*c), rf, out)
    return out


def prolong_add(pf, ec, c):
    q = _f64(pf).copy()
    n3, _ = _n_of(q)
    _padd(n3, _I3(*c), _f64(ec), q)
    return q


def divergence(u, bc, wall_hi=(0.0, 0.0, 0.0)):
    """z_I = sum_d u_d(upper face) - u_d(lower face); u: (3,nz,ny,nx) lower-face velocities."""
    u = _f64(u)
    n3, _ = _n_of(u)
    z = np.empty(u.shape[1:], dtype=np.float64)
    _div(n3, _I3(*bc), u, (C.c_double * 3)(*[float(v) for v in wall_hi]), z)
    return z


def project(L, bc, p, u):
    """Returns u - L grad p (new array)."""
    q = _f64(u).copy()
    n3, _ = _n_of(q)
    _proj(n3, _I3(*bc), _f64(L), _f64(p), q)
    return q


class Hierarchy:
    """Level hierarchy (shapes O4, coefficients O5) + V-cycle (O7) + solvers (O8-O11)."""

    def __init__(self, n, bc, L32, n_min=4, iso=False):
        L32 = np.ascontiguousarray(L32, dtype=np.float32)
        assert L32.shape == (3, n[2], n[1], n[0])
        self.n, self.bc = tuple(n), tuple(bc)
        self._h = _hcreate(_I3(*n), _I3(*bc), L32, int(n_min), int(bool(iso)))
        self.nlev = _hnlev(self._h)

    def __del__(self):
        if getattr(self, "_h", None):
            _hdestroy(self._h)
            self._h = None

    def shape(self, lev):
        n, c = _I3(), _I3()
        _hshape(self._h, lev, n, c)
        return tuple(n), tuple(c)

    def L(self, lev):
        n, _ = self.shape(lev)
        N = n[0] * n[1] * n[2]
        ptr = _hL(self._h, lev)
        return np.ctypeslib.as_array(ptr, shape=(3 * N,)).reshape(3, n[2], n[1], n[0]).copy()

    def set_params(self, nu1=2, nu2=2, nuc=32, omega0=1.0, omega_min=0.5, omega_down=0.125,
                   omega_up=0.03125, adaptive=True):
        _hparams(self._h, nu1, nu2, nuc, omega0, omega_min, omega_down, omega_up, int(adaptive))

    @property
    def omega(self):
        return float(_homega(self._h))

    @omega.setter
    def omega(self, w):
        _hsetomega(self._h, float(w))

    def vcycle(self, x, b, omega=1.0, sym=False):
        q = _f64(x).copy()
        _vcycle(self._h, q, _f64(b), float(omega), int(sym))
        return q

    def level_residual(self, lev, x, b):
        out = np.empty_like(_f64(x))
        _lres(self._h, lev, _f64(x), _f64(b), out)
        return out

    def level_sweeps(self, lev, x, b, omega=1.0, count=1, first_colour=0):
        q = _f64(x).copy()
        _lsweeps(self._h, lev, q, _f64(b), float(omega), int(count), int(first_colour))
        return q

    def level_cg_smooth(self, lev, x, b, iters):
        """m Jacobi-PCG iterations restarted from x on level lev (reading O12a)."""
        q = _f64(x).copy()
        _cgsmooth(self._h, lev, q, _f64(b), int(iters))
        return q

    def vcycle_cgs(self, x, b):
        q = _f64(x).copy()
        _vcycle_cgs(self._h, q, _f64(b))
        return q

    def solve(self, solver, z, p0=None, tol=1e-4, maxiter=50):
        """Returns dict(p, iterations, status, history, omegas, true_res)."""
        z = _f64(z)
        p = np.zeros_like(z) if p0 is None else _f64(p0).copy()
        hist = np.zeros(maxiter + 2, dtype=np.float64)
        status = C.c_int(0)
        if solver == GMG_RBGS:
            om = np.zeros(maxiter + 2, dtype=np.float64)
            rref = C.c_double(0.0)
            k = _solve_rbgs(self._h, p, z, float(tol), int(maxiter), hist, om, C.byref(status),
                            C.byref(rref))
            return dict(p=p, iterations=k, status=status.value, history=hist[:k + 1].copy(),
                        omegas=om[:k].copy(), r_ref=rref.value, true_res=float(hist[k]))
        if solver == GMG_CGS:
            rref = C.c_double(0.0)
            k = _solve_cgs(self._h, p, z, float(tol), int(maxiter), hist, C.byref(status), C.byref(rref))
            return dict(p=p, iterations=k, status=status.value, history=hist[:k + 1].copy(),
                        r_ref=rref.value, true_res=float(hist[k]))
        tr = C.c_double(0.0)
        k = _solve_pcg(self._h, 0 if solver == PCG else 1, p, z, float(tol), int(maxiter), hist,
                       C.byref(status), C.byref(tr))
        return dict(p=p, iterations=k, status=status.value, history=hist[:k + 1].copy(),
                    true_res=tr.value)
