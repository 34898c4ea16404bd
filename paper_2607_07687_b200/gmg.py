"""Thin ctypes binding of the C-ABI library (include/gmg.h -> libgmg.so).

Argument marshalling only: every step of the solve runs in the CUDA kernels of
``csrc/``.  PyTorch is used to allocate device memory and to name the stream.  There is no
CPU fallback: importing this module without the built library, or calling it without a
CUDA device, raises.

``lib`` exposes the raw ``gmg_*`` entry points; ``GMG`` wraps one context with methods of
the same names (``set_coeffs``, ``solve``, ``stats``, ``op_residual`` ...).
Arrays are torch float32 CUDA tensors, C-ordered ``[k][j][i]`` (x fastest); ``L`` has
shape ``(3, nz, ny, nx)``.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgmg.so")

# GMG_CGS: the paper's own GMG-PCG, the V-cycle with a Jacobi-PCG smoother (include/gmg.h)
PCG, GMG_PCG, GMG_RBGS, GMG_CGS = 0, 1, 2, 3
BC_PERIODIC, BC_NEUMANN = 0, 1
OK, NOT_CONVERGED = 0, 1
EINVAL, ESTATE, ECUDA, ENOMEM, EBREAKDOWN = -1, -2, -3, -4, -5
COARSEN_ANISO, COARSEN_ISO = 0, 1


class Params(C.Structure):
    _fields_ = [("nu_pre", C.c_int), ("nu_post", C.c_int), ("nu_coarse", C.c_int),
                ("omega0", C.c_float), ("omega_min", C.c_float), ("omega_down", C.c_float),
                ("omega_up", C.c_float), ("adaptive", C.c_int), ("coarsen_mode", C.c_int),
                ("n_min", C.c_int), ("fast_path", C.c_int), ("use_graph", C.c_int),
                ("tma_min_cells", C.c_int), ("cluster_tail", C.c_int),
                ("fused_norm", C.c_int), ("uniform_tiles", C.c_int), ("small_cg", C.c_int)]


class Stats(C.Structure):
    _fields_ = [("solver", C.c_int), ("status", C.c_int), ("iterations", C.c_int),
                ("levels", C.c_int), ("omega_final", C.c_double), ("resid_ref", C.c_double),
                ("resid_init_rel", C.c_double), ("resid_final_rel", C.c_double),
                ("gpu_ms", C.c_double), ("bytes_algorithmic", C.c_double),
                ("kernel_launches", C.c_longlong), ("history_len", C.c_int),
                ("uniform_fraction", C.c_double), ("bytes_as_run", C.c_double),
                ("uniform_fraction_residual", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_I3 = C.c_int * 3
_vp = C.c_void_p


class Plan(C.Structure):
    _fields_ = [("levels", C.c_int), ("n", (C.c_int * 3) * 24), ("c", (C.c_int * 3) * 24),
                ("tail_start", C.c_int), ("workspace_bytes", C.c_size_t)]

# name -> (restype, argtypes); every symbol include/gmg.h declares
SIGNATURES = {
    "gmg_plan": (C.c_int, [C.c_int, C.c_int, C.c_int, _I3, C.POINTER(Params), C.POINTER(Plan)]),
    "gmg_create": (C.c_int, [C.POINTER(_vp), C.c_int, C.c_int, C.c_int, _I3]),
    "gmg_destroy": (None, [_vp]),
    "gmg_last_error": (C.c_char_p, [_vp]),
    "gmg_default_params": (None, [C.POINTER(Params)]),
    "gmg_set_params": (C.c_int, [_vp, C.POINTER(Params)]),
    "gmg_get_params": (C.c_int, [_vp, C.POINTER(Params)]),
    "gmg_workspace_bytes": (C.c_size_t, [_vp]),
    "gmg_set_workspace": (C.c_int, [_vp, _vp, C.c_size_t]),
    "gmg_set_coeffs": (C.c_int, [_vp, _vp, _vp]),
    "gmg_solve": (C.c_int, [_vp, _vp, _vp, C.c_float, C.c_int, C.c_int, _vp]),
    "gmg_solve_host": (C.c_int, [_vp, _vp, _vp, C.c_float, C.c_int, C.c_int, _vp]),
    "gmg_solve_host_cold": (C.c_int, [_vp, _vp, _vp, C.c_float, C.c_int, C.c_int, _vp]),
    "gmg_stats": (C.c_int, [_vp, C.POINTER(Stats)]),
    "gmg_history": (C.c_int, [_vp, C.POINTER(C.c_double), C.c_int]),
    "gmg_omega_history": (C.c_int, [_vp, C.POINTER(C.c_double), C.c_int]),
    "gmg_set_omega": (C.c_int, [_vp, C.c_float]),
    "gmg_num_levels": (C.c_int, [_vp]),
    "gmg_level_shape": (C.c_int, [_vp, C.c_int, _I3, _I3]),
    "gmg_level_coeffs": (C.c_int, [_vp, C.c_int, _vp, _vp]),
    "gmg_op_residual": (C.c_int, [_vp, C.c_int, _vp, _vp, _vp, _vp]),
    "gmg_op_smooth": (C.c_int, [_vp, C.c_int, _vp, _vp, C.c_float, C.c_int, C.c_int, _vp]),
    "gmg_op_restrict": (C.c_int, [_vp, C.c_int, _vp, _vp, _vp]),
    "gmg_op_residual_restrict": (C.c_int, [_vp, C.c_int, _vp, _vp, _vp, _vp]),
    "gmg_op_prolong": (C.c_int, [_vp, C.c_int, _vp, _vp, _vp]),
    "gmg_op_vcycle": (C.c_int, [_vp, _vp, _vp, C.c_float, C.c_int, _vp]),
    "gmg_op_sweep_with_norm": (C.c_int, [_vp, C.c_int, _vp, _vp, _vp, C.c_float, C.c_int,
                                         C.POINTER(C.c_double), C.POINTER(C.c_double), _vp]),
    "gmg_op_cg_smooth": (C.c_int, [_vp, C.c_int, _vp, _vp, C.c_int, _vp]),
    "gmg_op_vcycle_cgs": (C.c_int, [_vp, _vp, _vp, _vp]),
    "gmg_op_norm2": (C.c_int, [_vp, C.c_int, _vp, C.POINTER(C.c_double), _vp]),
    "gmg_divergence": (C.c_int, [_vp, _vp, C.POINTER(C.c_float), _vp, _vp]),
    "gmg_project": (C.c_int, [_vp, _vp, _vp, _vp]),
    "gmg_pressure_step": (C.c_int, [_vp, _vp, _vp, C.POINTER(C.c_float), _vp, C.c_float, C.c_int, C.c_int, _vp]),
    "gmg_describe_plan": (C.c_int, [_vp, C.c_char_p, C.c_size_t]),
    "gmg_residual_norm2_noalloc": (C.c_int, [C.c_int, C.c_int, C.c_int, _I3, _vp, _vp, _vp, _vp, _vp,
                                             C.c_char_p, C.c_size_t]),
}


def load_library(path: str = LIB_PATH) -> C.CDLL:
    if not os.path.exists(path):
        raise RuntimeError(
            f"{path} is missing: build it with `python -m paper_2607_07687_b200.build` "
            "(there is no CPU fallback)")
    dll = C.CDLL(path)
    for name, (res, args) in SIGNATURES.items():
        f = getattr(dll, name)          # AttributeError if the symbol is not exported
        f.restype = res
        f.argtypes = args
    return dll


lib = load_library()


def plan(n, bc, **params):
    """Host-only level table: (shapes, factors, tail_start, workspace_bytes).  No GPU needed."""
    prm = Params()
    lib.gmg_default_params(C.byref(prm))
    for k, v in params.items():
        setattr(prm, k, v)
    out = Plan()
    rc = lib.gmg_plan(int(n[0]), int(n[1]), int(n[2]), _I3(*[int(b) for b in bc]), C.byref(prm), C.byref(out))
    if rc != OK:
        raise ValueError(f"gmg_plan rejected n={tuple(n)} bc={tuple(bc)} (code {rc})")
    shapes = [tuple(out.n[l]) for l in range(out.levels)]
    factors = [tuple(out.c[l]) for l in range(out.levels)]
    return shapes, factors, out.tail_start, out.workspace_bytes


NOALLOC_MAX_CELLS = 1 << 24


def residual_norm2_noalloc(n, bc, L, p, b, out, stream=None):
    """out[0] = ||b - A p||_2 over the active cells, through the entry point that allocates nothing
    (static device scratch; at most NOALLOC_MAX_CELLS cells).  L, p, b: float32 CUDA tensors; out: a
    float64 CUDA tensor the caller made beforehand.  Stream-ordered, no host synchronisation."""
    if stream is None:
        stream = torch.cuda.current_stream(out.device).cuda_stream
    err = C.create_string_buffer(512)
    rc = lib.gmg_residual_norm2_noalloc(int(n[0]), int(n[1]), int(n[2]), _I3(*[int(v) for v in bc]),
                                        _vp(L.data_ptr()), _vp(p.data_ptr()), _vp(b.data_ptr()),
                                        _vp(out.data_ptr()), _vp(stream), err, 512)
    if rc != OK:
        raise GMGError(rc, err.value.decode())
    return out


class GMGError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"gmg error {code}: {msg}")
        self.code = code


def _ptr(t: torch.Tensor) -> int:
    return t.data_ptr()


class GMG:
    """One solver context for an (nx, ny, nz) grid with per-axis boundary conditions."""

    def __init__(self, n, bc, device="cuda:0", **params):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2607_07687_b200 needs a CUDA device (no CPU fallback)")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.n = tuple(int(v) for v in n)
        self.bc = tuple(int(v) for v in bc)
        h = _vp()
        rc = lib.gmg_create(C.byref(h), self.n[0], self.n[1], self.n[2], _I3(*self.bc))
        if rc != OK:
            raise GMGError(rc, "gmg_create failed (bad extents / boundary conditions?)")
        self._h = h
        self._ws = None
        self._L = None
        if params:
            self.set_params(**params)
        else:
            self._alloc_workspace()

    # -- life cycle -----------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            lib.gmg_destroy(self._h)
            self._h = None
            self._ws = None
            self._L = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, allow_warning=False):
        if rc < 0 or (rc > 0 and not allow_warning):
            raise GMGError(rc, lib.gmg_last_error(self._h).decode())
        return rc

    def _stream(self):
        return _vp(torch.cuda.current_stream(self.device).cuda_stream)

    def _alloc_workspace(self):
        nbytes = lib.gmg_workspace_bytes(self._h)
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self._ws.data_ptr() + 255) // 256 * 256
        self._check(lib.gmg_set_workspace(self._h, _vp(base), nbytes))

    def default_params(self) -> Params:
        p = Params()
        lib.gmg_default_params(C.byref(p))
        return p

    def get_params(self) -> Params:
        p = Params()
        self._check(lib.gmg_get_params(self._h, C.byref(p)))
        return p

    def set_params(self, **kw):
        p = self.get_params()
        for k, v in kw.items():
            if not hasattr(p, k):
                raise TypeError(f"unknown parameter {k}")
            setattr(p, k, v)
        self._check(lib.gmg_set_params(self._h, C.byref(p)))
        self._alloc_workspace()
        if self._L is not None:
            self.set_coeffs(self._L)

    # -- setup and solve ------------------------------------------------------------------
    def _vec(self, t, lev=0):
        n, _ = self.level_shape(lev)
        assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
        assert t.numel() == n[0] * n[1] * n[2], (t.shape, n)
        return _vp(_ptr(t))

    def set_coeffs(self, L: torch.Tensor):
        assert L.is_cuda and L.dtype == torch.float32 and L.is_contiguous()
        assert tuple(L.shape) == (3, self.n[2], self.n[1], self.n[0]), L.shape
        self._L = L                                    # kept by pointer in the library
        self._check(lib.gmg_set_coeffs(self._h, _vp(_ptr(L)), self._stream()))

    def solve(self, p: torch.Tensor, z: torch.Tensor, tol=1e-4, maxiter=50, solver=GMG_RBGS):
        """In place on p.  Returns the status code (OK or NOT_CONVERGED)."""
        return self._check(lib.gmg_solve(self._h, self._vec(p), self._vec(z), float(tol),
                                         int(maxiter), int(solver), self._stream()),
                           allow_warning=True)

    def solve_host(self, p_host: torch.Tensor, z_host: torch.Tensor, tol=1e-4, maxiter=50,
                   solver=GMG_RBGS):
        """p_host / z_host: CPU float32 tensors (pinned for full copy bandwidth)."""
        for t in (p_host, z_host):
            assert (not t.is_cuda) and t.dtype == torch.float32 and t.is_contiguous()
            assert t.numel() == self.n[0] * self.n[1] * self.n[2]
        return self._check(lib.gmg_solve_host(self._h, _vp(_ptr(p_host)), _vp(_ptr(z_host)),
                                              float(tol), int(maxiter), int(solver),
                                              self._stream()), allow_warning=True)

    def solve_host_cold(self, p_host_out: torch.Tensor, z_host: torch.Tensor, tol=1e-4, maxiter=50,
                        solver=GMG_RBGS):
        """Zero initial guess (made on the device); p_host_out receives the solution."""
        for t in (p_host_out, z_host):
            assert (not t.is_cuda) and t.dtype == torch.float32 and t.is_contiguous()
            assert t.numel() == self.n[0] * self.n[1] * self.n[2]
        return self._check(lib.gmg_solve_host_cold(self._h, _vp(_ptr(p_host_out)), _vp(_ptr(z_host)),
                                                   float(tol), int(maxiter), int(solver),
                                                   self._stream()), allow_warning=True)

    def stats(self) -> dict:
        s = Stats()
        self._check(lib.gmg_stats(self._h, C.byref(s)))
        return s.as_dict()

    def history(self):
        n = self.stats()["history_len"]
        buf = (C.c_double * max(n, 1))()
        m = lib.gmg_history(self._h, buf, n)
        return [buf[i] for i in range(m)]

    def omega_history(self):
        n = self.stats()["iterations"]
        buf = (C.c_double * max(n, 1))()
        m = lib.gmg_omega_history(self._h, buf, n)
        return [buf[i] for i in range(m)]

    def set_omega(self, omega):
        self._check(lib.gmg_set_omega(self._h, float(omega)))

    # -- level table and per-operator hooks -----------------------------------------------
    def num_levels(self) -> int:
        return lib.gmg_num_levels(self._h)

    def level_shape(self, lev):
        n, c = _I3(), _I3()
        self._check(lib.gmg_level_shape(self._h, lev, n, c))
        return tuple(n), tuple(c)

    def _new(self, lev):
        n, _ = self.level_shape(lev)
        return torch.empty((n[2], n[1], n[0]), dtype=torch.float32, device=self.device)

    def level_coeffs(self, lev) -> torch.Tensor:
        n, _ = self.level_shape(lev)
        out = torch.empty((3, n[2], n[1], n[0]), dtype=torch.float32, device=self.device)
        self._check(lib.gmg_level_coeffs(self._h, lev, _vp(_ptr(out)), self._stream()))
        return out

    def op_residual(self, lev, p, b):
        r = self._new(lev)
        self._check(lib.gmg_op_residual(self._h, lev, self._vec(p, lev), self._vec(b, lev),
                                        _vp(_ptr(r)), self._stream()))
        return r

    def op_smooth(self, lev, p, b, omega=1.0, nsweeps=1, first_colour=0):
        """In place on p."""
        self._check(lib.gmg_op_smooth(self._h, lev, self._vec(p, lev), self._vec(b, lev),
                                      float(omega), int(nsweeps), int(first_colour),
                                      self._stream()))
        return p

    def op_restrict(self, lev, r_fine):
        out = self._new(lev + 1)
        self._check(lib.gmg_op_restrict(self._h, lev, self._vec(r_fine, lev), _vp(_ptr(out)),
                                        self._stream()))
        return out

    def op_residual_restrict(self, lev, p, b):
        out = self._new(lev + 1)
        self._check(lib.gmg_op_residual_restrict(self._h, lev, self._vec(p, lev),
                                                 self._vec(b, lev), _vp(_ptr(out)),
                                                 self._stream()))
        return out

    def op_prolong(self, lev, e_coarse, p_fine):
        """In place on p_fine."""
        self._check(lib.gmg_op_prolong(self._h, lev, self._vec(e_coarse, lev + 1),
                                       self._vec(p_fine, lev), self._stream()))
        return p_fine

    def op_vcycle(self, p, z, omega=1.0, symmetric=False):
        """In place on p."""
        self._check(lib.gmg_op_vcycle(self._h, self._vec(p), self._vec(z), float(omega),
                                      int(bool(symmetric)), self._stream()))
        return p

    def op_sweep_with_norm(self, lev, src, b, omega=1.0, first_colour=0):
        """One fused red+black sweep out of place; returns (dst, sum r^2 of src, sum b^2 active)."""
        dst = self._new(lev)
        rr, bb = C.c_double(0.0), C.c_double(0.0)
        self._check(lib.gmg_op_sweep_with_norm(self._h, lev, self._vec(src, lev), _vp(_ptr(dst)),
                                               self._vec(b, lev), float(omega), int(first_colour),
                                               C.byref(rr), C.byref(bb), self._stream()))
        return dst, rr.value, bb.value

    def op_cg_smooth(self, lev, x, b, iters):
        """In place on x."""
        self._check(lib.gmg_op_cg_smooth(self._h, lev, self._vec(x, lev), self._vec(b, lev),
                                         int(iters), self._stream()))
        return x

    def op_vcycle_cgs(self, p, z):
        """In place on p."""
        self._check(lib.gmg_op_vcycle_cgs(self._h, self._vec(p), self._vec(z), self._stream()))
        return p

    def op_norm2(self, lev, r) -> float:
        out = C.c_double(0.0)
        self._check(lib.gmg_op_norm2(self._h, lev, self._vec(r, lev), C.byref(out),
                                     self._stream()))
        return out.value

    def divergence(self, u: torch.Tensor, wall_hi=(0.0, 0.0, 0.0), out=None) -> torch.Tensor:
        """z = div u; u: (3, nz, ny, nx) lower-face velocities.  out: optional result tensor."""
        assert u.is_cuda and u.dtype == torch.float32 and u.is_contiguous()
        assert tuple(u.shape) == (3, self.n[2], self.n[1], self.n[0])
        z = self._new(0) if out is None else out
        self._vec(z)
        wh = (C.c_float * 3)(*[float(v) for v in wall_hi])
        self._check(lib.gmg_divergence(self._h, _vp(_ptr(u)), wh, _vp(_ptr(z)), self._stream()))
        return z

    def project(self, u: torch.Tensor, p: torch.Tensor) -> torch.Tensor:
        """In place on u: u -= L grad p."""
        assert u.is_cuda and u.dtype == torch.float32 and u.is_contiguous()
        assert tuple(u.shape) == (3, self.n[2], self.n[1], self.n[0])
        self._check(lib.gmg_project(self._h, _vp(_ptr(u)), self._vec(p), self._stream()))
        return u

    def pressure_step(self, L: torch.Tensor, u: torch.Tensor, p: torch.Tensor, wall_hi=(0.0, 0.0, 0.0),
                      tol=1e-4, maxiter=50, solver=GMG_RBGS):
        """set_coeffs(L) -> div u -> solve (p in/out) -> u -= L grad p, one host synchronisation.
        Returns the solve's status code; u is projected in place (stream-ordered)."""
        shape3 = (3, self.n[2], self.n[1], self.n[0])
        for t in (L, u):
            assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and tuple(t.shape) == shape3
        wh = (C.c_float * 3)(*[float(v) for v in wall_hi])
        rc = lib.gmg_pressure_step(self._h, _vp(_ptr(L)), _vp(_ptr(u)), wh, self._vec(p), float(tol),
                                   int(maxiter), int(solver), self._stream())
        self._check(rc, allow_warning=True)
        self._L = L          # kept by pointer
        return rc

    def describe_plan(self) -> str:
        buf = C.create_string_buffer(4096)
        self._check(lib.gmg_describe_plan(self._h, buf, 4096))
        return buf.value.decode()
