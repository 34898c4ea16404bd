"""One pressure step of a staggered projection method on the library's entry points
("predictor + corrector steps", one Poisson solve each):

    gmg_set_coeffs(L)  ->  z = gmg_divergence(u*)  ->  gmg_solve(p, z)  ->  gmg_project(u*, p)

(one call, gmg_pressure_step: the four are enqueued back to back with a single host
synchronisation; `fused=False` issues the four calls one by one) with p kept from the previous step as the initial guess (the warm start behind Table 1's ~2
V-cycles per step).  Argument marshalling only: every step runs in the CUDA
kernels behind include/gmg.h."""
import torch

from . import gmg


class PressureStepper:
    def __init__(self, n, bc, solver=gmg.GMG_RBGS, tol=1e-4, maxiter=50, device="cuda:0", fused=True,
                 **params):
        self.g = gmg.GMG(n, bc, device=device, **params)
        self.fused = fused
        self.solver, self.tol, self.maxiter = solver, tol, maxiter
        nx, ny, nz = n
        self.p = torch.zeros((nz, ny, nx), dtype=torch.float32, device=device)
        self.z = torch.empty_like(self.p)   # same buffers every step: the solve graph is reused
        self._L = None            # gmg_set_coeffs keeps the pointer: hold the tensor

    def step(self, L: torch.Tensor, ustar: torch.Tensor, wall_hi=(0.0, 0.0, 0.0)):
        """L, ustar: device tensors [3][nz][ny][nx]; ustar is projected IN PLACE.  Passing the same
        L tensor, rewritten in place, every step keeps the captured solve graph.
        Returns (status code, stats dict of the solve)."""
        self._L = L
        if self.fused:
            rc = self.g.pressure_step(L, ustar, self.p, wall_hi, tol=self.tol, maxiter=self.maxiter,
                                      solver=self.solver)
            return rc, self.g.stats()
        self.g.set_coeffs(L)
        z = self.g.divergence(ustar, wall_hi, out=self.z)
        rc = self.g.solve(self.p, z, tol=self.tol, maxiter=self.maxiter, solver=self.solver)
        st = self.g.stats()
        self.g.project(ustar, self.p)
        return rc, st

    def close(self):
        self.g.close()
