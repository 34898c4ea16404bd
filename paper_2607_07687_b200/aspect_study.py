"""Aspect-ratio study shaped like PAPER.md Fig. 2 (S3.2, lines 47-51): V-cycles to tol for the
impulsive start of a uniform flow past a sphere in an (N b) x b x b box, with the classical
isotropic coarsening and with the paper's anisotropic coarsening.

    python -m paper_2607_07687_b200.aspect_study [--base 32] [--aspects 1 2 4 8 16] [--case sphere|cylinder2d]

Needs a CUDA device (the solves run through the C-ABI library).  Inputs are synthetic
(workloads.impulsive_sphere); the paper's own cases and sizes are not reproduced."""
import argparse
import json

import torch

from . import gmg
from . import workloads as W


def run(aspects=(1, 2, 4, 8, 16), base=32, tol=1e-4, maxiter=200, case="sphere"):
    """case: "sphere" (Fig. 2 right, 3-D) or "cylinder2d" (Fig. 2 left, an (N b) x b x 1 grid)."""
    rows = []
    make = W.impulsive_sphere if case == "sphere" else W.impulsive_cylinder_2d
    for N in aspects:
        wl = make(N, base)
        L = torch.from_numpy(wl.L).cuda()
        z = torch.from_numpy(wl.z).cuda()
        row = {"aspect": N, "grid": list(wl.n)}
        for name, mode in (("iso", gmg.COARSEN_ISO), ("aniso", gmg.COARSEN_ANISO)):
            g = gmg.GMG(wl.n, wl.bc, coarsen_mode=mode)
            try:
                g.set_coeffs(L)
                p = torch.zeros_like(z)
                rc = g.solve(p, z, tol=tol, maxiter=maxiter, solver=gmg.GMG_RBGS)
                st = g.stats()
                row[name] = {"levels": g.num_levels(), "vcycles": st["iterations"],
                             "converged": rc == gmg.OK, "resid": st["resid_final_rel"],
                             "ms": st["gpu_ms"]}
            finally:
                g.close()
        rows.append(row)
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--base", type=int, default=32)
    ap.add_argument("--aspects", type=int, nargs="+", default=[1, 2, 4, 8, 16])
    ap.add_argument("--case", default="sphere", choices=["sphere", "cylinder2d"])
    ap.add_argument("--json", action="store_true")
    a = ap.parse_args()
    rows = run(a.aspects, a.base, case=a.case)
    if a.json:
        print(json.dumps(rows))
        return
    print(f"{'N':>3} {'grid':>16} | {'iso: levels':>11} {'V-cycles':>8} {'ms':>8} | "
          f"{'aniso: levels':>13} {'V-cycles':>8} {'ms':>8}")
    for r in rows:
        i, an = r["iso"], r["aniso"]
        print(f"{r['aspect']:>3} {'x'.join(map(str, r['grid'])):>16} | {i['levels']:>11} "
              f"{i['vcycles']:>8} {i['ms']:>8.2f} | {an['levels']:>13} {an['vcycles']:>8} {an['ms']:>8.2f}")


if __name__ == "__main__":
    main()
