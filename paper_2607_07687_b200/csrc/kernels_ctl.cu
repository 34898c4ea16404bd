// kernels_ctl.cu -- single-thread control kernels: the solve loop's scalar logic runs on the
// device so that a whole solve is one CUDA-graph launch (a WHILE conditional node) with no
// host round trip (BASELINE.json:north_star).  `cond` is the graph's conditional handle
// (use_cond = 0 for the plain-launch, host-driven loop used when graphs are disabled).
//
// GMG-RBGS loop and adaptive relaxation: DESIGN.md readings O8, O9 (PAPER.md:43 S3.1 "relaxation
// factor adapts to residual growth or decay after each V-cycle").  PCG recurrences: reading O10
// (PAPER.md:31, 39).
#include "gmg_internal.h"

namespace gmgk {

__device__ __forceinline__ void set_cond(cudaGraphConditionalHandle cond, int use_cond, int go) {
    if (use_cond) cudaGraphSetConditional(cond, go ? 1u : 0u);
}

// omega of the cycle AFTER the one about to run, if that one shrinks the residual (reading O8's
// decay branch; the same operations as k_ctl_rbgs_cycle_end, so the values compare equal)
__device__ __forceinline__ double speculate_omega(const DevScalars* sc) {
    if (!sc->adaptive) return sc->omega;
    double w = sc->omega + sc->omega_up;
    if (!(w < 1.0)) w = 1.0;
    return w;
}

__global__ void k_ctl_init(DevScalars* sc, double tol, int maxiter, int adaptive, double omega_min,
                           double omega_down, double omega_up, int predict) {
    sc->predict = predict;
    sc->expect_last = 0;
    sc->run_s1n = 1;
    sc->need_first = 0;
    sc->tol = tol;
    sc->maxiter = maxiter;
    sc->adaptive = adaptive;
    sc->omega_min = omega_min;
    sc->omega_down = omega_down;
    sc->omega_up = omega_up;
    sc->omega_one = 1.0f;
    sc->omega_f = (float)sc->omega;
    sc->iter = 0;
    sc->status = GMG_OK;
    sc->done = 0;
}

void ctl_init(DevScalars* sc, double tol, int maxiter, int adaptive, double omega_min,
              double omega_down, double omega_up, int predict, cudaStream_t s) {
    k_ctl_init<<<1, 1, 0, s>>>(sc, tol, maxiter, adaptive, omega_min, omega_down, omega_up, predict);
}

// After the reference norm (red[RREF]) and the initial residual norm (red[RR]).
__global__ void k_ctl_begin(DevScalars* sc, double* hist, double* omegas,
                            cudaGraphConditionalHandle cond, int use_cond) {
    const double r_ref = sqrt(sc->red[RED_RREF]);
    const double rho = sqrt(sc->red[RED_RR]);
    sc->r_ref = r_ref;
    sc->rho = rho;
    sc->rho_prev = rho;
    sc->iter = 0;
    sc->beta = 0.0;
    sc->alpha = 0.0;
    sc->rho_cg = 1.0;
    int done;
    if (r_ref == 0.0) {  // zero right-hand side: 0 iterations, p unchanged
        hist[0] = 0.0;
        sc->status = GMG_OK;
        done = 1;
    } else {
        hist[0] = rho / r_ref;
        // reading O9 as the oracle writes it: go on while rho > tol r_ref, converged iff
        // rho <= tol r_ref -- a NaN norm (NaN/Inf in z or p) is neither: stop, NOT converged
        const bool fin = isfinite(rho) && isfinite(r_ref);       // overflowed FP32 squares give Inf
        const bool conv = fin && rho <= sc->tol * r_ref;
        const bool go = fin && rho > sc->tol * r_ref && sc->maxiter > 0;
        sc->status = conv ? GMG_OK : GMG_NOT_CONVERGED;
        done = !go;
    }
    if (omegas) omegas[0] = sc->omega;
    sc->omega_f = (float)sc->omega;
    sc->omega_spec_f = (float)speculate_omega(sc);
    sc->redo_first = 0;
    sc->need_first = 0;
    sc->expect_last = (!done && sc->predict && sc->maxiter <= 1) ? 1 : 0;  // no rate known yet
    sc->run_s1n = !sc->expect_last;
    sc->done = done;
    set_cond(cond, use_cond, !done);
}

void ctl_begin(DevScalars* sc, double* hist, double* omegas, cudaGraphConditionalHandle cond,
               int use_cond, cudaStream_t s) {
    k_ctl_begin<<<1, 1, 0, s>>>(sc, hist, omegas, cond, use_cond);
}

// After a V-cycle and the new residual norm (red[RR]):  O8 omega update, O9 stopping test.
__global__ void k_ctl_rbgs_cycle_end(DevScalars* sc, double* hist, double* omegas,
                                     cudaGraphConditionalHandle cond, int use_cond) {
    const int k = sc->iter + 1;
    const double rho_new = sqrt(sc->red[RED_RR]);
    hist[k] = rho_new / sc->r_ref;
    if (sc->adaptive) {
        double w = sc->omega;
        if (rho_new > sc->rho) {  // growth -> under-relax more
            w -= sc->omega_down;
            if (!(w > sc->omega_min)) w = sc->omega_min;
        } else {                  // decay -> recover slowly
            w += sc->omega_up;
            if (!(w < 1.0)) w = 1.0;
        }
        sc->omega = w;
        sc->omega_f = (float)w;
    }
    sc->rho_prev = sc->rho;
    sc->rho = rho_new;
    sc->iter = k;
    const bool fin = isfinite(rho_new) && isfinite(sc->r_ref);
    const bool conv = fin && rho_new <= sc->tol * sc->r_ref;        // false for a NaN / Inf norm ...
    const bool go = fin && rho_new > sc->tol * sc->r_ref && k < sc->maxiter;   // ... and so is this
    sc->status = conv ? GMG_OK : GMG_NOT_CONVERGED;
    const int done = !go;
    if (!done) omegas[k] = sc->omega;
    // fused_norm path.  This cycle's norm came either from the next cycle's first sweep, which then
    // already ran with omega_spec_f (re-run it if the omega update went the other way), or -- the
    // cycle was expected to be the last -- from the plain norm pass, and that sweep is still to run.
    if (sc->expect_last) {
        sc->need_first = !done;
        sc->redo_first = 0;
    } else {
        sc->need_first = 0;
        sc->redo_first = (!done && sc->omega_f != sc->omega_spec_f) ? 1 : 0;
    }
    sc->omega_spec_f = (float)speculate_omega(sc);
    // expect the NEXT cycle to be the last if it is the maxiter-th, or if one more reduction by the
    // factor just seen lands a factor two below the tolerance
    const double rho_old = sc->rho_prev;   // the norm before this cycle
    const bool rate_says = rho_new < rho_old && 2.0 * rho_new * (rho_new / rho_old) <= sc->tol * sc->r_ref;
    sc->expect_last = (!done && sc->predict && (k + 1 >= sc->maxiter || rate_says)) ? 1 : 0;
    sc->run_s1n = !sc->expect_last;
    sc->done = done;
    set_cond(cond, use_cond, !done);
}

void ctl_rbgs_cycle_end(DevScalars* sc, double* hist, double* omegas,
                        cudaGraphConditionalHandle cond, int use_cond, cudaStream_t s) {
    k_ctl_rbgs_cycle_end<<<1, 1, 0, s>>>(sc, hist, omegas, cond, use_cond);
}

// PCG: after p, r updates and red[RR] = r.r (recursive residual drives the test).
__global__ void k_ctl_pcg_check(DevScalars* sc, double* hist, cudaGraphConditionalHandle cond,
                                int use_cond) {
    if (sc->status == GMG_EBREAKDOWN) {
        sc->done = 1;
        set_cond(cond, use_cond, 0);
        return;
    }
    const int k = sc->iter + 1;
    const double rn = sqrt(sc->red[RED_RR]);
    hist[k] = rn / sc->r_ref;
    sc->rho_prev = sc->rho;
    sc->rho = rn;
    sc->iter = k;
    const bool fin = isfinite(rn) && isfinite(sc->r_ref);
    const bool conv = fin && rn <= sc->tol * sc->r_ref;      // a NaN / Inf norm: not converged, stop
    const bool go = fin && rn > sc->tol * sc->r_ref && k < sc->maxiter;
    sc->status = conv ? GMG_OK : GMG_NOT_CONVERGED;
    const int done = !go;
    sc->done = done;
    set_cond(cond, use_cond, !done);
}
void ctl_pcg_check(DevScalars* sc, double* hist, cudaGraphConditionalHandle cond, int use_cond,
                   cudaStream_t s) {
    k_ctl_pcg_check<<<1, 1, 0, s>>>(sc, hist, cond, use_cond);
}

__global__ void k_ctl_set_hook_omega(DevScalars* sc, float omega) { sc->omega_hook = omega; }
void ctl_set_hook_omega(DevScalars* sc, float omega, cudaStream_t s) {
    k_ctl_set_hook_omega<<<1, 1, 0, s>>>(sc, omega);
}

__global__ void k_ctl_set_omega(DevScalars* sc, double omega) {
    sc->omega = omega;
    sc->omega_f = (float)omega;
    sc->omega_one = 1.0f;
}
void ctl_set_omega(DevScalars* sc, double omega, cudaStream_t s) {
    k_ctl_set_omega<<<1, 1, 0, s>>>(sc, omega);
}

}  // namespace gmgk
