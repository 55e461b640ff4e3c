// Device-side branch and convergence control of Alg. 1 (stop rule P:186-190, Thm 1).
// One Ctrl block per problem lives in device memory; the last CTA of each layer kernel calls
// control_finish_layer(), so no scalar crosses to the host between layers.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/sp2_b200.h"

namespace sp2 {

constexpr int kMaxPartials = 1024;   // per-CTA FP64 partial slots (>= largest grid of a layer kernel)

enum { MODE_STANDARD = 0, MODE_GENERALIZED = 1 };

// Device layout of the per-layer scalars of the generalized network: {th1, th2, th3, c} per layer, c = weight of the
// layer's output S_n in the output mix sum_i c_i S_i (Eq. 18; 0 when no mix is formed).
constexpr int kThetaStride = 4;

struct CtrlCore {
    // ---- problem constants (written by the host before launch)
    double N_occ, eps_alt, tol;
    double eps_min, eps_max;         // spectral bounds (given, or written by the Gershgorin kernel)
    int    N, mode, max_layers, auto_bounds;
    // ---- state
    int    n;                        // layers applied so far
    int    running;                  // 1 while another layer has to run
    int    stop_reason;              // SP2_STOP_* once finished
    int    pending_stop;             // stop test of the layer in flight already fired (applied after it)
    int    sigma_prev, sigma_prev2;  // sigma_{n}, sigma_{n-1} of applied layers
    int    error;                    // sp2_status_t < 0 raised on the device
    int    launches;                 // kernels that did work (for sp2_last_launch_count)
    double N_S;                      // Tr S_n (measured)
    double fro2;                     // ||S_n||_F^2 = N_X of layer n+1
    double iderr_prev, iderr_prev2;  // IdErr_n, IdErr_{n-1}
    double nx_inflight;              // N_X of the layer in flight (exact, FP64 pre-trace)
    double acc_h, acc_l;             // accelerated scheme (section V.A): lower bound of the occupied, upper bound of
                                     // the unoccupied eigenvalues of S_n (rescaled HOMO / LUMO estimates)
    double homo, lumo;               // the caller's estimates in energy units (rescaled once the bounds are known)
    int    accelerated;              // 1: weights of reading C27 instead of sigma = +-1
    int    pad_acc_;
    double noise_kappa;              // reading C25: stop when IdErr_n <= kappa |Tr X_n(tc) - N_X|; 0 disables
    float  theta[4];                 // th1, th2, th3, c of the NEXT layer (FP32: the epilogue's arithmetic type)
    unsigned int done_counter;       // CTAs finished in the current kernel
    unsigned int round_counter;      // round-boundary check-ins of all layer kernels of this solve (round sync);
                                     // monotonic: layer n+1's targets start at n (n_rounds - 1) gridDim.x
    unsigned int round_sync_broken;  // a round wait timed out once (CTAs not co-resident): stop waiting in this solve
    unsigned int pad_rs_;
};
struct Ctrl : CtrlCore {
    double partial[kMaxPartials][4]; // per-CTA {Tr S, ||S||_F^2, Tr X (diag), unused}
};

// Decide layer n+1 from N_S = Tr S_n and N_X = ||S_n||_F^2, exactly in Alg. 1's order:
// IdErr, sigma, (W_n, B_n) -> theta, stop tests.  The stop tests belong to layer n+1 and take effect after
// that layer has been applied (reading C1 of DESIGN.md).  thetas = per-layer [L][3] list in generalized mode.
__device__ inline void control_plan_next(CtrlCore* c, sp2_layer_stat_t* stats, const double* thetas) {
    const int m = c->n + 1;                      // layer about to run
    if (c->mode == MODE_GENERALIZED) {
        if (c->n >= c->max_layers) { c->running = 0; c->stop_reason = SP2_STOP_MAX_LAYERS; return; }
        if (!(isfinite(c->N_S) && isfinite(c->fro2))) {      // a NaN/Inf in H or an overflowing network
            c->running = 0; c->stop_reason = SP2_STOP_NONFINITE; c->error = SP2_ERR_NONFINITE;
            return;
        }
        c->theta[0] = (float)thetas[kThetaStride * c->n + 0];
        c->theta[1] = (float)thetas[kThetaStride * c->n + 1];
        c->theta[2] = (float)thetas[kThetaStride * c->n + 2];
        c->theta[3] = (float)thetas[kThetaStride * c->n + 3];
        if (stats) {
            stats[m - 1].trace_X = c->fro2;
            stats[m - 1].iderr = c->N_S - c->fro2;
            stats[m - 1].sigma = 0;
            stats[m - 1].stop_reason = (m == c->max_layers) ? SP2_STOP_MAX_LAYERS : SP2_STOP_NONE;
        }
        c->running = 1;
        return;
    }
    const double N_S = c->N_S, N_X = c->fro2, N_occ = c->N_occ;
    const double iderr = N_S - N_X;                                            // IdErr_m
    if (!(isfinite(N_S) && isfinite(N_X))) {
        c->running = 0; c->stop_reason = SP2_STOP_NONFINITE; c->error = SP2_ERR_NONFINITE;
        return;
    }
    int sigma;
    if (c->accelerated) {
        // Section V.A, reading C27: A(x) = (a x + 1 - a)^2 with a = 2 / (2 - l), B(x) = 2 a x - (a x)^2
        // with a = 2 / (1 + h); the branch whose occupation is closer to N_occ (Alg. 1's rule on the new traces).
        if (m == 1) {                                   // rescale the estimates once the spectral bounds are known
            c->acc_h = (c->eps_max - c->homo) / (c->eps_max - c->eps_min);
            c->acc_l = (c->eps_max - c->lumo) / (c->eps_max - c->eps_min);
            if (!(c->acc_l >= 0.0 && c->acc_l < c->acc_h && c->acc_h <= 1.0)) {
                c->running = 0; c->error = SP2_ERR_INVALID_ARG;
                return;
            }
        }
        const double h = c->acc_h, l = c->acc_l, n_dim = (double)c->N;
        const double aA = 2.0 / (2.0 - l), aB = 2.0 / (1.0 + h);
        const double trA = aA * aA * N_X + 2.0 * aA * (1.0 - aA) * N_S + (1.0 - aA) * (1.0 - aA) * n_dim;
        const double trB = 2.0 * aB * N_S - aB * aB * N_X;
        const double d = fabs(trB - N_occ) - fabs(trA - N_occ) - (double)c->sigma_prev * c->eps_alt;
        if (d > 0.0) sigma = 1;
        else if (d < 0.0) sigma = -1;
        else sigma = (c->sigma_prev != 0) ? -c->sigma_prev : 1;
        if (sigma > 0) {
            c->theta[0] = (float)(aA * aA);
            c->theta[1] = (float)(2.0 * aA * (1.0 - aA));
            c->theta[2] = (float)((1.0 - aA) * (1.0 - aA));
            const double hl = aA * l + 1.0 - aA;
            c->acc_h = (aA * h + 1.0 - aA) * (aA * h + 1.0 - aA);
            c->acc_l = fmax((1.0 - aA) * (1.0 - aA), hl * hl);
        } else {
            c->theta[0] = (float)(-aB * aB);
            c->theta[1] = (float)(2.0 * aB);
            c->theta[2] = 0.0f;
            c->acc_h = fmin(2.0 * aB * h - aB * aB * h * h, 2.0 * aB - aB * aB);
            c->acc_l = 2.0 * aB * l - aB * aB * l * l;
        }
        c->theta[3] = 0.0f;
    } else {
        const double d = fabs(2.0 * N_S - N_X - N_occ) - fabs(N_X - N_occ) - (double)c->sigma_prev * c->eps_alt;
        if (d > 0.0) sigma = 1;
        else if (d < 0.0) sigma = -1;
        else sigma = (c->sigma_prev != 0) ? -c->sigma_prev : 1;                   // Sign(0): alternate (C4)
        c->theta[0] = (float)sigma;            // W_m = sigma I
        c->theta[1] = (float)(1 - sigma);      // B_m = (I - W_m) S_{m-1}
        c->theta[2] = 0.0f;
        c->theta[3] = 0.0f;
    }
    int pend = SP2_STOP_NONE;
    if (iderr <= 0.0) pend = SP2_STOP_IDERR_NONPOS;
    else if (!c->accelerated && m > 2 && c->sigma_prev != c->sigma_prev2 &&
             iderr > 4.5 * c->iderr_prev2 * c->iderr_prev2)   // Thm 1 holds for the plain alternating pair only
        pend = SP2_STOP_PARAM_FREE;        // sigma_{m-1} != sigma_{m-2} and IdErr_m > 4.5 IdErr_{m-2}^2
    else if (c->tol > 0.0 && iderr <= c->tol) pend = SP2_STOP_TOL;
    else if (m >= c->max_layers) pend = SP2_STOP_MAX_LAYERS;
    c->pending_stop = pend;
    c->nx_inflight = N_X;
    if (stats) {
        stats[m - 1].trace_X = N_X;
        stats[m - 1].iderr = iderr;
        stats[m - 1].sigma = sigma;
        stats[m - 1].stop_reason = pend;
    }
    c->sigma_prev2 = c->sigma_prev;
    c->sigma_prev = sigma;
    c->iderr_prev2 = c->iderr_prev;
    c->iderr_prev = iderr;
    c->running = 1;
}

// Book-keeping after layer n has been applied: N_S = Tr S_n (measured), ||S_n||_F^2, then either stop (the
// layer's own stop test had fired) or plan layer n+1.
__device__ inline void control_finish_layer(CtrlCore* c, sp2_layer_stat_t* stats, const double* thetas, double trS,
                                            double fro2, double trX) {
    c->n += 1;
    c->launches += 1;
    c->N_S = trS;
    c->fro2 = fro2;
    if (stats) {
        stats[c->n - 1].trace_S = trS;
        stats[c->n - 1].trace_X_diag = trX;
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        stats[c->n - 1].t_end_ns = t;
    }
    c->done_counter = 0;
    // (round_counter is never reset inside a solve: the layer kernel's round targets count from c->n)
    // Reading C25: "IdErr_n <= 0" at the resolution of the arithmetic.  iderr_prev = IdErr_n of the layer just
    // applied; |trX - nx_inflight| = measured error of the tensor-core trace of X_n.
    if (c->mode == MODE_STANDARD && c->pending_stop == SP2_STOP_NONE && c->n > 2 &&
        c->noise_kappa > 0.0 && c->iderr_prev <= c->noise_kappa * fabs(trX - c->nx_inflight)) {
        c->pending_stop = SP2_STOP_NOISE_FLOOR;
        if (stats) stats[c->n - 1].stop_reason = SP2_STOP_NOISE_FLOOR;
    }
    if (c->mode == MODE_STANDARD && c->pending_stop != SP2_STOP_NONE) {
        c->running = 0;
        c->stop_reason = c->pending_stop;
        return;
    }
    control_plan_next(c, stats, thetas);
}

}  // namespace sp2
