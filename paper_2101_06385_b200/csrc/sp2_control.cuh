// Device-side branch and convergence control of Alg. 1 (stop rule P:186-190, Thm 1).
// One Ctrl block per problem lives in device memory; the last CTA of each layer kernel calls
// control_finish_layer(), so no scalar crosses to the host between layers.
//
// Arithmetic: every trace is a 64-bit integer in 2^40 FIXED POINT, and the control step uses integer arithmetic only.
// Why not FP64: on this part the FP64 datapath sleeps after a few idle cycles and an isolated FP64 instruction pays
// ~170 cycles to wake it (measured: 1 DFMA + 16 FFMAs = 260 cycles per iteration against 84 for the sum of their
// latencies; back-to-back DFMAs run at 9).  The ~40 FP64 instructions of an FP64 control step, interleaved with
// integer code, cost ~6000 cycles -- as much as a whole N = 256 layer on the tensor cores -- and the FP64 shuffle
// reductions in front of it as much again.  Fixed point is also exact where FP64 is not: integer adds do not round,
// so sums are order-independent (bit-reproducible) and the subtraction IdErr = N_S - N_X itself loses nothing.  An FP32
// value v converts exactly as llrint(v 2^40) for |v| < 8.4e6 (resolution 9.1e-13): all traces of a spectrum in [0, 1]
// with N <= 2^22 fit.  What is NOT exact is N_X = ||S||_F^2: only Tr S (and the diagonal squares) are converted element
// by element; off-diagonal squares are first summed in FP32 over at most 32 elements and that partial sum is converted,
// so N_X carries up to 31 * 2^-24 relative error in the worst case (measured 1e-11 relative = 5e-8 absolute at
// N = 16384, tests/test_gpu_fullsize.py).  The host converts the per-layer statistics back to doubles.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/sp2_b200.h"

namespace sp2 {

constexpr int kMaxPartials = 1024;   // per-CTA partial slots (>= largest grid of a layer kernel)

enum { MODE_STANDARD = 0, MODE_GENERALIZED = 1 };

// Device layout of the per-layer scalars of the generalized network: {th1, th2, th3, c} per layer (FP32, the epilogue's
// arithmetic type), c = weight of the layer's output S_n in the output mix sum_i c_i S_i (Eq. 18; 0 when no
// mix is formed).
constexpr int kThetaStride = 4;

// ---- 2^40 fixed point
typedef long long fx_t;
constexpr int kFxBits = 40;
constexpr float kFxScaleF = 1099511627776.0f;             // 2^40
constexpr double kFxScale = 1099511627776.0;
constexpr double kFxInv = 1.0 / 1099511627776.0;
constexpr float kFxInvF = 1.0f / 1099511627776.0f;
__device__ __forceinline__ fx_t fx_from_float(float x) { return __float2ll_rn(x * kFxScaleF); }
// x^2 exactly: the product and its rounding error, both converted
__device__ __forceinline__ fx_t fx_square(float x) {
    const float p = x * x;
    return fx_from_float(p) + fx_from_float(fmaf(x, x, -p));
}
__host__ __device__ inline double fx_to_double(fx_t v) { return (double)v * kFxInv; }
inline fx_t fx_from_double_host(double x) { return (fx_t)llrint(x * kFxScale); }

struct CtrlCore {
    // ---- problem constants (written by the host before launch)
    fx_t   N_occ, eps_alt, tol;      // fixed point; tol <= 0: no tolerance test
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
    fx_t   N_S;                      // Tr S_n (measured)
    fx_t   fro2;                     // ||S_n||_F^2 = N_X of layer n+1
    fx_t   iderr_prev, iderr_prev2;  // IdErr_n, IdErr_{n-1}
    fx_t   nx_inflight;              // N_X of the layer in flight: ||S_{n-1}||_F^2 from the fixed-point sums (see above)
    int    nonfinite;                // a trace of the current iterate was NaN / Inf / out of range
    int    kappa_q16;                // reading C25: stop when IdErr_n <= kappa |Tr X_n(tc) - N_X|; kappa * 2^16; 0 disables
    float  acc_h, acc_l;             // accelerated scheme (section V.A): lower bound of the occupied, upper bound of
                                     // the unoccupied eigenvalues of S_n (rescaled HOMO / LUMO estimates)
    double homo, lumo;               // the caller's estimates in energy units (rescaled once the bounds are known)
    int    accelerated;              // 1: weights of reading C27 instead of sigma = +-1
    int    pad_acc_;
    float  theta[4];                 // th1, th2, th3, c of the NEXT layer
    unsigned int done_counter;       // CTAs finished in the current kernel
    unsigned int round_counter;      // round-boundary check-ins of all layer kernels of this solve (round sync);
                                     // monotonic: layer n+1's targets start at n (n_rounds - 1) gridDim.x
    unsigned int round_sync_broken;  // a round wait timed out once (CTAs not co-resident): stop waiting in this solve
    int layer_gen;                   // persistent mode: layers applied, published with release semantics (grid barrier)
    // blocked-sparse variant (reading C28)
    unsigned long long tau2_fx48;    // tau^2 in 2^48 fixed point (block norms^2 are compared with it)
    unsigned long long work_active;  // 128-wide K-blocks the MMA warps multiplied, summed over tiles and layers
    unsigned long long work_dense;   // ... and how many a dense layer would have
};
struct Ctrl : CtrlCore {
    alignas(32) double partial[kMaxPartials][4]; // HBM kernels (bounds, initial layer, observables): per-CTA FP64 partial sums
    alignas(32) fx_t ipartial[kMaxPartials][4];  // layer kernel: per-CTA {Tr S, ||S||_F^2, Tr X (diag), non-finite flag}
};

// The statistics travel as raw fixed-point integers in the double-typed fields; the host converts them.
__device__ __forceinline__ void stat_store(double* field, fx_t v) { *reinterpret_cast<fx_t*>(field) = v; }

// a 2^41 > 9 b^2 for 0 < a, 0 <= b < 2^60 (128-bit integers): IdErr_n > 4.5 IdErr_{n-2}^2 in 2^40 fixed point
__device__ __forceinline__ bool fx_gt_4p5_square(fx_t a, fx_t b) {
    const unsigned long long ua = (unsigned long long)a, ub = (unsigned long long)b;
    const unsigned long long lhs_hi = ua >> 23, lhs_lo = ua << 41;
    const unsigned long long sq_hi = __umul64hi(ub, ub), sq_lo = ub * ub;
    const unsigned long long rhs_lo = sq_lo * 9ull, rhs_hi = sq_hi * 9ull + __umul64hi(sq_lo, 9ull);
    return lhs_hi > rhs_hi || (lhs_hi == rhs_hi && lhs_lo > rhs_lo);
}
__device__ __forceinline__ fx_t fx_abs(fx_t v) { return v < 0 ? -v : v; }

// Decide layer n+1 from N_S = Tr S_n and N_X = ||S_n||_F^2, exactly in Alg. 1's order:
// IdErr, sigma, (W_n, B_n) -> theta, stop tests.  The stop tests belong to layer n+1 and take effect after
// that layer has been applied (reading C1 of DESIGN.md).  thetas = per-layer [L][kThetaStride] list in generalized mode.
__device__ inline void control_plan_next(CtrlCore* c, sp2_layer_stat_t* stats, const float* thetas) {
    const int m = c->n + 1;                      // layer about to run
    if (c->mode == MODE_GENERALIZED) {
        if (c->n >= c->max_layers) { c->running = 0; c->stop_reason = SP2_STOP_MAX_LAYERS; return; }
        if (c->nonfinite) {                      // a NaN/Inf in H or an overflowing network
            c->running = 0; c->stop_reason = SP2_STOP_NONFINITE; c->error = SP2_ERR_NONFINITE;
            return;
        }
        c->theta[0] = thetas[kThetaStride * c->n + 0];
        c->theta[1] = thetas[kThetaStride * c->n + 1];
        c->theta[2] = thetas[kThetaStride * c->n + 2];
        c->theta[3] = thetas[kThetaStride * c->n + 3];
        if (stats) {
            stat_store(&stats[m - 1].trace_X, c->fro2);
            stat_store(&stats[m - 1].iderr, c->N_S - c->fro2);
            stats[m - 1].sigma = 0;
            stats[m - 1].stop_reason = (m == c->max_layers) ? SP2_STOP_MAX_LAYERS : SP2_STOP_NONE;
        }
        c->running = 1;
        return;
    }
    const fx_t N_S = c->N_S, N_X = c->fro2, N_occ = c->N_occ;
    const fx_t iderr = N_S - N_X;                                            // IdErr_m
    if (c->nonfinite) {
        c->running = 0; c->stop_reason = SP2_STOP_NONFINITE; c->error = SP2_ERR_NONFINITE;
        return;
    }
    int sigma;
    if (c->accelerated) {
        // Section V.A, reading C27: A(x) = (a x + 1 - a)^2 with a = 2 / (2 - l), B(x) = 2 a x - (a x)^2
        // with a = 2 / (1 + h); the branch whose occupation is closer to N_occ (Alg. 1's rule on the new traces).
        if (m == 1) {                                   // rescale the estimates once the spectral bounds are known
            const double w = c->eps_max - c->eps_min;
            c->acc_h = (float)(c->eps_max - c->homo) / (float)w;
            c->acc_l = (float)(c->eps_max - c->lumo) / (float)w;
            if (!(c->acc_l >= 0.f && c->acc_l < c->acc_h && c->acc_h <= 1.f)) {
                c->running = 0; c->error = SP2_ERR_INVALID_ARG;
                return;
            }
        }
        const float h = c->acc_h, l = c->acc_l;
        const float aA = 2.f / (2.f - l), aB = 2.f / (1.f + h);
        const float uA = -l / (2.f - l);                 // 1 - aA without cancellation
        const float uB = (h - 1.f) / (1.f + h);          // 1 - aB
        // occupation errors of the two candidates from the DEVIATIONS of the traces (the coefficients of each
        // candidate sum to one): Tr A - N_occ = a^2 dX + 2 a (1 - a) dS + (1 - a)^2 (N - N_occ),
        //                        Tr B - N_occ = 2 a dS - a^2 dX - (1 - a)^2 N_occ
        const float dS = (float)(N_S - N_occ) * kFxInvF, dX = (float)(N_X - N_occ) * kFxInvF;
        const float nocc = (float)N_occ * kFxInvF, nrem = (float)c->N - nocc;
        const float eA = aA * aA * dX + 2.f * aA * uA * dS + uA * uA * nrem;
        const float eB = 2.f * aB * dS - aB * aB * dX - uB * uB * nocc;
        const float d = fabsf(eB) - fabsf(eA) - (float)c->sigma_prev * ((float)c->eps_alt * kFxInvF);
        if (d > 0.f) sigma = 1;
        else if (d < 0.f) sigma = -1;
        else sigma = (c->sigma_prev != 0) ? -c->sigma_prev : 1;
        if (sigma > 0) {
            c->theta[0] = aA * aA;
            c->theta[1] = 2.f * aA * uA;
            c->theta[2] = uA * uA;
            const float hl = aA * l + uA;
            c->acc_h = (aA * h + uA) * (aA * h + uA);
            c->acc_l = fmaxf(uA * uA, hl * hl);
        } else {
            c->theta[0] = -aB * aB;
            c->theta[1] = 2.f * aB;
            c->theta[2] = 0.0f;
            c->acc_h = fminf(2.f * aB * h - aB * aB * h * h, 2.f * aB - aB * aB);
            c->acc_l = 2.f * aB * l - aB * aB * l * l;
        }
        c->theta[3] = 0.0f;
    } else {
        const fx_t d = fx_abs(2 * N_S - N_X - N_occ) - fx_abs(N_X - N_occ) - (fx_t)c->sigma_prev * c->eps_alt;
        if (d > 0) sigma = 1;
        else if (d < 0) sigma = -1;
        else sigma = (c->sigma_prev != 0) ? -c->sigma_prev : 1;                   // Sign(0): alternate (C4)
        c->theta[0] = (float)sigma;            // W_m = sigma I
        c->theta[1] = (float)(1 - sigma);      // B_m = (I - W_m) S_{m-1}
        c->theta[2] = 0.0f;
        c->theta[3] = 0.0f;
    }
    int pend = SP2_STOP_NONE;
    if (iderr <= 0) pend = SP2_STOP_IDERR_NONPOS;
    else if (!c->accelerated && m > 2 && c->sigma_prev != c->sigma_prev2 &&
             fx_gt_4p5_square(iderr, c->iderr_prev2))     // Thm 1 holds for the plain alternating pair only
        pend = SP2_STOP_PARAM_FREE;        // sigma_{m-1} != sigma_{m-2} and IdErr_m > 4.5 IdErr_{m-2}^2
    else if (c->tol > 0 && iderr <= c->tol) pend = SP2_STOP_TOL;
    else if (m >= c->max_layers) pend = SP2_STOP_MAX_LAYERS;
    c->pending_stop = pend;
    c->nx_inflight = N_X;
    if (stats) {
        stat_store(&stats[m - 1].trace_X, N_X);
        stat_store(&stats[m - 1].iderr, iderr);
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
__device__ inline void control_finish_layer(CtrlCore* c, sp2_layer_stat_t* stats, const float* thetas, fx_t trS,
                                            fx_t fro2, fx_t trX, bool nonfinite) {
    c->n += 1;
    c->launches += 1;
    c->N_S = trS;
    c->fro2 = fro2;
    c->nonfinite = nonfinite ? 1 : 0;
    if (stats) {
        stat_store(&stats[c->n - 1].trace_S, trS);
        stat_store(&stats[c->n - 1].trace_X_diag, trX);
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        stats[c->n - 1].t_end_ns = t;
    }
    c->done_counter = 0;
    // (round_counter is never reset inside a solve: the layer kernel's round targets count from c->n)
    // Reading C25: "IdErr_n <= 0" at the resolution of the arithmetic.  iderr_prev = IdErr_n of the layer just
    // applied; |trX - nx_inflight| = measured error of the tensor-core trace of X_n.
    if (c->mode == MODE_STANDARD && c->pending_stop == SP2_STOP_NONE && c->n > 2 && c->kappa_q16 > 0 && !nonfinite) {
        // IdErr_n <= kappa err with kappa = kappa_q16 / 2^16: 128-bit product, shifted right by 16
        const unsigned long long err = (unsigned long long)fx_abs(trX - c->nx_inflight);
        const unsigned long long plo = err * (unsigned long long)c->kappa_q16;
        const unsigned long long phi = __umul64hi(err, (unsigned long long)c->kappa_q16);
        const bool below = (phi >> 16) != 0ull ||                       // kappa err >= 2^64 / 2^16: above any IdErr
                           (unsigned long long)c->iderr_prev <= ((phi << 48) | (plo >> 16));
        if (below) {
            c->pending_stop = SP2_STOP_NOISE_FLOOR;
            if (stats) stats[c->n - 1].stop_reason = SP2_STOP_NOISE_FLOOR;
        }
    }
    if (c->mode == MODE_STANDARD && c->pending_stop != SP2_STOP_NONE) {
        c->running = 0;
        c->stop_reason = c->pending_stop;
        return;
    }
    control_plan_next(c, stats, thetas);
}

}  // namespace sp2
