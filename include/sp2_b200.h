/* sp2_b200.h -- C ABI of libsp2b200.so: the SP2 density-matrix hot path of arxiv 2101.06385
 * ("Mixed Precision Fermi-Operator Expansion on Tensor Cores From a Machine Learning Perspective")
 * as hand-written sm_100a CUDA.  Citations: P:n = line n of the paper text.
 *
 * What the library computes (Alg. 1, with Alg. 2, as the activation):
 *   S_0 = (eps_max I - H) / (eps_max - eps_min)                      (W_0, B_0 of Alg. 1)
 *   X_n = f(S_{n-1}) = S_{n-1}^2 ~ FP32[ X0 X0 + X0 X1 + (X0 X1)^T ]   (Eq. 15) with
 *         X0 = FP16[c S], X1 = FP16[c S - X0]                         (Eqs. 12-13; c = 2^k, see opts)
 *   standard:    S_n = sigma_n X_n + (1 - sigma_n) S_{n-1},  sigma_n from the trace rule of Alg. 1
 *   generalized: S_n = th1 X_n + th2 S_{n-1} + th3 I                  (Eq. 17 in matrix form)
 * with the branch / convergence control evaluated on the device.
 *
 * Conventions for every entry point
 *   - Matrices are dense, row-major, FP32, assumed symmetric; only the LOWER triangle of H is read.
 *   - Pointers named *_dev are CUDA device pointers, *_host are host pointers; the caller owns all of
 *     them; inputs are never modified.  `stream` is a cudaStream_t passed as void* (NULL = default stream).
 *   - All work is enqueued on `stream`; each solve call ends with ONE cudaStreamSynchronize after copying
 *     the per-layer statistics back (no host round trip per layer).
 *   - A handle serialises its own calls (one solve at a time per handle; use one handle per host thread / stream)
 *     and belongs to the device that was current at sp2_create; a call with another current device returns
 *     SP2_ERR_INVALID_ARG.
 *   - Every parameter that can change a RESULT is in sp2_opts_t.  The environment is read once, at sp2_create, for
 *     four pure performance toggles only (results are bit-identical for any setting; defaults in brackets):
 *     SP2_ROUND_SYNC [1] and SP2_ROUND_SYNC_SPINS [65536] (the round synchronisation of the layer kernel and the
 *     bound of its wait), SP2_TAIL_SPLIT [1] (column strips for the last, partial round), SP2_K_INTERLEAVE [32]
 *     (K-blocks per chunk of the K-interleave of two rounds, "edge:mid" for longer end chunks, 0 = off) --
 *     DESIGN.md section 6.
 *   - Return value: SP2_OK (0); > 0 = result written but flagged; < 0 = error, outputs undefined.
 *     No exceptions, no stdout.  There is no CPU fallback: without a CUDA device calls return SP2_ERR_CUDA.
 *   - Hang guard: every mbarrier wait inside the kernels is bounded (2^26 polls, seconds); a wait that runs out --
 *     only a protocol bug or a faulted peer CTA can cause it -- executes `trap`.  The launch then fails with a
 *     sticky CUDA error, the call returns SP2_ERR_CUDA and, as after any device-side fault, the CUDA context is
 *     unusable for the caller.  (Built with -DSP2_DEBUG the kernel also prints the barrier to the device's stdout
 *     first; release builds print nothing.)
 */
#ifndef SP2_B200_H
#define SP2_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sp2_handle_s* sp2_handle_t;   /* owns workspace, TMA tensor maps, CUDA graphs */

typedef enum {
    SP2_OK = 0,
    SP2_NOT_CONVERGED = 1,          /* max_layers reached before any convergence test fired; D = S_{max_layers} */
    SP2_ERR_INVALID_ARG = -1,
    SP2_ERR_BOUNDS_DEGENERATE = -2, /* eps_max <= eps_min (given, or Gershgorin of a multiple of I) */
    SP2_ERR_NONFINITE = -3,         /* a trace became NaN/Inf */
    SP2_ERR_WORKSPACE = -4,         /* problem larger than the handle was created for */
    SP2_ERR_CUDA = -5,              /* a CUDA call failed; sp2_last_cuda_error() has the text */
    SP2_ERR_UNSUPPORTED_N = -6
} sp2_status_t;

/* stop_reason values (Alg. 1's two tests; tol / max_layers are the caller's extra tests) */
enum { SP2_STOP_NONE = 0, SP2_STOP_IDERR_NONPOS = 1, SP2_STOP_PARAM_FREE = 2, SP2_STOP_TOL = 3,
       SP2_STOP_MAX_LAYERS = 4, SP2_STOP_NONFINITE = 5,
       /* Alg. 1's first test "IdErr_n <= 0" taken at the resolution of the arithmetic (reading C25):
          after layer n, IdErr_n <= kappa |Tr X_n(tensor core) - N_X(fixed-point ||S||_F^2)|, i.e. the estimate has
          dropped below the measured error of the trace it is built from.  Reduces to test 1 in exact arithmetic. */
       SP2_STOP_NOISE_FLOOR = 6 };

/* Per-layer statistics, entry n-1 describes layer n (n = 1..n_layers), Alg. 1's notation. */
typedef struct {
    /* The three traces are accumulated on the device as 64-bit integers in 2^40 fixed point (order-independent, so
       bit-reproducible; reading C29) and converted to double by the host. */
    double trace_S;       /* N_S = Tr[S_n] after the layer: the FP32 diagonal of S_n, each entry converted exactly */
    double trace_X;       /* N_X = Tr[X_n] used by the control, evaluated as ||S_{n-1}||_F^2 (= Tr[S^2] for
                             symmetric S) while S_{n-1} was written: FP32 partial sums of <= 32 squares,
                             added as integers (relative error <= 31 * 2^-24, measured 1e-11)               */
    double trace_X_diag;  /* cross-check: sum of the diagonal of the tensor-core X_n, entries converted exactly */
    double iderr;         /* IdErr_n = N_S(before) - N_X = Tr[S_{n-1} - S_{n-1}^2]           */
    int    sigma;         /* +1: S_n = X_n ; -1: S_n = 2 S_{n-1} - X_n ; 0 in generalized runs               */
    int    stop_reason;   /* SP2_STOP_* : nonzero only on the last layer                                     */
    unsigned long long t_end_ns; /* device %globaltimer when the layer's last CTA finished (per-layer timeline) */
} sp2_layer_stat_t;

typedef struct {
    int    auto_bounds;     /* 1: Gershgorin bounds computed on the device; 0: use eps_min/eps_max verbatim  */
    double eps_min, eps_max;
    double tol;             /* > 0: also stop when IdErr_n <= tol (absolute); <= 0: paper's rule only        */
    int    max_layers;      /* 1..handle's max_layers                                                        */
    double eps_alt;         /* Alg. 1's small epsilon, default 0                                     */
    int    fp16_scale_log2; /* k: the split is applied to 2^k S (exact rescale; 0 = Eq. 13 literally).
                               -1 = library default (13): keeps X1 out of FP16's subnormal range            */
    int    control;         /* 0: device-side loop in a CUDA graph (WHILE node); 1: host-stepped (debug:
                               one sync per layer); 2: max_layers plain stream launches of the layer kernel, each
                               guarded on the device (a launch after convergence returns at once), no graph;
                               3: ONE persistent cooperative launch runs every layer, with a grid-wide barrier
                               between layers and the operand pairs swapped inside the kernel (same tiles, same
                               order, same bits as 0; measured no faster than 0: the barrier costs what the kernel
                               boundary costs -- kept as the graph-free form of the device-side loop)          */
    int    tile_config;     /* 0: choose by N; 1: 128x128 1-CTA; 2: 128x256 1-CTA (never chosen by 0: kept as the
                               comparison point of the tile-shape measurements); 3: 256x256 2-CTA;
                               4: 128x128 1-CTA with the enhanced accumulation of sp2_refine_energy in EVERY
                               layer (accuracy option, about 2x the time of 3 at large N)  */
    int    exact_diag;      /* 1 (default): diag(X_n)_i = sum_j S_ij^2 is taken from row sums of squares of the
                               FP32 S_{n-1} (FP32 partial sums added as 2^44 fixed-point integers; the same
                               identity that gives N_X = ||S||_F^2) instead of the
                               tensor-core accumulator, whose truncating FP32 accumulation biases the large
                               diagonal by ~ (3N/32) ulp, ramping along the diagonal (reading C24);
                               0: Alg. 2 literally (tensor-core diagonal). Single-matrix path only.           */
    int    accelerated;     /* 1: accelerated Deep-NN SP2 (section V.A): real-valued sigma_n from the
                               HOMO / LUMO estimates below -- each layer is the SP2 polynomial composed with the
                               steepest affine map that keeps the eigenvalue order and the range [0,1] (DESIGN.md
                               reading C27; the paper's own W_n, B_n are in its unavailable supplement).  The
                               parameter-free stop test is not applied (Theorem 1 covers the plain pair only).
                               sp2_density_matrix only.  0 (default): Alg. 1.                                  */
    double homo, lumo;      /* estimates of the highest occupied / lowest unoccupied eigenvalue of H (energy
                               units), eps_min <= homo < lumo <= eps_max; they must bound the gap from inside:
                               homo >= true HOMO, lumo <= true LUMO ("prior knowledge").  The batched
                               call takes per-matrix estimates through its own arguments instead.             */
    double noise_kappa;     /* kappa of the noise-floor stop (reading C25: Alg. 1's "IdErr_n <= 0", P:136,
                               at the resolution of the arithmetic): stop after layer n > 2 when
                               IdErr_n <= kappa |Tr X_n(tensor core) - N_X|.  < 0: library default (0.125);
                               0: test disabled (Alg. 1's printed tests, tol and max_layers only)              */
    int    enh_kc;          /* enhanced accumulation (tile_config 4, sp2_refine_energy): K-blocks of 64 the tensor
                               core accumulates before the chunk sum is folded into the error-free FP32 pair
                               (DESIGN.md section 9).  <= 0: library default (4 = 256 values of K; 2 is
                               ~10 % more accurate in idempotency for ~12 % more time, 8 the reverse)            */
    double trunc_tau;       /* blocked-sparse variant for decaying matrices (DESIGN.md section 9 NEXT-4):
                               > 0: before every square, the off-diagonal 128 x 128 blocks of S with Frobenius norm
                               <= trunc_tau count as zero (reading C28): their operand tiles are neither
                               loaded nor multiplied, and N_X = ||S'||_F^2 leaves them out.  0 (default): dense.
                               sp2_density_matrix / sp2_generalized(_wb) with tile_config 0 or 1, N <= 16384;
                               exact_diag does not apply (the diagonal of X comes from the masked products).
                               With trunc_tau > 0, sp2_density_matrix keeps N <= 256 on the layer kernel (the
                               resident one-launch path has no such variant); sp2_generalized_mix, sp2_refine_energy's
                               layers and the batched calls do not take it: _mix returns SP2_ERR_INVALID_ARG, the
                               others ignore the field.                                                          */
} sp2_opts_t;

/* Fill *o with defaults: auto_bounds=1, tol=0, max_layers=120, eps_alt=0, fp16_scale_log2=-1, control=0,
 * tile_config=0, exact_diag=1, accelerated=0, homo=lumo=0, noise_kappa=-1, enh_kc=0, trunc_tau=0. */
void sp2_default_opts(sp2_opts_t* o);

/* Create a handle able to solve one matrix up to N_max, or a batch of batch_max matrices of N <= 256,
 * with at most max_layers layers.  Allocates the device workspace up front: sp2_workspace_bytes() bytes.
 * Three more allocations happen lazily, on the first call that needs them, and stay with the handle:
 * sp2_generalized_mix's running sum (Np (Np + 32) floats, Np = N_max rounded up to 256), the two device staging
 * matrices of sp2_density_matrix_host (2 N^2 floats of the largest N seen), and the blocked-sparse variant's block
 * norms (a few KB).  sp2_workspace_bytes_lazy() returns their total for a given N_max.  The handle also caches one
 * instantiated CUDA graph per distinct (N, tile configuration, scale, flags); the cache is emptied when it reaches
 * 16 entries. */
sp2_status_t sp2_create(sp2_handle_t* h, int N_max, int batch_max, int max_layers);
sp2_status_t sp2_destroy(sp2_handle_t h);
size_t       sp2_workspace_bytes(int N_max, int batch_max, int max_layers);
size_t       sp2_workspace_bytes_lazy(int N_max);

/* Alg. 1: H (N x N, leading dimension ldh >= N) -> D (leading dimension ldd >= N).
 * stats_host: [opts->max_layers] entries (may be NULL); n_layers: layers executed (may be NULL);
 * bounds_out[2]: the spectral bounds used (may be NULL).  0 <= N_occ <= N.
 * N <= 256 with contiguous buffers (ldh == ldd == N) and default tile_config / control: solved by ONE launch of the
 * batched path's resident kernel (the matrix stays on chip across all layers; exact_diag does not apply there). */
sp2_status_t sp2_density_matrix(sp2_handle_t h, const float* H_dev, int N, int ldh, double N_occ,
                                const sp2_opts_t* opts, float* D_dev, int ldd,
                                sp2_layer_stat_t* stats_host, int* n_layers, double bounds_out[2],
                                void* stream);

/* Same call with HOST buffers: copies H to the device, solves, copies D back (end-to-end path).  Only the lower
 * triangle of H_host is read, so for N > 1024 only it is copied (row bands of 256 rows up to the band's last diagonal
 * element: about half the bytes); D_host receives the full symmetric matrix.  The three phases are serial by nature: the
 * first layer needs the bounds, which need all of H, and D exists only after the last layer. */
sp2_status_t sp2_density_matrix_host(sp2_handle_t h, const float* H_host, int N, int ldh, double N_occ,
                                     const sp2_opts_t* opts, float* D_host, int ldd,
                                     sp2_layer_stat_t* stats_host, int* n_layers, double bounds_out[2],
                                     void* stream);

/* Generalized network (Eq. 17): L fixed layers S_n = th1 S_{n-1}^2 + th2 S_{n-1} + th3 I,
 * theta_host = [L][3] doubles; no convergence test.  eps_min >= eps_max -> Gershgorin bounds.
 * opts may be NULL (defaults); only fp16_scale_log2, control, tile_config are read. */
sp2_status_t sp2_generalized(sp2_handle_t h, const float* H_dev, int N, int ldh,
                             const double* theta_host, int L, double eps_min, double eps_max,
                             const sp2_opts_t* opts, float* X_L_dev, int ldx,
                             sp2_layer_stat_t* stats_host, void* stream);

/* The same network with the output mix of Eq. 18: the optimised finite-temperature Fermi-operator
 * expansion  F~(H) = I - sum_{i=0..L} c_i E_i,  E_0 = (H - eps_min I) / (eps_max - eps_min) -- the rescaled H in
 * NATURAL order, as Eq. 17's eps_0 (reading C26; Alg. 1's S_0 is the reversed one, S_0 = I - E_0) --
 * E_n = th_{n,1} E_{n-1}^2 + th_{n,2} E_{n-1} + th_{n,3} I  (Eq. 17).  F~ then decreases with energy like the Fermi
 * function of Eq. 20.  theta_host = [L][3], c_host = [L+1] (c_0 weights E_0).  The sum is accumulated in FP32 by the layer epilogues
 * (one more N x N workspace matrix, allocated on the first call).  F_dev: N x N, leading dimension ldf.
 * tile_config 2 and 4 are not available for this call (SP2_ERR_INVALID_ARG). */
sp2_status_t sp2_generalized_mix(sp2_handle_t h, const float* H_dev, int N, int ldh, const double* theta_host,
                                 const double* c_host, int L, double eps_min, double eps_max,
                                 const sp2_opts_t* opts, float* F_dev, int ldf, sp2_layer_stat_t* stats_host,
                                 void* stream);

/* Convenience form of the same network with per-layer branch, weight and bias scalars (BASELINE north_star):
 * S_n = w_n (sigma_n X_n + (1 - sigma_n) S_{n-1}) + b_n I, i.e. theta_n = (w sigma, w (1 - sigma), b).
 * sigma == NULL means all +1. */
sp2_status_t sp2_generalized_wb(sp2_handle_t h, const float* H_dev, int N, int ldh, const int* sigma,
                                const double* weights, const double* biases, int L,
                                double eps_min, double eps_max, const sp2_opts_t* opts,
                                float* X_L_dev, int ldx, sp2_layer_stat_t* stats_host, void* stream);

/* Final refinement and energy (Eq. 16; Alg. 1's last line) -- the step right after the path.
 * S (N x N, lds >= N) is a converged SP2 iterate (D of sp2_density_matrix), last_sigma the sign of its last layer
 * (stats[n_layers-1].sigma).  Computes, as two layers composed in one step,
 *     last_sigma = -1:  D' = 2 S^2 - S^4          last_sigma = +1:  D' = (2 S - S^2)^2
 * (the alternation is continued from the last applied sign: DESIGN.md reading C15) in enhanced precision --
 * "single precision with double accumulation": FP16 hi/lo operands as in Eq. 15, but the tensor core
 * accumulates only opts->enh_kc K-blocks (default 4 = 256 values of K) at a time and the chunk sums are added in an
 * error-free FP32 pair -- and the observables Tr[X H], Tr[X], IdErr = Tr[X - X^2] of X = S (in) and X = D' (out), in
 * FP64.  H: the Hamiltonian (lower triangle read).  S_dev may equal D_dev.  opts may be NULL (defaults); only
 * fp16_scale_log2 and enh_kc are read. */
typedef struct {
    double energy_in, trace_in, iderr_in;
    double energy_out, trace_out, iderr_out;
} sp2_refine_result_t;
sp2_status_t sp2_refine_energy(sp2_handle_t h, const float* S_dev, int N, int lds, int last_sigma,
                               const float* H_dev, int ldh, const sp2_opts_t* opts, float* D_dev, int ldd,
                               sp2_refine_result_t* result, void* stream);

/* Batched small-N: B independent matrices H[B][N][N] (contiguous, N <= 256), one launch, one CTA
 * cluster per matrix, per-matrix branch sequence and stop layer.  N_occ: [B] values, or one value if
 * nocc_is_scalar.  homo_lumo: NULL, or -- with opts->accelerated = 1 -- [B][2] per-matrix HOMO / LUMO estimates in
 * energy units for the accelerated weights of section V.A (repeated small solves in molecular dynamics,
 * P:226, are that scheme's use case); opts->homo / lumo are not read by this call.  stats_host:
 * [B][opts->max_layers] (may be NULL); n_layers: [B]; status_out: [B] per-matrix sp2_status_t (may be NULL).
 * Returns the worst per-matrix status. */
sp2_status_t sp2_density_matrix_batched(sp2_handle_t h, const float* H_dev, int N, int B,
                                        const double* N_occ, int nocc_is_scalar, const double* homo_lumo,
                                        const sp2_opts_t* opts, float* D_dev, sp2_layer_stat_t* stats_host,
                                        int* n_layers, int* status_out, void* stream);

/* The generalized network (Eq. 17) on a batch of small matrices: the same L layers
 * S_n = th1 S_{n-1}^2 + th2 S_{n-1} + th3 I (theta_host = [L][3], shared by the batch) applied to each of the B
 * inputs H[B][N][N] (N <= 256), one launch.  eps_min >= eps_max -> per-matrix Gershgorin bounds.  X_L_dev:
 * [B][N][N]; stats_host: [B][L] (may be NULL); status_out: [B] (may be NULL).  opts may be NULL; only
 * fp16_scale_log2 is read. */
sp2_status_t sp2_generalized_batched(sp2_handle_t h, const float* H_dev, int N, int B, const double* theta_host,
                                     int L, double eps_min, double eps_max, const sp2_opts_t* opts,
                                     float* X_L_dev, sp2_layer_stat_t* stats_host, int* status_out, void* stream);

/* Stand-alone pieces of the path (rows a1, a3 of DESIGN.md), asynchronous on `stream` except where noted. */
/* Eqs. 12-13: hi = FP16[2^k X], lo = FP16[2^k X - hi]; X N x N (ldx), hi/lo N x N (ldo), as uint16 bits */
sp2_status_t sp2_split_fp16(const float* X_dev, int N, int ldx, unsigned short* hi_dev, unsigned short* lo_dev,
                            int ldo, int fp16_scale_log2, void* stream);
/* Gershgorin bounds of the lower-triangle-symmetrised H; synchronises; bounds_host[2] = {eps_min, eps_max}. */
sp2_status_t sp2_gershgorin(sp2_handle_t h, const float* H_dev, int N, int ldh, double bounds_host[2], void* stream);

/* Gershgorin bounds WITHOUT any allocation, for callers that cannot call cudaMalloc and so cannot own a handle
 * (sp2_create allocates): hosts whose own arena or caching allocator already holds all of HBM, so that a library's
 * cudaMalloc fails although the arena has room; time-step loops that cannot take the device-wide synchronisation a
 * cudaMalloc / cudaFree implies; plug-ins that receive only pointers and a stream.  Same kernels and same bits as
 * sp2_gershgorin; the scratch they need (per-tile sums, diagonal, per-block extrema) is a static __device__ array inside
 * the library: sp2_gershgorin_static_bytes() bytes (about 2.2 MB) that every GPU which loads libsp2b200.so holds until
 * the process exits.
 *   H_dev       in : N x N, leading dimension ldh >= N, device memory, lower triangle read, not modified
 *   bounds_dev  out: 2 doubles in DEVICE memory, {eps_min, eps_max}; NaN, NaN if a row of H is not finite
 *   N           1 <= N <= SP2_GERSHGORIN_STATIC_MAX_N; larger N returns SP2_ERR_UNSUPPORTED_N and enqueues nothing
 *                   (sp2_gershgorin_static_last_error() has the sentence; use sp2_gershgorin with a handle instead)
 * The call only enqueues on `stream` (one 4-byte memset, two kernels, one 16-byte device-to-device copy) and returns;
 * it does not synchronise and calls no cudaMalloc, cudaFree or other allocating routine.
 *   - First call on a device: it also asks the runtime for the array's address on that device (cudaGetSymbolAddress,
 *     with that device current) and for the SM count, which makes the runtime load the kernels.  Make this first call
 *     before any stream capture; later calls on that device skip the set-up.
 *   - All calls on a device share the one array, and it keeps the previous call's contents.  The call clears the one
 *     word that must start at zero itself; everything else it reads it has written first.  Two calls that can run on the
 *     GPU at the same time (different streams without an event between them, or two host threads) race on the array and
 *     return garbage: order them. */
#define SP2_GERSHGORIN_STATIC_MAX_N 4096
sp2_status_t sp2_gershgorin_static(const float* H_dev, int N, int ldh, double* bounds_dev, void* stream);
int          sp2_gershgorin_static_max_n(void);       /* SP2_GERSHGORIN_STATIC_MAX_N of the loaded library */
size_t       sp2_gershgorin_static_bytes(void);       /* size of the static scratch, per GPU               */
const char*  sp2_gershgorin_static_last_error(void);  /* text of this thread's last failed call, "" if none */

const char* sp2_status_string(sp2_status_t s);
const char* sp2_last_cuda_error(void);
/* Number of kernels the last solve call on this handle launched (graph nodes executed are counted by the
 * device-side layer counter: setup kernels + layers + copy-out). */
int         sp2_last_launch_count(sp2_handle_t h);
/* Device-side durations (CUDA events on `stream`) of the three phases of the last sp2_density_matrix_host call on
 * this handle, in ms: {host -> device copy of H, the solve, device -> host copy of D}. */
void        sp2_last_host_timing(sp2_handle_t h, double ms[3]);
/* Bytes the last sp2_density_matrix_host call on this handle copied: out[0] host -> device, out[1] device -> host. */
void        sp2_last_host_bytes(sp2_handle_t h, double out[2]);
/* Blocked-sparse variant (opts->trunc_tau > 0): out[0] = 128-wide block products the tensor cores executed during the
 * last single-matrix solve on this handle, summed over tiles and layers; out[1] = what a dense solve of the same layers
 * would have executed.  Both 0 after a dense solve. */
void        sp2_last_sparse_work(sp2_handle_t h, double out[2]);
/* Diagnostic: 1 if, during the last single-matrix solve on this handle, a round-synchronisation wait of the layer
 * kernel ran out and the kernel gave the synchronisation up (performance only: results are unaffected). */
int         sp2_last_round_sync_broken(sp2_handle_t h);
const char* sp2_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SP2_B200_H */
