// Internal declarations shared by the .cu files of libsp2b200.so (not part of the C ABI).
#pragma once
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/sp2_b200.h"
#include "sp2_control.cuh"

namespace sp2 {

// ---- HBM-bound kernels (sp2_elementwise.cu)
// part: scratch of gershgorin_part_floats(N) floats (per-tile row / column sums, see k_gershgorin_rows)
cudaError_t launch_gershgorin(const float* H, int N, long long ldh, float* part, double* diag, Ctrl* ctrl,
                              int num_sms, cudaStream_t st);
inline size_t gershgorin_part_floats(int N) { return 2 * (size_t)((N + 63) / 64) * (size_t)N; }
cudaError_t launch_affine_split(const float* H, int N, long long ldh, float* S, __half* hi, __half* lo, long long ld,
                                long long ldf, float scale, Ctrl* ctrl, sp2_layer_stat_t* stats, const float* thetas,
                                unsigned long long* rowsq, float* mix, float c0, unsigned long long* bn, int nb,
                                int num_sms, cudaStream_t st);
cudaError_t launch_copy_sym(const float* S, long long ld, float* D, long long ldd, int N, int num_sms, cudaStream_t st);
cudaError_t launch_one_minus(const float* M, long long ldm, float* F, long long ldo, int N, float d, int num_sms,
                             cudaStream_t st);

// Row sums of squares r_i = sum_j S_ij^2 (= diag(S^2)_i for symmetric S) are kept in 2^44 fixed point so that the
// atomic accumulation is order-independent (bit-reproducible results).  FP32 values convert exactly (power-of-two
// scale), without touching the FP64 datapath (see sp2_control.cuh).
constexpr int kRowSqBits = 44;
constexpr float kRowSqScaleF = 17592186044416.0f;          // 2^44
constexpr float kRowSqInvF = 1.0f / 17592186044416.0f;
__device__ __forceinline__ unsigned long long rowsq_fix(float x) {
    return (unsigned long long)__float2ll_rn(x * kRowSqScaleF);
}
cudaError_t launch_energy_traces(const float* X, long long ldx, const float* H, long long ldh, int N, Ctrl* ctrl,
                                 double* out, int plan, sp2_layer_stat_t* stats, const float* thetas,
                                 unsigned long long* rowsq, int num_sms, cudaStream_t st);
cudaError_t launch_split(const float* X, int N, long long ldx, __half* hi, __half* lo, long long ldo, float scale,
                         int num_sms, cudaStream_t st);

// Leading dimensions of the workspace matrices: rows are padded by 128 bytes so that walking down a column (the
// mirrored accesses of the epilogue, the 128-byte rows of a TMA box) does not stride by a power of two, which
// would map a whole panel slice onto a few L2 sets.
inline long long ws_ld_f32(int Np) { return (long long)Np + 32; }
inline long long ws_ld_f16(int Np) { return (long long)Np + 64; }

// ---- fused symmetric square layer (sp2_square_tiled.cu)
enum TileConfig { TILE_AUTO = 0, TILE_128x128 = 1, TILE_128x256 = 2, TILE_256x256_PAIR = 3,
                  TILE_128x128_ENH = 4 /* enhanced accumulation, refinement layers only */ };

// One unit of work of a layer kernel: rows [(I * E + (sub * CG + rank) * 128), +128) per CTA of supertile (I, J),
// I >= J, E = supertile edge; columns [J * E + col0, + ncols).  ncols = E except for the items of the last, partial
// round, which the host cuts into narrower ones (ncols = E/2 or E/4) so that more CTAs share that round.
struct WorkItem {
    short I, J;
    short sub, col0;
    short ncols, pad0;
    int pad1;
};

struct LayerParams {
    Ctrl* ctrl;
    sp2_layer_stat_t* stats;
    const float* thetas;           // generalized mode: [L][kThetaStride] on the device
    float* S;                      // FP32 master, Np x Np, updated in place; below the diagonal chunks only the UPPER
                                   // triangle is kept current (it is what the epilogue reads back): see k_copy_sym
    float* mix;                    // output mix M = sum_i c_i S_i (Eq. 18), same layout as S; nullptr = none
    __half* hi_out;                // next layer's operands (the other ping-pong pair)
    __half* lo_out;
    __half* hi_in;                 // this layer's operand pair (persistent mode: the output pair of odd layers)
    __half* lo_in;
    int persist;                   // 1: one launch runs layer after layer (grid barrier in between) until the control stops
    unsigned long long* rowsq_cur; // r_i of S_{n-1} (read at the diagonal, then zeroed); nullptr = tensor-core diagonal
    unsigned long long* rowsq_next;// r_i of S_n (accumulated by this launch)
    const WorkItem* items;         // work list in launch order: item w runs on CTA slot w % n_slots in round w / n_slots
    long long ld;                  // leading dimension of S (floats)
    long long ldf;                 // leading dimension of hi/lo (halves)
    int N, Np;
    int n_items;                   // length of the work list
    int n_slots;                   // CTA slots (CTAs / CG) of the launch
    float scale;                   // c = 2^k of the split
    float inv_scale2;              // 1 / c^2
    int enh_kc;                    // enhanced accumulation: K-blocks (of 64) per tensor-core accumulation chunk
    int ki_edge, ki_mid;           // K-interleave of the two rounds of an epoch (see ki_range): K-blocks per chunk at both
                                   // ends of K and in between; ki_edge = 0: one tile after the other
    int round_sync;                // 1: producers of all CTAs meet at every round boundary (keeps the wave in lockstep)
    unsigned int round_spins;      // bound of that wait in 64 ns sleeps (a CTA that is not co-resident must not hang it)
    unsigned long long cond_handle;  // cudaGraphConditionalHandle (0 = none)
    // blocked-sparse variant (reading C28): squared Frobenius norms of the 128 x 128 blocks of S_{n-1} (read)
    // and of S_n (written), nb x nb each, 2^48 fixed point; nullptr = dense.  tau^2 lives in Ctrl.
    const unsigned long long* bn_cur;
    unsigned long long* bn_next;
    int nb;
};

// Supertile edge for a tile configuration (128 or 256) and CTAs launched per supertile-slot.
int tile_super_edge(int cfg);
int tile_subs(int cfg);        // 128-row work items per supertile
int tile_cta_group(int cfg);
int layer_slots(int cfg, int n_items, int num_sms);   // CTA slots a launch of n_items uses
size_t tile_smem_bytes(int cfg);
// Launch one layer: reads hi/lo through the tensor maps (K-major, 128B swizzle, box 64 x 128), writes S, hi_out, lo_out.
// tm_hi / tm_lo: the input pair of the launch's first layer; tm_hi1 / tm_lo1: the other pair (read by the odd layers of a
// persistent launch; pass the first pair again otherwise).
cudaError_t launch_layer(int cfg, const CUtensorMap& tm_hi, const CUtensorMap& tm_lo, const CUtensorMap& tm_hi1,
                         const CUtensorMap& tm_lo1, const LayerParams& p, int num_sms, cudaStream_t st);
cudaError_t layer_kernel_setup(int cfg);   // cudaFuncSetAttribute(max dynamic smem), once per process

// ---- resident small-N kernel (sp2_resident.cu): whole solve in one launch, one CTA (pair) per matrix
struct ResidentParams {
    const float* H;                // [B][N][N]
    float* D;                      // [B][N][N]
    const long long* N_occ;        // [B] or [1], 2^40 fixed point
    int nocc_is_scalar;
    int N, B;
    int auto_bounds;
    double eps_min, eps_max;
    long long tol, eps_alt;        // 2^40 fixed point
    int kappa_q16;                 // noise-floor kappa * 2^16
    int max_layers;
    int mode;                      // MODE_STANDARD / MODE_GENERALIZED
    const float* thetas;           // generalized: [L][kThetaStride] on the device
    int accelerated;               // standard mode with the accelerated weights (section V.A, reading C27)
    const double* homo_lumo;       // accelerated: [B][2] HOMO / LUMO estimates in energy units (device)
    float scale, inv_scale2;
    sp2_layer_stat_t* stats;       // [B][max_layers] (device)
    int* n_layers;                 // [B]
    int* status;                   // [B]
    double* bounds;                // [B][2]
};
cudaError_t resident_kernel_setup();
cudaError_t launch_resident(const ResidentParams& p, int num_sms, cudaStream_t st);
size_t resident_smem_bytes(int N);

}  // namespace sp2
