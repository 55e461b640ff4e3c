// HBM-bound kernels of the path (rows a1-a3 of DESIGN.md): Gershgorin bounds, initial affine layer + first
// hi/lo split, stand-alone split.  All read H's lower triangle only (2 B per matrix element).
#include "sp2_kernels.h"
#include "sp2_ptx.cuh"

namespace sp2 {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Map a linear index t over the lower triangle (I >= J) of an nt x nt tile grid to (I, J).  Float estimate plus
// integer correction: exact, and no FP64 (the FP64 pipe of sm_100 is narrow).
__device__ __forceinline__ void tri_decode(long long t, int& I, int& J) {
    long long i = (long long)((sqrtf(8.0f * (float)t + 1.0f) - 1.0f) * 0.5f);
    while ((i + 1) * (i + 2) / 2 <= t) ++i;
    while (i * (i + 1) / 2 > t) --i;
    I = (int)i;
    J = (int)(t - i * (i + 1) / 2);
}

// Both kernels below walk 64 x 64 tiles of the lower triangle with 256 threads; thread t owns the float4 at
// row (t / 16) + 16 k, k = 0..3, columns 4 (t % 16) .. +3: a row of the tile is one 256-byte segment read by 16 lanes.
constexpr int ET = 64;
__device__ __forceinline__ float4 ld_tile4(const float* __restrict__ H, int N, long long ldh, int i, int j, bool vec) {
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (i >= N) return v;
    const float* p = H + (long long)i * ldh + j;
    if (vec && j + 3 < N) return __ldg(reinterpret_cast<const float4*>(p));
    if (j < N) v.x = __ldg(p);
    if (j + 1 < N) v.y = __ldg(p + 1);
    if (j + 2 < N) v.z = __ldg(p + 2);
    if (j + 3 < N) v.w = __ldg(p + 3);
    return v;
}
// sum over the 16 lanes that share a tile row (lanes differ in bits 0-3)
__device__ __forceinline__ float row16_sum(float v) {
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ------------------------------------------------------------------------------------------------ a1
// Gershgorin radii of the lower-triangle-symmetrised H: R_i = sum_{j<i} |H_ij| + sum_{j>i} |H_ji|: element (i,j),
// i > j, adds |H_ij| to R_i (row sum) and to R_j (column sum).  FP32 sums inside a 64 x 64 tile in a fixed order;
// every tile writes its 64 row sums and 64 column sums to slots of their own (no atomics), and the finalize kernel
// adds the slots of a row in index order in FP64: the bounds are bit-reproducible run to run.
//   part[J][i]       = row sums of tile (I = i / 64, J), J <= I
//   part[nt + I][j]  = column sums of tile (I, J = j / 64), I >= J
__global__ void __launch_bounds__(256) k_gershgorin_rows(const float* __restrict__ H, int N, long long ldh,
                                                         float* __restrict__ part, double* __restrict__ diag) {
    __shared__ float colacc[16][ET];
    const int nt = (N + ET - 1) / ET;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    const int c4 = (threadIdx.x & 15) * 4, r0 = threadIdx.x >> 4;
    const bool vec = ((ldh & 3) == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        int I, J;
        tri_decode(t, I, J);
        const int j = J * ET + c4;
        float4 v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = ld_tile4(H, N, ldh, I * ET + r0 + 16 * k, j, vec);
        float cs0 = 0.f, cs1 = 0.f, cs2 = 0.f, cs3 = 0.f;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int i = I * ET + r0 + 16 * k;
            float4 a = v[k];
            if (I == J) {                                   // diagonal tile: strictly-lower entries only; pick up H_ii
                if (i < N) {
                    if (j == i) diag[i] = (double)a.x; else if (j + 1 == i) diag[i] = (double)a.y;
                    else if (j + 2 == i) diag[i] = (double)a.z; else if (j + 3 == i) diag[i] = (double)a.w;
                }
                if (j >= i) a.x = 0.f;
                if (j + 1 >= i) a.y = 0.f;
                if (j + 2 >= i) a.z = 0.f;
                if (j + 3 >= i) a.w = 0.f;
            }
            a.x = fabsf(a.x); a.y = fabsf(a.y); a.z = fabsf(a.z); a.w = fabsf(a.w);
            cs0 += a.x; cs1 += a.y; cs2 += a.z; cs3 += a.w;
            const float rs = row16_sum((a.x + a.y) + (a.z + a.w));
            if ((threadIdx.x & 15) == 0 && i < N) part[(long long)J * N + i] = rs;
        }
        *reinterpret_cast<float4*>(&colacc[r0][c4]) = make_float4(cs0, cs1, cs2, cs3);
        __syncthreads();
        if (threadIdx.x < ET) {
            float c = 0.f;
#pragma unroll
            for (int g = 0; g < 16; ++g) c += colacc[g][threadIdx.x];
            const int jj = J * ET + threadIdx.x;
            if (jj < N) part[(long long)(nt + I) * N + jj] = c;
        }
        __syncthreads();
    }
}

// R_i from the per-tile slots, then eps_min = min_i (H_ii - R_i), eps_max = max_i (H_ii + R_i) -> ctrl.  One block per
// 64 rows; thread (r, g) adds the slots s = g, g + 4, g + 8, ... of row r in increasing order in FP64 and the four
// partial sums are combined as (p0 + p1) + (p2 + p3): a fixed order, so the bounds are bit-reproducible.  Per-block
// extrema -> ctrl->partial; the last block takes the extrema over the blocks (min / max are exact).
__global__ void __launch_bounds__(256) k_gershgorin_finalize(const float* __restrict__ part,
                                                             const double* __restrict__ diag, int N, Ctrl* ctrl) {
    __shared__ double ps[4][ET];
    __shared__ double smin[2], smax[2];
    const int nt = (N + ET - 1) / ET;
    const int Ib = blockIdx.x;
    const int r = threadIdx.x & (ET - 1), g = threadIdx.x >> 6;
    const int i = Ib * ET + r;
    // slots of a row of block Ib: row sums part[J], J = 0..Ib, then column sums part[nt + I], I = Ib..nt-1
    const int nslots = (Ib + 1) + (nt - Ib);
    double acc = 0.0;
    if (i < N)
        for (int s0 = g; s0 < nslots; s0 += 32) {           // eight loads in flight, then the adds in slot order
            float v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int sidx = s0 + 4 * u;
                const int slot = (sidx <= Ib) ? sidx : (nt + Ib + (sidx - Ib - 1));
                v[u] = (sidx < nslots) ? __ldg(part + (long long)slot * N + i) : 0.f;
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) acc += (double)v[u];
        }
    ps[g][r] = acc;
    __syncthreads();
    double lo = INFINITY, hi = -INFINITY;
    bool bad = false;
    if (threadIdx.x < ET) {
        if (i < N) {
            const double R = (ps[0][r] + ps[1][r]) + (ps[2][r] + ps[3][r]);
            lo = diag[i] - R;
            hi = diag[i] + R;
            // fmin / fmax drop NaNs: a non-finite row must poison the bounds (-> SP2_ERR_NONFINITE)
            bad = !isfinite(lo) || !isfinite(hi);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        bad = __any_sync(0xffffffffu, bad);
        if ((threadIdx.x & 31) == 0) { smin[threadIdx.x >> 5] = bad ? NAN : lo; smax[threadIdx.x >> 5] = bad ? NAN : hi; }
    }
    __syncthreads();
    __shared__ unsigned int s_last;
    if (threadIdx.x == 0) {
        const bool nan = isnan(smin[0]) || isnan(smin[1]);
        lo = fmin(smin[0], smin[1]); hi = fmax(smax[0], smax[1]);
        ctrl->partial[blockIdx.x][0] = nan ? NAN : lo;
        ctrl->partial[blockIdx.x][1] = nan ? NAN : hi;
        __threadfence();
        s_last = (atomicAdd(&ctrl->done_counter, 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (s_last != 0u && threadIdx.x < 32) {
        // last block: extrema over the blocks by one warp (strided loads, shuffle tree; min / max are exact, so any order
        // gives the same bits).  A serial loop of FP64 compares here cost more than the whole row pass (isolated FP64
        // instructions pay the datapath wake-up, see sp2_control.cuh).
        __threadfence();
        bool nan = false;
        lo = INFINITY; hi = -INFINITY;
        for (unsigned int b = threadIdx.x; b < gridDim.x; b += 32) {
            const double l = __ldcg(&ctrl->partial[b][0]), h = __ldcg(&ctrl->partial[b][1]);
            nan = nan || isnan(l) || isnan(h);
            lo = fmin(lo, l); hi = fmax(hi, h);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        nan = __any_sync(0xffffffffu, nan);
        if (threadIdx.x == 0) {
            ctrl->eps_min = nan ? NAN : lo;
            ctrl->eps_max = nan ? NAN : hi;
            ctrl->launches += 2;
            ctrl->done_counter = 0;
        }
    }
}

// ------------------------------------------------------------------------------------------------ a2
// S_0 = (eps_max I - H) / (eps_max - eps_min)  (W_0, B_0 of Alg. 1), written as FP32 master + FP16 hi/lo
// (Eqs. 12-13) at (i,j) and (j,i) from H's lower triangle (the mirror goes through shared memory so that both global
// writes are row segments); Tr S_0, ||S_0||_F^2 and the row sums of squares.  FP32 sums inside a tile (FP64 only for
// the diagonal entries), FP64 / fixed point across tiles.
// S == nullptr: the FP32 master is not written at this position (see k_affine_split)
__device__ __forceinline__ void store_s4(float* __restrict__ S, __half* __restrict__ hi, __half* __restrict__ lo,
                                         long long ld, long long ldf, int i, int j, const float (&s)[4], float scale,
                                         bool all4, const bool (&ok)[4], float* __restrict__ mix, float c0) {
    __half h[4], l[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) split_hi_lo(s[e], scale, h[e], l[e]);
    if (all4) {
        if (S) *reinterpret_cast<float4*>(S + (long long)i * ld + j) = make_float4(s[0], s[1], s[2], s[3]);
        *reinterpret_cast<uint2*>(hi + (long long)i * ldf + j) = *reinterpret_cast<uint2*>(h);
        *reinterpret_cast<uint2*>(lo + (long long)i * ldf + j) = *reinterpret_cast<uint2*>(l);
        if (mix)
            *reinterpret_cast<float4*>(mix + (long long)i * ld + j) = make_float4(c0 * s[0], c0 * s[1], c0 * s[2], c0 * s[3]);
    } else {
#pragma unroll
        for (int e = 0; e < 4; ++e)
            if (ok[e]) {
                if (mix) mix[(long long)i * ld + j + e] = c0 * s[e];
                if (S) S[(long long)i * ld + j + e] = s[e];
                hi[(long long)i * ldf + j + e] = h[e];
                lo[(long long)i * ldf + j + e] = l[e];
            }
    }
}

__global__ void __launch_bounds__(256, 4) k_affine_split(const float* __restrict__ H, int N, long long ldh,
                                                         float* __restrict__ S, __half* __restrict__ hi,
                                                         __half* __restrict__ lo, long long ld, long long ldf,
                                                         float scale, Ctrl* ctrl, sp2_layer_stat_t* stats,
                                                         const float* thetas, unsigned long long* __restrict__ rowsq,
                                                         float* __restrict__ mix, float c0,
                                                         unsigned long long* __restrict__ bn, int nb) {
    __shared__ float ts[ET][ET + 1];
    __shared__ float bsum[8];
    __shared__ float colacc[16][ET];
    __shared__ double red[8][2];
    const double e0 = ctrl->eps_min, e1 = ctrl->eps_max;
    if (!(e1 > e0) || !isfinite(e0) || !isfinite(e1)) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            // caller-given bounds were checked on the host: non-finite ones here are Gershgorin's of a non-finite H
            ctrl->error = (isfinite(e0) && isfinite(e1)) ? SP2_ERR_BOUNDS_DEGENERATE : SP2_ERR_NONFINITE;
            ctrl->running = 0;
        }
        return;
    }
    const float w0 = (float)(-1.0 / (e1 - e0));    // W_0
    const float b0 = (float)(e1 / (e1 - e0));      // B_0
    const int nt = (N + ET - 1) / ET;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    const int c4 = (threadIdx.x & 15) * 4, r0 = threadIdx.x >> 4;
    const bool vec_in = ((ldh & 3) == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
    double trS = 0.0, off2 = 0.0, dg2 = 0.0;       // ||S_0||_F^2 = 2 off2 + dg2
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        int I, J;
        tri_decode(t, I, J);
        const bool dtile = (I == J);
        const int j = J * ET + c4;
        float4 v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = ld_tile4(H, N, ldh, I * ET + r0 + 16 * k, j, vec_in);
        float offsq = 0.f;                          // squares of this thread's strictly-lower entries
        float cs[4] = {0.f, 0.f, 0.f, 0.f};         // the same per column (rows of the mirrored part)
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int lr = r0 + 16 * k, i = I * ET + lr;
            const float hv[4] = {v[k].x, v[k].y, v[k].z, v[k].w};
            float sv[4];
            bool ok[4];
            float rsq = 0.f;                        // row i: squares of its entries j <= i held by this thread
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int jj = j + e;
                ok[e] = (i < N) && (jj <= i);       // jj <= i < N
                float sx = ok[e] ? w0 * hv[e] : 0.f;
                if (ok[e] && jj == i) {
                    sx += b0;
                    const double sd = (double)sx;
                    trS += sd; dg2 += sd * sd;
                    rsq += sx * sx;
                } else {
                    const float q = sx * sx;
                    rsq += q; offsq += q; cs[e] += q;
                }
                sv[e] = sx;
                ts[lr][c4 + e] = sx;
            }
            const bool all4 = !dtile && (i < N);    // off-diagonal tile: j + 3 < J*64 + 64 <= i
            // of the FP32 master only the UPPER triangle (and the diagonal tiles) is ever read back: by the layer
            // epilogue at the mirrored address and by k_copy_sym -- below the diagonal tiles it is not written
            store_s4(dtile ? S : nullptr, hi, lo, ld, ldf, i, j, sv, scale, all4, ok, mix, c0);
            if (rowsq) {
                rsq = row16_sum(rsq);
                if ((threadIdx.x & 15) == 0 && i < N) atomicAdd(rowsq + i, rowsq_fix(rsq));
            }
        }
        off2 += (double)offsq;
        *reinterpret_cast<float4*>(&colacc[r0][c4]) = make_float4(cs[0], cs[1], cs[2], cs[3]);
        if (bn) {                                   // blocked-sparse variant: squared norms of the 128 x 128 blocks of S_0
            const float wsum = warp_sum(offsq);
            if ((threadIdx.x & 31) == 0) bsum[threadIdx.x >> 5] = wsum;
        }
        __syncthreads();
        if (bn && threadIdx.x == 0 && (I >> 1) != (J >> 1)) {
            const float tsum = ((bsum[0] + bsum[1]) + (bsum[2] + bsum[3])) + ((bsum[4] + bsum[5]) + (bsum[6] + bsum[7]));
            const unsigned long long v = (unsigned long long)__float2ll_rn(tsum * 281474976710656.0f);   // 2^48
            atomicAdd(bn + (size_t)(I >> 1) * nb + (J >> 1), v);
            atomicAdd(bn + (size_t)(J >> 1) * nb + (I >> 1), v);
        }
        if (rowsq && threadIdx.x < ET) {            // column j of the tile = row j of the mirrored part (j < i only)
            float c = 0.f;
#pragma unroll
            for (int g = 0; g < 16; ++g) c += colacc[g][threadIdx.x];
            const int jj = J * ET + threadIdx.x;
            if (jj < N && c != 0.f) atomicAdd(rowsq + jj, rowsq_fix(c));
        }
        // mirrored part: row jj = J*64 + lr, columns ii = I*64 + c4 .. +3, value s(ii, jj) for ii > jj
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int lr = r0 + 16 * k, jj = J * ET + lr, ii = I * ET + c4;
            float sv[4];
            bool ok[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                sv[e] = ts[c4 + e][lr];
                ok[e] = (ii + e < N) && (jj < ii + e);
            }
            const bool all4 = !dtile && (ii + 3 < N);
            if (jj < N) store_s4(S, hi, lo, ld, ldf, jj, ii, sv, scale, all4, ok, mix, c0);
        }
        __syncthreads();
    }
    trS = warp_sum(trS);
    double fro2 = warp_sum(2.0 * off2 + dg2);
    if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5][0] = trS; red[threadIdx.x >> 5][1] = fro2; }
    __syncthreads();
    __shared__ unsigned int s_last;
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < 8; ++w) { a += red[w][0]; b += red[w][1]; }
        ctrl->partial[blockIdx.x][0] = a;
        ctrl->partial[blockIdx.x][1] = b;
        ctrl->partial[blockIdx.x][2] = 0.0;
        __threadfence();
        s_last = (atomicAdd(&ctrl->done_counter, 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (s_last != 0u && threadIdx.x < 32) {
        // last block: one warp sums the per-block partials (lane l takes blocks l, l + 32, ... in order, then a fixed
        // shuffle tree: bit-reproducible) -- a serial FP64 loop over ~600 blocks took ~15 % of the kernel
        __threadfence();
        double s0 = 0.0, s1 = 0.0;
        for (unsigned int i = threadIdx.x; i < gridDim.x; i += 32) {
            s0 += __ldcg(&ctrl->partial[i][0]);
            s1 += __ldcg(&ctrl->partial[i][1]);
        }
        s0 = warp_sum(s0); s1 = warp_sum(s1);
        if (threadIdx.x == 0) {
            // N_S = Tr[S_0]; the control works in 2^40 fixed point (sp2_control.cuh)
            const bool fin = isfinite(s0) && isfinite(s1) && fabs(s0) < 4.0e6 && s1 < 4.0e6;
            ctrl->N_S = fin ? __double2ll_rn(s0 * kFxScale) : 0;
            ctrl->fro2 = fin ? __double2ll_rn(s1 * kFxScale) : 0;
            ctrl->nonfinite = fin ? 0 : 1;
            ctrl->n = 0;
            ctrl->done_counter = 0;
            ctrl->launches += 1;
            control_plan_next(ctrl, stats, thetas);
        }
    }
}

// ------------------------------------------------------------------------------------------------ a3
// Stand-alone split (Eqs. 12-13): hi = FP16[c X], lo = FP16[c X - hi].  4 elements per thread.
__global__ void __launch_bounds__(256) k_split_vec4(const float* __restrict__ X, int N, long long ldx,
                                                    __half* __restrict__ hi, __half* __restrict__ lo, long long ldo,
                                                    float scale) {
    const int n4 = N >> 2;
    const long long total = (long long)N * n4;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(idx / n4), j = (int)(idx % n4) * 4;
        const float4 x = __ldg(reinterpret_cast<const float4*>(X + (long long)i * ldx + j));
        __half h[4], l[4];
        split_hi_lo(x.x, scale, h[0], l[0]);
        split_hi_lo(x.y, scale, h[1], l[1]);
        split_hi_lo(x.z, scale, h[2], l[2]);
        split_hi_lo(x.w, scale, h[3], l[3]);
        *reinterpret_cast<uint2*>(hi + (long long)i * ldo + j) = *reinterpret_cast<uint2*>(h);
        *reinterpret_cast<uint2*>(lo + (long long)i * ldo + j) = *reinterpret_cast<uint2*>(l);
    }
}
__global__ void __launch_bounds__(256) k_split_scalar(const float* __restrict__ X, int N, long long ldx,
                                                      __half* __restrict__ hi, __half* __restrict__ lo,
                                                      long long ldo, float scale) {
    const long long total = (long long)N * N;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(idx / N), j = (int)(idx % N);
        __half h, l;
        split_hi_lo(__ldg(X + (long long)i * ldx + j), scale, h, l);
        hi[(long long)i * ldo + j] = h;
        lo[(long long)i * ldo + j] = l;
    }
}

// ------------------------------------------------------------------------------------------------ NEXT-1
// Observables of a symmetric X against H (both read through their lower triangles, reading C22):
//   out[0] = Tr[X H] = sum_i X_ii H_ii + 2 sum_{i>j} X_ij H_ij   (the energy alpha = Tr[D H])
//   out[1] = Tr[X],  out[2] = ||X||_F^2 = Tr[X^2]  ->  IdErr = Tr[X - X^2] = out[1] - out[2]
// FP32 products summed per thread over one tile (16 elements), FP64 across tiles; per-block partials are summed
// in fixed order by the last block.  If `plan` is set, that block also seeds the control block with N_S, N_X and
// plans layer 1 (used by the refinement, whose two layers have given thetas).
__global__ void __launch_bounds__(256) k_energy_traces(const float* __restrict__ X, long long ldx,
                                                       const float* __restrict__ H, long long ldh, int N, Ctrl* ctrl,
                                                       double* __restrict__ out, int plan, sp2_layer_stat_t* stats,
                                                       const float* thetas, unsigned long long* __restrict__ rowsq) {
    __shared__ double red[8][3];
    __shared__ float colacc[16][ET];
    const int nt = (N + ET - 1) / ET;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    const int c4 = (threadIdx.x & 15) * 4, r0 = threadIdx.x >> 4;
    const bool vx = ((ldx & 3) == 0) && ((reinterpret_cast<uintptr_t>(X) & 15) == 0);
    const bool vh = ((ldh & 3) == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
    double e = 0.0, tr = 0.0, f2 = 0.0;
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        int I, J;
        tri_decode(t, I, J);
        const int j = J * ET + c4;
        float eo = 0.f, fo = 0.f;                   // off-diagonal partial sums of this tile
        float cs[4] = {0.f, 0.f, 0.f, 0.f};         // squares per column (rows of the mirrored part)
        float4 xt[4], ht[4];                        // all eight loads of the tile in flight before the first use
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            xt[k] = ld_tile4(X, N, ldx, I * ET + r0 + 16 * k, j, vx);
            ht[k] = ld_tile4(H, N, ldh, I * ET + r0 + 16 * k, j, vh);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int i = I * ET + r0 + 16 * k;
            const float4 x4 = xt[k], h4 = ht[k];
            const float xv[4] = {x4.x, x4.y, x4.z, x4.w}, hv[4] = {h4.x, h4.y, h4.z, h4.w};
            float rsq = 0.f;                        // row i: squares of its entries j <= i held by this thread
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int jj = j + q;
                if (i < N && jj < i) {
                    const float sq = xv[q] * xv[q];
                    eo = fmaf(xv[q], hv[q], eo); fo += sq; rsq += sq; cs[q] += sq;
                } else if (i < N && jj == i) {
                    const double xd = (double)xv[q];
                    e += xd * (double)hv[q]; tr += xd; f2 += xd * xd;
                    rsq += xv[q] * xv[q];
                }
            }
            if (rowsq) {
                rsq = row16_sum(rsq);
                if ((threadIdx.x & 15) == 0 && i < N) atomicAdd(rowsq + i, rowsq_fix(rsq));
            }
        }
        if (rowsq) {                                // uniform over the block
            *reinterpret_cast<float4*>(&colacc[r0][c4]) = make_float4(cs[0], cs[1], cs[2], cs[3]);
            __syncthreads();
            if (threadIdx.x < ET) {
                float c = 0.f;
#pragma unroll
                for (int g = 0; g < 16; ++g) c += colacc[g][threadIdx.x];
                const int jc = J * ET + threadIdx.x;
                if (jc < N && c != 0.f) atomicAdd(rowsq + jc, rowsq_fix(c));
            }
            __syncthreads();
        }
        e += 2.0 * (double)eo;
        f2 += 2.0 * (double)fo;
    }
    e = warp_sum(e); tr = warp_sum(tr); f2 = warp_sum(f2);
    if ((threadIdx.x & 31) == 0) { red[threadIdx.x >> 5][0] = e; red[threadIdx.x >> 5][1] = tr; red[threadIdx.x >> 5][2] = f2; }
    __syncthreads();
    __shared__ unsigned int s_last;
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0, c = 0.0;
        for (int w = 0; w < 8; ++w) { a += red[w][0]; b += red[w][1]; c += red[w][2]; }
        ctrl->partial[blockIdx.x][0] = a;
        ctrl->partial[blockIdx.x][1] = b;
        ctrl->partial[blockIdx.x][2] = c;
        __threadfence();
        s_last = (atomicAdd(&ctrl->done_counter, 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (s_last != 0u && threadIdx.x < 32) {             // last block: one warp, fixed order (see k_affine_split)
        __threadfence();
        double s0 = 0.0, s1 = 0.0, s2 = 0.0;
        for (unsigned int i = threadIdx.x; i < gridDim.x; i += 32) {
            s0 += __ldcg(&ctrl->partial[i][0]);
            s1 += __ldcg(&ctrl->partial[i][1]);
            s2 += __ldcg(&ctrl->partial[i][2]);
        }
        s0 = warp_sum(s0); s1 = warp_sum(s1); s2 = warp_sum(s2);
        if (threadIdx.x == 0) {
            out[0] = s0; out[1] = s1; out[2] = s2;
            ctrl->done_counter = 0;
            ctrl->launches += 1;
            if (plan) {
                const bool fin = isfinite(s1) && isfinite(s2) && fabs(s1) < 4.0e6 && s2 < 4.0e6;
                ctrl->N_S = fin ? __double2ll_rn(s1 * kFxScale) : 0;
                ctrl->fro2 = fin ? __double2ll_rn(s2 * kFxScale) : 0;
                ctrl->nonfinite = fin ? 0 : 1;
                ctrl->n = 0;
                control_plan_next(ctrl, stats, thetas);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ copy-out
// D = the symmetric matrix whose UPPER triangle (incl. diagonal) is stored in S.  The layer kernel keeps only the
// upper triangle of the FP32 master current below the diagonal chunks (that is the part its epilogue reads back, at the
// mirrored address), so the result is mirrored once here instead of once per layer.  64 x 64 tiles, transposed
// through shared memory so that both global writes are row segments.
__global__ void __launch_bounds__(256) k_copy_sym(const float* __restrict__ S, long long ld, float* __restrict__ D,
                                                  long long ldd, int N) {
    __shared__ float ts[ET][ET + 1];
    const int nt = (N + ET - 1) / ET;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    const int c4 = (threadIdx.x & 15) * 4, r0 = threadIdx.x >> 4;
    const bool vs = ((ld & 3) == 0) && ((reinterpret_cast<uintptr_t>(S) & 15) == 0);
    const bool vd = ((ldd & 3) == 0) && ((reinterpret_cast<uintptr_t>(D) & 15) == 0);
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        int I, J;
        tri_decode(t, I, J);                        // I >= J: source block rows J*64.., columns I*64..
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int lr = r0 + 16 * k;
            const float4 v = ld_tile4(S, N, ld, J * ET + lr, I * ET + c4, vs);
            ts[lr][c4] = v.x; ts[lr][c4 + 1] = v.y; ts[lr][c4 + 2] = v.z; ts[lr][c4 + 3] = v.w;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int lr = r0 + 16 * k;
            float u[4], l[4];                       // upper block row lr, lower block row lr
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int lc = c4 + e;
                // diagonal tile: (lr, lc) is authoritative only for lr <= lc
                u[e] = (I != J || lr <= lc) ? ts[lr][lc] : ts[lc][lr];
                l[e] = (I != J || lc <= lr) ? ts[lc][lr] : ts[lr][lc];
            }
            const int gu = J * ET + lr, gl = I * ET + lr;
            const int cu = I * ET + c4, cl = J * ET + c4;
            if (gu < N) {
                if (vd && cu + 3 < N) *reinterpret_cast<float4*>(D + (long long)gu * ldd + cu) = make_float4(u[0], u[1], u[2], u[3]);
                else
                    for (int e = 0; e < 4; ++e) if (cu + e < N) D[(long long)gu * ldd + cu + e] = u[e];
            }
            if (I != J && gl < N) {
                if (vd && cl + 3 < N) *reinterpret_cast<float4*>(D + (long long)gl * ldd + cl) = make_float4(l[0], l[1], l[2], l[3]);
                else
                    for (int e = 0; e < 4; ++e) if (cl + e < N) D[(long long)gl * ldd + cl + e] = l[e];
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------ NEXT-2
// F = d I - M  (Eq. 18: the Fermi-operator approximation is 1 - sum_i c_i eps_i; d = 1 - c_0 after the
// change of variable of generalized_impl), N x N, M with leading dimension ldm, F with ldo.
__global__ void __launch_bounds__(256) k_one_minus(const float* __restrict__ M, long long ldm, float* __restrict__ F,
                                                   long long ldo, int N, float d) {
    const long long total = (long long)N * N;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(idx / N), j = (int)(idx % N);
        F[(long long)i * ldo + j] = (i == j ? d : 0.0f) - M[(long long)i * ldm + j];
    }
}

// ------------------------------------------------------------------------------------------------ launchers

// Grid of a persistent tile kernel: as many blocks as are co-resident (one wave), so that the grid-stride loops end
// together; more blocks than that run in waves and the last wave's blocks start late (k_copy_sym: 1184 blocks on 1036
// resident slots cost 14 %).
template <class K>
static int resident_grid(K kernel, int threads, long long work, long long cap, int num_sms) {
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
    long long g = (long long)per_sm * num_sms;
    if (cap > 0 && g > cap) g = cap;
    if (g > work) g = work;
    return (int)(g < 1 ? 1 : g);
}
cudaError_t launch_gershgorin(const float* H, int N, long long ldh, float* part, double* diag, Ctrl* ctrl,
                              int num_sms, cudaStream_t st) {
    const int nt = (N + ET - 1) / ET;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    const int grid = resident_grid(k_gershgorin_rows, 256, ntiles, 0, num_sms);
    if (nt > kMaxPartials) return cudaErrorInvalidValue;
    k_gershgorin_rows<<<grid, 256, 0, st>>>(H, N, ldh, part, diag);
    k_gershgorin_finalize<<<nt, 256, 0, st>>>(part, diag, N, ctrl);
    return cudaGetLastError();
}

cudaError_t launch_affine_split(const float* H, int N, long long ldh, float* S, __half* hi, __half* lo, long long ld,
                                long long ldf, float scale, Ctrl* ctrl, sp2_layer_stat_t* stats, const float* thetas,
                                unsigned long long* rowsq, float* mix, float c0, unsigned long long* bn, int nb,
                                int num_sms, cudaStream_t st) {
    const int nt = (N + ET - 1) / ET;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    const int grid = resident_grid(k_affine_split, 256, ntiles, kMaxPartials, num_sms);
    k_affine_split<<<grid, 256, 0, st>>>(H, N, ldh, S, hi, lo, ld, ldf, scale, ctrl, stats, thetas, rowsq, mix, c0, bn, nb);
    return cudaGetLastError();
}

cudaError_t launch_split(const float* X, int N, long long ldx, __half* hi, __half* lo, long long ldo, float scale,
                         int num_sms, cudaStream_t st) {
    const bool vec = (N % 4 == 0) && (ldx % 4 == 0) && (ldo % 4 == 0) && ((uintptr_t)X % 16 == 0) &&
                     ((uintptr_t)hi % 8 == 0) && ((uintptr_t)lo % 8 == 0);
    const long long work = vec ? (long long)N * (N / 4) : (long long)N * N;
    long long blocks = (work + 255) / 256;
    const long long cap = (long long)num_sms * 32;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    if (vec) k_split_vec4<<<(int)blocks, 256, 0, st>>>(X, N, ldx, hi, lo, ldo, scale);
    else k_split_scalar<<<(int)blocks, 256, 0, st>>>(X, N, ldx, hi, lo, ldo, scale);
    return cudaGetLastError();
}

}  // namespace sp2

namespace sp2 {
cudaError_t launch_copy_sym(const float* S, long long ld, float* D, long long ldd, int N, int num_sms, cudaStream_t st) {
    const int nt = (N + ET - 1) / ET;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    k_copy_sym<<<resident_grid(k_copy_sym, 256, ntiles, 0, num_sms), 256, 0, st>>>(S, ld, D, ldd, N);
    return cudaGetLastError();
}
cudaError_t launch_one_minus(const float* M, long long ldm, float* F, long long ldo, int N, float d, int num_sms,
                             cudaStream_t st) {
    long long blocks = ((long long)N * N + 255) / 256;
    if (blocks > (long long)num_sms * 32) blocks = (long long)num_sms * 32;
    k_one_minus<<<(int)blocks, 256, 0, st>>>(M, ldm, F, ldo, N, d);
    return cudaGetLastError();
}
cudaError_t launch_energy_traces(const float* X, long long ldx, const float* H, long long ldh, int N, Ctrl* ctrl,
                                 double* out, int plan, sp2_layer_stat_t* stats, const float* thetas,
                                 unsigned long long* rowsq, int num_sms, cudaStream_t st) {
    const int nt = (N + ET - 1) / ET;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    const int grid = resident_grid(k_energy_traces, 256, ntiles, kMaxPartials, num_sms);
    k_energy_traces<<<grid, 256, 0, st>>>(X, ldx, H, ldh, N, ctrl, out, plan, stats, thetas, rowsq);
    return cudaGetLastError();
}
}  // namespace sp2
