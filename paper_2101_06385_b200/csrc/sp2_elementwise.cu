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

// Map a linear index t over the lower triangle (I >= J) of an nt x nt tile grid to (I, J).
__device__ __forceinline__ void tri_decode(long long t, int& I, int& J) {
    long long i = (long long)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
    while ((i + 1) * (i + 2) / 2 <= t) ++i;
    while (i * (i + 1) / 2 > t) --i;
    I = (int)i;
    J = (int)(t - i * (i + 1) / 2);
}

// ------------------------------------------------------------------------------------------------ a1
// Gershgorin radii of the lower-triangle-symmetrised H: R_i = sum_{j<i} |H_ij| + sum_{j>i} |H_ji|.
// One 64x64 lower-triangle tile per block iteration: element (i,j), i>j, adds |H_ij| to R_i and to R_j.
constexpr int GT = 64;
__global__ void __launch_bounds__(256) k_gershgorin_rows(const float* __restrict__ H, int N, long long ldh,
                                                         double* __restrict__ R, double* __restrict__ diag) {
    __shared__ float colacc[4][GT];
    const int nt = (N + GT - 1) / GT;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    const int tx = threadIdx.x & 63, ty = threadIdx.x >> 6;   // ty 0..3 ; warps 2*ty, 2*ty+1
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        int I, J;
        tri_decode(t, I, J);
        const int j = J * GT + tx;
        float v[16];
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const int i = I * GT + ty + 4 * r;
            float x = 0.f;
            if (i < N && j < i) x = fabsf(__ldg(H + (long long)i * ldh + j));
            if (i < N && j == i) diag[i] = (double)__ldg(H + (long long)i * ldh + j);
            v[r] = x;
        }
        float csum = 0.f;
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            csum += v[r];
            const float rs = warp_sum(v[r]);                  // 32 of the 64 columns of row i
            const int i = I * GT + ty + 4 * r;
            if ((threadIdx.x & 31) == 0 && i < N && rs != 0.f) atomicAdd(R + i, (double)rs);
        }
        colacc[ty][tx] = csum;
        __syncthreads();
        if (ty == 0 && j < N) {
            const float c = colacc[0][tx] + colacc[1][tx] + colacc[2][tx] + colacc[3][tx];
            if (c != 0.f) atomicAdd(R + j, (double)c);
        }
        __syncthreads();
    }
}

// eps_min = min_i (H_ii - R_i), eps_max = max_i (H_ii + R_i) -> ctrl (one block).
__global__ void __launch_bounds__(1024) k_gershgorin_finalize(const double* __restrict__ R,
                                                              const double* __restrict__ diag, int N, Ctrl* ctrl,
                                                              double* bounds_out) {
    __shared__ double smin[32], smax[32];
    double lo = INFINITY, hi = -INFINITY;
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        lo = fmin(lo, diag[i] - R[i]);
        hi = fmax(hi, diag[i] + R[i]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if ((threadIdx.x & 31) == 0) { smin[threadIdx.x >> 5] = lo; smax[threadIdx.x >> 5] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) { lo = fmin(lo, smin[w]); hi = fmax(hi, smax[w]); }
        if (ctrl) { ctrl->eps_min = lo; ctrl->eps_max = hi; ctrl->launches += 2; }
        if (bounds_out) { bounds_out[0] = lo; bounds_out[1] = hi; }
    }
}

// ------------------------------------------------------------------------------------------------ a2
// S_0 = (eps_max I - H) / (eps_max - eps_min)  (W_0, B_0 of Alg. 1), written as FP32 master + FP16 hi/lo
// (Eqs. 12-13), both triangles from H's lower triangle; Tr S_0 and ||S_0||_F^2 in FP64.  32x32 tiles, the
// mirrored tile goes through shared memory so that both global writes are coalesced.
constexpr int AT = 32;
__global__ void __launch_bounds__(256) k_affine_split(const float* __restrict__ H, int N, long long ldh,
                                                      float* __restrict__ S, __half* __restrict__ hi,
                                                      __half* __restrict__ lo, long long ld, long long ldf,
                                                      float scale, Ctrl* ctrl,
                                                      sp2_layer_stat_t* stats, const double* thetas,
                                                      unsigned long long* __restrict__ rowsq) {
    __shared__ float ts[AT][AT + 1];
    __shared__ double colsq[8][AT];
    __shared__ double red[8][2];
    __shared__ int is_last;
    const double e0 = ctrl->eps_min, e1 = ctrl->eps_max;
    if (!(e1 > e0) || !isfinite(e0) || !isfinite(e1)) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            ctrl->error = SP2_ERR_BOUNDS_DEGENERATE;
            ctrl->running = 0;
        }
        return;
    }
    const float w0 = (float)(-1.0 / (e1 - e0));    // W_0
    const float b0 = (float)(e1 / (e1 - e0));      // B_0
    const int nt = (N + AT - 1) / AT;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;    // 8 rows per pass
    double trS = 0.0, fro2 = 0.0;
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        int I, J;
        tri_decode(t, I, J);
        double csq = 0.0;                                    // this thread's column j, rows of this warp
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int li = ty + 8 * r;
            const int i = I * AT + li, j = J * AT + tx;
            float s = 0.f;
            double rsq = 0.0;
            if (i < N && j <= i) {
                s = w0 * __ldg(H + (long long)i * ldh + j);
                if (i == j) s += b0;
                S[(long long)i * ld + j] = s;
                __half h, l;
                split_hi_lo(s, scale, h, l);
                hi[(long long)i * ldf + j] = h;
                lo[(long long)i * ldf + j] = l;
                const double sd = (double)s;
                rsq = sd * sd;
                if (i == j) { trS += sd; fro2 += sd * sd; }
                else { fro2 += 2.0 * sd * sd; csq += rsq; }
            }
            ts[li][tx] = s;
            if (rowsq) {                                     // row i: sum over this warp's 32 columns (j <= i)
                rsq = warp_sum(rsq);
                if (tx == 0 && i < N) atomicAdd(rowsq + i, rowsq_fix(rsq));
            }
        }
        colsq[ty][tx] = csq;
        __syncthreads();
        if (rowsq && ty == 0) {                              // column j (= row j of the mirrored part), j < i only
            double c = 0.0;
#pragma unroll
            for (int w8 = 0; w8 < 8; ++w8) c += colsq[w8][tx];
            const int j = J * AT + tx;
            if (j < N && c != 0.0) atomicAdd(rowsq + j, rowsq_fix(c));
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int lj = ty + 8 * r;                      // row of the mirrored tile = column of the source
            const int jj = J * AT + lj, ii = I * AT + tx;   // write S[jj][ii] = s(ii, jj) for ii > jj
            if (ii < N && jj < ii) {
                const float s = ts[tx][lj];
                S[(long long)jj * ld + ii] = s;
                __half h, l;
                split_hi_lo(s, scale, h, l);
                hi[(long long)jj * ldf + ii] = h;
                lo[(long long)jj * ldf + ii] = l;
            }
        }
        __syncthreads();
    }
    trS = warp_sum(trS);
    fro2 = warp_sum(fro2);
    if (tx == 0) { red[ty][0] = trS; red[ty][1] = fro2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < 8; ++w) { a += red[w][0]; b += red[w][1]; }
        ctrl->partial[blockIdx.x][0] = a;
        ctrl->partial[blockIdx.x][1] = b;
        ctrl->partial[blockIdx.x][2] = 0.0;
        __threadfence();
        const unsigned int done = atomicAdd(&ctrl->done_counter, 1u);
        is_last = (done == gridDim.x - 1);
        if (is_last) {
            __threadfence();
            double s0 = 0.0, s1 = 0.0;
            for (unsigned int i = 0; i < gridDim.x; ++i) {
                s0 += ((volatile double*)ctrl->partial[i])[0];
                s1 += ((volatile double*)ctrl->partial[i])[1];
            }
            ctrl->N_S = s0;          // N_S = Tr[S_0]
            ctrl->fro2 = s1;
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

// ------------------------------------------------------------------------------------------------ launchers
cudaError_t launch_gershgorin(const float* H, int N, long long ldh, double* R, double* diag, Ctrl* ctrl,
                              double* bounds_out, int num_sms, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(R, 0, sizeof(double) * (size_t)N, st);
    if (e != cudaSuccess) return e;
    const int nt = (N + GT - 1) / GT;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    const int grid = (int)(ntiles < (long long)num_sms * 16 ? ntiles : (long long)num_sms * 16);
    k_gershgorin_rows<<<grid, 256, 0, st>>>(H, N, ldh, R, diag);
    k_gershgorin_finalize<<<1, 1024, 0, st>>>(R, diag, N, ctrl, bounds_out);
    return cudaGetLastError();
}

cudaError_t launch_affine_split(const float* H, int N, long long ldh, float* S, __half* hi, __half* lo, long long ld,
                                long long ldf, float scale, Ctrl* ctrl, sp2_layer_stat_t* stats, const double* thetas,
                                unsigned long long* rowsq, int num_sms, cudaStream_t st) {
    const int nt = (N + AT - 1) / AT;
    const long long ntiles = (long long)nt * (nt + 1) / 2;
    long long cap = (long long)num_sms * 6;
    if (cap > kMaxPartials) cap = kMaxPartials;
    const int grid = (int)(ntiles < cap ? ntiles : cap);
    k_affine_split<<<grid, 256, 0, st>>>(H, N, ldh, S, hi, lo, ld, ldf, scale, ctrl, stats, thetas, rowsq);
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
