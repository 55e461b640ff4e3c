// Measures the issue interval of tcgen05.mma.kind::f16 (K = 16, both operands in shared memory) on B200 for the shapes
// the layer kernels use: the tile choice of the library (sp2_api.cu: choose_tile_config, TileCfg::CAT in
// sp2_square_tiled.cu) rests on the fact that an MMA with N = 128 is NOT issued twice as often as one with N = 256.
// One CTA (or one CTA pair) issues `reps` rounds of a pattern of MMAs from shared-memory tiles, commits, and waits; prints
// "name cycles_per_mma" lines (k_rate) and "name cycles_per_stage" lines for the layer kernel's ring of stages without
// its loads (k_ring).  Built and run by tests/test_probe_hardware.py.  What it showed (B200):
//   * an MMA issued under `if (lane == 0)` costs ~105 cycles whatever its N <= 128 (the compiler wraps it in a loop of
//     R2UR.BROADCASTs); issued by an elect.sync thread in warp-uniform control flow it runs at the pipe rate (N = 128:
//     64 cycles, N = 256: 128);
//   * inside a ring of stages (wait, MMAs, commit) the issuing thread's own instructions between two stages are NOT
//     hidden by the pipe: 3 x N = 128 per K-step, 768 cycles of pipe time per stage, takes 1086 with per-stage elect and
//     full descriptor arithmetic, 1009 with one-add descriptors, 841 with the whole loop in one elected thread.
#include <cstdio>
#include <cuda_runtime.h>
#include "../../paper_2101_06385_b200/csrc/sp2_ptx.cuh"

using namespace sp2;

// pattern: 0 = three N-wide MMAs per K-step into ONE accumulator (the layer kernel's hh, hl, lh)
//          1 = the same, alternating between TWO accumulators
//          2 = one MMA with 2N columns + one with N (TileCfg::CAT)
//          3 = a single descriptor pair over and over (same operands)
//          4 = pattern 0 issued by TWO warps, each into an accumulator of its own (1.5 K-steps each)
//          5 = pattern 2 with a tcgen05.commit after every four K-steps (the layer kernel's per-stage release)
//          6 = pattern 0 with that commit
// ELECT: the issuing thread is chosen by elect.sync inside warp-uniform control flow (the compiler then moves the MMA's
// operands to uniform registers directly) instead of `if (lane == 0)` (a divergent branch: every MMA is wrapped in a
// loop of R2UR.BROADCASTs)
template <int CG, bool ELECT>
__global__ void __launch_bounds__(128, 1) k_rate(long long* out, int N, int pattern, int reps, int fill) {
    extern __shared__ uint8_t raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(raw) + 1023) & ~uintptr_t(1023));
    __shared__ uint64_t bar[2];
    __shared__ uint32_t slot;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = (CG == 2) ? cluster_ctarank() : 0u;
    // operands: zeros, or (fill = 1) pseudo-random finite FP16 values in (-2, 2) -- data-dependent switching power
    for (int i = threadIdx.x; i < 131072 / 4; i += blockDim.x) {
        uint32_t x = (uint32_t)i * 2654435761u + 12345u;
        x ^= x >> 13; x *= 0x5bd1e995u; x ^= x >> 15;
        reinterpret_cast<uint32_t*>(smem)[i] = fill ? (x & 0xbfffbfffu) : 0u;      // exponent < 16: |v| < 2
    }
    if (warp == 0) {
        if (lane == 0) { mbar_init(&bar[0], 1); mbar_init(&bar[1], 1); fence_barrier_init(); }
        __syncwarp();
        tmem_alloc<CG>(&slot, 512);
        tmem_relinquish<CG>();
    }
    fence_proxy_async_smem();
    tc_fence_before();
    if (CG == 2) cluster_sync_all(); else __syncthreads();
    tc_fence_after();
    const uint32_t tm = *((volatile uint32_t*)&slot);
    // stage layout of the layer kernel: A_hi | A_lo | B_hi | B_lo, 16 KB each (128 rows x 64 K, 128-byte swizzle)
    const uint32_t a_hi = smem_u32(smem), a_lo = a_hi + 16384, b_hi = a_hi + 32768, b_lo = a_hi + 49152;
    const uint32_t idN = umma_idesc_f16(128 * CG, N), id2N = umma_idesc_f16(128 * CG, 2 * N > 256 ? 256 : 2 * N);
    long long t0 = 0, t1 = 0;
    if (rank == 0 && (warp == 0 || (pattern == 4 && warp == 1)) && (ELECT ? elect_one() : lane == 0)) {
        t0 = clock64();
        for (int r = 0; r < reps; ++r) {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint64_t dah = umma_desc_sw128(a_hi + k * 32), dal = umma_desc_sw128(a_lo + k * 32);
                const uint64_t dbh = umma_desc_sw128(b_hi + k * 32), dbl = umma_desc_sw128(b_lo + k * 32);
                if (pattern == 0 || pattern == 6) {
                    umma_f16<CG>(tm, dah, dbh, idN, 1u); umma_f16<CG>(tm, dah, dbl, idN, 1u); umma_f16<CG>(tm, dal, dbh, idN, 1u);
                } else if (pattern == 1) {
                    const uint32_t d0 = tm + ((k & 1) ? 256 : 0), d1 = tm + ((k & 1) ? 0 : 256);
                    umma_f16<CG>(d0, dah, dbh, idN, 1u); umma_f16<CG>(d1, dah, dbl, idN, 1u); umma_f16<CG>(d0, dal, dbh, idN, 1u);
                } else if (pattern == 2 || pattern == 5) {
                    umma_f16<CG>(tm, dah, dbh, id2N, 1u); umma_f16<CG>(tm, dal, dbh, idN, 1u);
                } else if (pattern == 3) {
                    const uint64_t da = umma_desc_sw128(a_hi), db = umma_desc_sw128(b_hi);
                    umma_f16<CG>(tm, da, db, idN, 1u); umma_f16<CG>(tm, da, db, idN, 1u); umma_f16<CG>(tm, da, db, idN, 1u);
                } else {
                    const uint32_t d = tm + (warp ? 256 : 0);
                    if (((k & 1) != 0) == (warp != 0)) {
                        umma_f16<CG>(d, dah, dbh, idN, 1u); umma_f16<CG>(d, dah, dbl, idN, 1u); umma_f16<CG>(d, dal, dbh, idN, 1u);
                    }
                }
            }
            if (pattern >= 5) { if (CG == 1) umma_commit(&bar[1]); else umma_commit_pair(&bar[1], 0x1); }
        }
        if (CG == 1) umma_commit(&bar[warp]); else umma_commit_pair(&bar[warp], 0x1);
        mbar_wait(&bar[warp], 0);
        t1 = clock64();
        if (blockIdx.x < CG) out[warp] = t1 - t0;
    }
    __syncwarp();
    tc_fence_before();
    if (CG == 2) cluster_sync_all(); else __syncthreads();
    if (warp == 0) tmem_dealloc<CG>(tm, 512);
}

template <int CG, bool ELECT = false>
static double run(long long* dev, int N, int pattern, int reps, int fill = 0, int grid = 1) {
    cudaFuncSetAttribute(k_rate<CG, ELECT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 132096);
    long long h[2] = {0, 0};
    for (int rep = 0; rep < 2; ++rep) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(CG * grid); cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = 132096;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = CG; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        cudaLaunchKernelEx(&cfg, k_rate<CG, ELECT>, dev, N, pattern, reps, fill);
        cudaMemcpy(h, dev, 16, cudaMemcpyDeviceToHost);
    }
    const int per_round = (pattern == 2 || pattern == 5) ? 8 : 12;
    const long long cyc = (pattern == 4) ? (h[0] > h[1] ? h[0] : h[1]) : h[0];
    return (double)cyc / ((double)reps * per_round);
}

// The layer kernel's pipeline without the loads: warp 0 plays the producer (waits for a stage to be released, marks it
// full), warp 1 issues a stage's MMAs (pattern 2: CAT; else three N = 128 MMAs per K-step) and releases it with a
// tcgen05.commit.  nstages = depth of the ring; prints cycles per stage (four K-steps).
template <bool CAT, bool CHEAP, int LOOPIN = 0>
__global__ void __launch_bounds__(128, 1) k_ring(long long* out, int nstages, int total) {
    extern __shared__ uint8_t raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(raw) + 1023) & ~uintptr_t(1023));
    __shared__ uint64_t full_bar[8], empty_bar[8], done_bar;
    __shared__ uint32_t slot;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < 196608 / 4; i += blockDim.x) reinterpret_cast<uint32_t*>(smem)[i] = 0x3c003c00u;
    if (warp == 0) {
        if (lane == 0) {
            for (int i = 0; i < 8; ++i) { mbar_init(&full_bar[i], 1); mbar_init(&empty_bar[i], 1); }
            mbar_init(&done_bar, 1);
            fence_barrier_init();
        }
        __syncwarp();
        tmem_alloc<1>(&slot, 512);
        tmem_relinquish<1>();
    }
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tm = *((volatile uint32_t*)&slot);
    const long long t0 = clock64();
    if (warp == 0) {
        int s = 0; uint32_t ph = 0;
        for (int t = 0; t < total; ++t) {
            mbar_wait(&empty_bar[s], ph ^ 1u);
            if (elect_one()) mbar_arrive(&full_bar[s]);
            __syncwarp();
            if (++s == nstages) { s = 0; ph ^= 1u; }
        }
    } else if (warp == 1 && LOOPIN) {
        // the whole loop runs in ONE elected thread (no per-stage elect / warp barrier)
        if (elect_one()) {
            int s = 0; uint32_t ph = 0;
            const uint64_t d0 = umma_desc_sw128(smem_u32(smem));
            uint32_t st16 = 0;
            mbar_wait(&full_bar[0], 0);
            tc_fence_after();
            for (int t = 0; t < total; ++t) {
                int s1 = s + 1; uint32_t ph1 = ph;
                if (s1 == nstages) { s1 = 0; ph1 ^= 1u; }
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint64_t dah = d0 + (uint64_t)(st16 + 2 * k), dal = d0 + (uint64_t)(st16 + 1024 + 2 * k);
                    const uint64_t dbh = d0 + (uint64_t)(st16 + 2048 + 2 * k), dbl = d0 + (uint64_t)(st16 + 3072 + 2 * k);
                    if (CAT) {
                        umma_f16<1>(tm, dah, dbh, umma_idesc_f16(128, 256), 1u);
                        umma_f16<1>(tm, dal, dbh, umma_idesc_f16(128, 128), 1u);
                    } else {
                        umma_f16<1>(tm, dah, dbh, umma_idesc_f16(128, 128), 1u);
                        umma_f16<1>(tm, dah, dbl, umma_idesc_f16(128, 128), 1u);
                        umma_f16<1>(tm, dal, dbh, umma_idesc_f16(128, 128), 1u);
                    }
                }
                umma_commit(&empty_bar[s]);
                if (t == total - 1) umma_commit(&done_bar);
                if (t + 1 < total) { mbar_wait(&full_bar[s1], ph1); tc_fence_after(); }
                st16 = (st16 == 8192u) ? 0u : st16 + 4096u;
                s = s1; ph = ph1;
            }
            mbar_wait(&done_bar, 0);
            out[0] = clock64() - t0;
        }
        __syncwarp();
    } else if (warp == 1) {
        int s = 0; uint32_t ph = 0;
        const uint64_t d0 = umma_desc_sw128(smem_u32(smem));
        uint32_t st16 = 0;                                  // (stage offset) >> 4, three 64 KB regions
        for (int t = 0; t < total; ++t) {
            mbar_wait(&full_bar[s], ph);
            tc_fence_after();
            if (elect_one()) {
                const uint32_t a_hi = smem_u32(smem) + (uint32_t)(s % 3) * 65536u, a_lo = a_hi + 16384, b_hi = a_hi + 32768, b_lo = a_hi + 49152;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    uint64_t dah, dal, dbh, dbl;
                    if (CHEAP) {                            // one add per descriptor
                        dah = d0 + (uint64_t)(st16 + 2 * k); dal = d0 + (uint64_t)(st16 + 1024 + 2 * k);
                        dbh = d0 + (uint64_t)(st16 + 2048 + 2 * k); dbl = d0 + (uint64_t)(st16 + 3072 + 2 * k);
                    } else {
                        dah = umma_desc_sw128(a_hi + k * 32); dal = umma_desc_sw128(a_lo + k * 32);
                        dbh = umma_desc_sw128(b_hi + k * 32); dbl = umma_desc_sw128(b_lo + k * 32);
                    }
                    if (CAT) {
                        umma_f16<1>(tm, dah, dbh, umma_idesc_f16(128, 256), 1u);
                        umma_f16<1>(tm, dal, dbh, umma_idesc_f16(128, 128), 1u);
                    } else {
                        umma_f16<1>(tm, dah, dbh, umma_idesc_f16(128, 128), 1u);
                        umma_f16<1>(tm, dah, dbl, umma_idesc_f16(128, 128), 1u);
                        umma_f16<1>(tm, dal, dbh, umma_idesc_f16(128, 128), 1u);
                    }
                }
                umma_commit(&empty_bar[s]);
                if (t == total - 1) umma_commit(&done_bar);
            }
            __syncwarp();
            st16 = (st16 == 8192u) ? 0u : st16 + 4096u;
            if (++s == nstages) { s = 0; ph ^= 1u; }
        }
        mbar_wait(&done_bar, 0);
        if (lane == 0) out[0] = clock64() - t0;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<1>(tm, 512);
}
template <bool CAT, bool CHEAP, int LOOPIN = 0>
static double run_ring(long long* dev, int nstages) {
    cudaFuncSetAttribute(k_ring<CAT, CHEAP, LOOPIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, 197632);
    long long h = 0;
    const int total = 512;
    for (int rep = 0; rep < 2; ++rep) {
        k_ring<CAT, CHEAP, LOOPIN><<<1, 128, 197632>>>(dev, nstages, total);
        cudaError_t e = cudaMemcpy(&h, dev, 8, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { fprintf(stderr, "k_ring: %s\n", cudaGetErrorString(e)); return -1.0; }
    }
    return (double)h / total;
}

int main() {
    long long* dev;
    cudaMalloc(&dev, 16);
    printf("ring_3x128_stages3 %.1f\n", run_ring<false, false>(dev, 3));
    printf("ring_cat_stages3 %.1f\n", run_ring<true, false>(dev, 3));
    printf("ring_3x128_cheap_desc_stages3 %.1f\n", run_ring<false, true>(dev, 3));
    printf("ring_cat_cheap_desc_stages3 %.1f\n", run_ring<true, true>(dev, 3));
    printf("ring_cat_cheap_desc_stages6 %.1f\n", run_ring<true, true>(dev, 6));
    printf("ring_3x128_one_thread_loop %.1f\n", run_ring<false, true, 1>(dev, 3));
    const int reps = 500;
    printf("cg1_n64_one_acc %.1f\n", run<1>(dev, 64, 0, reps));
    printf("cg1_n128_one_acc %.1f\n", run<1>(dev, 128, 0, reps));
    printf("cg1_n256_one_acc %.1f\n", run<1>(dev, 256, 0, reps));
    printf("cg1_n128_two_acc %.1f\n", run<1>(dev, 128, 1, reps));
    printf("cg1_n128_same_operands %.1f\n", run<1>(dev, 128, 3, reps));
    printf("cg1_cat_256_plus_128 %.1f\n", run<1>(dev, 128, 2, reps));
    printf("cg1_n128_two_warps %.1f\n", run<1>(dev, 128, 4, reps));
    printf("cg1_cat_with_stage_commits %.1f\n", run<1>(dev, 128, 5, reps));
    printf("cg1_n128_with_stage_commits %.1f\n", run<1>(dev, 128, 6, reps));
    printf("cg1_n128_one_acc_elect %.1f\n", run<1, true>(dev, 128, 0, reps));
    printf("cg1_n64_one_acc_elect %.1f\n", run<1, true>(dev, 64, 0, reps));
    printf("cg1_cat_elect %.1f\n", run<1, true>(dev, 128, 2, reps));
    printf("cg1_cat_with_stage_commits_elect %.1f\n", run<1, true>(dev, 128, 5, reps));
    printf("cg1_n128_elect_random_data %.1f\n", run<1, true>(dev, 128, 0, reps, 1));
    printf("cg1_cat_elect_random_data %.1f\n", run<1, true>(dev, 128, 2, reps, 1));
    printf("cg1_cat_elect_random_data_148_ctas %.1f\n", run<1, true>(dev, 128, 2, 4 * reps, 1, 148));
    printf("cg1_n256_random_data %.1f\n", run<1, true>(dev, 256, 0, reps, 1));
    printf("cg2_n256_random_data_74_pairs %.1f\n", run<2, true>(dev, 256, 0, 4 * reps, 1, 74));
    printf("cg2_n128_one_acc %.1f\n", run<2>(dev, 128, 0, reps));
    printf("cg2_n256_one_acc %.1f\n", run<2>(dev, 256, 0, reps));
    return cudaDeviceSynchronize() == cudaSuccess ? 0 : 1;
}
