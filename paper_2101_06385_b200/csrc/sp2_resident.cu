// Batched small-N path (row a10 of DESIGN.md; paper: "batching ... would most likely benefit the SP2 method for
// small N"): the WHOLE solve of one matrix (bounds, initial layer, every SP2 layer, control, output) in one
// CTA (N <= 128) or one 2-CTA cluster (N <= 256); a launch covers the whole batch, clusters loop over matrices.
//
// Residency: each CTA owns 128 rows.  Its FP16 hi/lo row panels live in shared memory in the UMMA K-major
// 128B-swizzled layout and are at the same time the A operand (its M rows) and its half of the B operand of a
// cta_group::2 MMA (M = 256, N = 256), so no operand ever moves.  The FP32 master S lives in the upper half of
// TMEM (columns NP..2NP-1, lane = row), the accumulator in the lower half.
//
// Work split of the epilogue.  The matrix is cut into 32 x 32 blocks; the 32 rows of a block row ("row group" g,
// one TMEM lane quarter of one CTA) belong to two warps, each taking 16 of a block's 32 columns.  The MMA computes
// the full square, so an off-diagonal block pair {g, c} can be finalised from either of its two accumulator copies:
// it is given to the row group g with (c - g) mod NG in 1 .. NG/2 - 1 (the pairs at distance NG/2 go to the outer
// groups).  Every group then owns its diagonal block plus NG/2 - 1 or NG/2 off-diagonal ones, so the triangular work
// is even across the warps and the two CTAs.  Each value is written to (i,j) and mirrored to (j,i) in the panels
// (through distributed shared memory when row j belongs to the peer CTA), which keeps S exactly symmetric (an
// antisymmetric rounding residue would be amplified by the 2S - S^2 branch).
//
// Per layer: MMA (one elected thread) -> epilogue (8 warps) -> cluster barrier -> the control step (one thread,
// Alg. 1) runs WHILE the next layer's MMAs are already issued (their operands do not depend on sigma; a layer is
// wasted only when the stop comes from the noise-floor test, which needs the layer's own trace) -> block barrier.
#include "sp2_kernels.h"
#include "sp2_ptx.cuh"

namespace sp2 {

template <int NP_, int CG_, int CW_>
struct ResCfg {
    static constexpr int NP = NP_, CG = CG_;
    static constexpr int CW = CW_;                        // columns of a 32 x 32 block per warp (16 or 8)
    static constexpr int WPG = 32 / CW;                   // warps per row group
    static constexpr int KBLK = NP / 64;
    static constexpr int PANEL_BYTES = KBLK * 16384;      // 128 rows x NP fp16
    static constexpr int TMEM_COLS = 2 * NP;
    static constexpr int NG = NP / 32;                    // row groups = column chunks of 32
    // warps 0 .. 4 WPG - 1: epilogue (warp w owns TMEM lanes 32 (w % 4) .. +31 and columns CW (w / 4) .. + CW - 1 of
    // every block of its row group), the last warp: MMA issue + TMEM alloc
    static constexpr int EPI_WARPS = 4 * WPG;
    static constexpr int THREADS = (EPI_WARPS + 1) * 32;
    static constexpr int MMA_WARP = EPI_WARPS;
    static constexpr int STAGE_FLOATS = EPI_WARPS * 32 * (CW + 1);
};

struct ResShared {
    uint64_t mma_bar;
    uint32_t tmem_slot;
    uint32_t pad0;
    long long part[2][16][4];    // [iteration parity][warp][trS, fro2, trX (2^40 fixed point), non-finite flag]
    float rrow[4][128];          // Gershgorin: per column-part row sums of the off-diagonal entries
    float dii[128];              // Gershgorin: diagonal entries
    float rcol[4][256];          // Gershgorin: column sums of the blocks finalised by row group q of this CTA
    float mm[4][2];              // per-warp min(d - R), max(d + R)
    CtrlCore ctrl;
};

__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t cta) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;\n" : "=r"(r) : "r"(addr), "r"(cta));
    return r;
}
__device__ __forceinline__ void st_cluster_u16(uint32_t addr, unsigned short v) {
    asm volatile("st.shared::cluster.u16 [%0], %1;\n" ::"r"(addr), "h"(v) : "memory");
}
__device__ __forceinline__ void st_shared_u16(uint32_t addr, unsigned short v) {
    asm volatile("st.shared.u16 [%0], %1;\n" ::"r"(addr), "h"(v) : "memory");
}
__device__ __forceinline__ float ld_cluster_f32(uint32_t addr) {
    float v;
    asm volatile("ld.shared::cluster.f32 %0, [%1];\n" : "=f"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ double ld_cluster_f64(uint32_t addr) {
    double v;
    asm volatile("ld.shared::cluster.f64 %0, [%1];\n" : "=d"(v) : "r"(addr) : "memory");
    return v;
}
// byte offset of element (row t, column j) inside a 128-row K-major panel with 128-byte swizzle
__device__ __forceinline__ uint32_t panel_off(int t, int j) {
    return (uint32_t)((j >> 6) * 16384 + (t >> 3) * 1024 + (t & 7) * 128 + ((((j & 63) >> 3) ^ (t & 7)) << 4) +
                      (j & 7) * 2);
}

// Does row group g finalise the block in column chunk c?  Every unordered pair {g, c} exactly once (see the header).
template <int NG>
__device__ __forceinline__ bool owns_block(int g, int c) {
    const int d = (c - g) & (NG - 1);
    if (d < NG / 2) return true;                          // the diagonal block and the next NG/2 - 1 chunks
    if (d > NG / 2) return false;
    return NG == 8 ? (g < 2 || g >= 6) : (g == 0 || g == NG - 1);
}

// The trace sums are 2^40 fixed-point integers and the control step is integer-only (sp2_control.cuh): with FP64
// shuffle reductions and an FP64 control step a pass spent more time waking the FP64 datapath than on its MMAs.
__device__ __forceinline__ long long to_fix(float x) { return fx_from_float(x); }
__device__ __forceinline__ long long sq_fix(float x) { return fx_square(x); }
__device__ __forceinline__ long long ld_cluster_s64(uint32_t addr) {
    long long v;
    asm volatile("ld.shared::cluster.s64 %0, [%1];\n" : "=l"(v) : "r"(addr) : "memory");
    return v;
}

// Stores with a compile-time byte offset folded into the instruction (REMOTE: the address is a shared::cluster one).
template <bool REMOTE, int IMM>
__device__ __forceinline__ void st_u16_imm(uint32_t addr, uint32_t v) {
    if (REMOTE) asm volatile("st.shared::cluster.u16 [%0+%2], %1;\n" ::"r"(addr), "h"((unsigned short)v), "n"(IMM) : "memory");
    else asm volatile("st.shared.u16 [%0+%2], %1;\n" ::"r"(addr), "h"((unsigned short)v), "n"(IMM) : "memory");
}
__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};\n" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
// hi/lo split of two already-scaled values (the master is kept as c S, see the layer loop): Eqs. 12-13
__device__ __forceinline__ void split_scaled2(float a0, float a1, uint32_t& hi2, uint32_t& lo2) {
    const __half2 h = __floats2half2_rn(a0, a1);
    const float2 hf = __half22float2(h);
    const __half2 l = __floats2half2_rn(a0 - hf.x, a1 - hf.y);
    hi2 = *reinterpret_cast<const uint32_t*>(&h);
    lo2 = *reinterpret_cast<const uint32_t*>(&l);
}
template <int CW> __device__ __forceinline__ void tmem_ld_cw(uint32_t taddr, uint32_t (&v)[CW]);
template <> __device__ __forceinline__ void tmem_ld_cw<16>(uint32_t taddr, uint32_t (&v)[16]) { tmem_ld_32x32_x16(taddr, v); }
template <> __device__ __forceinline__ void tmem_ld_cw<8>(uint32_t taddr, uint32_t (&v)[8]) { tmem_ld_32x32_x8(taddr, v); }
template <int CW> __device__ __forceinline__ void tmem_st_cw(uint32_t taddr, const uint32_t (&v)[CW]);
template <> __device__ __forceinline__ void tmem_st_cw<16>(uint32_t taddr, const uint32_t (&v)[16]) { tmem_st_32x32_x16(taddr, v); }
template <> __device__ __forceinline__ void tmem_st_cw<8>(uint32_t taddr, const uint32_t (&v)[8]) { tmem_st_32x32_x8(taddr, v); }

// Mirror stores of a CW-column part of a block: element e goes to panel row (j0 + e), column gi.  bh / bl = the hi /
// lo panel address of row (j0 + (e & 7)) at column gi; rows 8 further down are 1024 bytes on.  PRED: only e < lim.
#ifndef SP2_RES_EXP
#define SP2_RES_EXP 0        // timing experiments only (results are wrong when non-zero): 1 no remote mirror, 2 no mirror
#endif                       // at all, 4 no master traffic, 8 no own-row stores
template <int E, bool REMOTE, bool PRED, int CW>
__device__ __forceinline__ void mirror_cw(const uint32_t (&bh)[8], const uint32_t (&bl)[8], const uint32_t (&hp)[CW / 2],
                                          const uint32_t (&lp)[CW / 2], int lim) {
    if ((SP2_RES_EXP & 2) || ((SP2_RES_EXP & 1) && REMOTE)) return;
    if constexpr (E < CW) {
        constexpr int IMM = (E >> 3) * 1024;
        const uint32_t h = (E & 1) ? (hp[E >> 1] >> 16) : hp[E >> 1];
        const uint32_t l = (E & 1) ? (lp[E >> 1] >> 16) : lp[E >> 1];
        if (!PRED || E < lim) {
            st_u16_imm<REMOTE, IMM>(bh[E & 7], h);
            st_u16_imm<REMOTE, IMM>(bl[E & 7], l);
        }
        mirror_cw<E + 1, REMOTE, PRED, CW>(bh, bl, hp, lp, lim);
    }
}

template <int CG>
__device__ __forceinline__ void group_sync() {
    if (CG == 2) cluster_sync_all(); else __syncthreads();
}

#ifdef SP2_RES_TIMING
// experiment builds only: cycles per phase, summed over passes, for (CTA 0, warp 1): [0] MMA wait, [1] block loop,
// [2] reduce + publish, [3] cluster barrier, [4] MMA issue + control + block barrier, [5] passes, [6] load H + bounds,
// [7] output + end-of-matrix barrier
__device__ unsigned long long g_res_timing[8];
__device__ unsigned long long g_res_span[3 * 160];      // per CTA: cycles start -> end, globaltimer start, end
#define RT_MARK(i) do { if (rt_on) { const long long t_ = clock64(); rt_acc[i] += t_ - rt_t; rt_t = t_; } } while (0)
#else
#define RT_MARK(i) do { } while (0)
#endif

template <class C>
__global__ void __launch_bounds__(C::THREADS, 1) k_sp2_resident(const ResidentParams p) {
#ifdef SP2_RES_TIMING
    const bool rt_on = (blockIdx.x == 0 && threadIdx.x == 32);
    long long rt_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0}, rt_t = clock64();
    const long long rt_c0 = clock64();
    unsigned long long rt_g0;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(rt_g0));
#endif
    constexpr int NP = C::NP, CG = C::CG, NG = C::NG, CW = C::CW, WPG = C::WPG, EW = C::EPI_WARPS;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* hiP = smem;
    uint8_t* loP = smem + C::PANEL_BYTES;
    float* stage = reinterpret_cast<float*>(smem + 2 * C::PANEL_BYTES);
    ResShared* sh = reinterpret_cast<ResShared*>(smem + 2 * C::PANEL_BYTES + C::STAGE_FLOATS * 4);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = (CG == 2) ? cluster_ctarank() : 0u;
    const int cluster_id = blockIdx.x / CG, n_clusters = gridDim.x / CG;
    const int N = p.N;

    if (warp == C::MMA_WARP) {
        if (lane == 0) {
            mbar_init(&sh->mma_bar, 1);
            fence_barrier_init();
        }
        __syncwarp();
        tmem_alloc<CG>(&sh->tmem_slot, C::TMEM_COLS);
        tmem_relinquish<CG>();
    }
    tc_fence_before();
    group_sync<CG>();
    tc_fence_after();
    const uint32_t tmem_base = *((volatile uint32_t*)&sh->tmem_slot);
    const uint32_t hi_addr = smem_u32(hiP), lo_addr = smem_u32(loP);
    uint32_t mma_uses = 0;                        // MMA batches issued so far (uniform over the cluster)

    const int q = warp & 3;
    const int hf = (warp >> 2) & (WPG - 1);       // which CW of a block's 32 columns this warp takes
    const int tl = q * 32 + lane;                  // row inside this CTA's panel (TMEM lane)
    const int gi = (int)rank * 128 + tl;           // global row
    const int g = (int)rank * 4 + q;               // row group
    float* stg = stage + (warp & (EW - 1)) * (32 * (CW + 1));
    const uint32_t t_acc = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(CW * hf);
    const uint32_t t_S = t_acc + NP;
    const float cs = p.scale, inv2 = p.inv_scale2;
    const float inv_c = 1.0f / cs;                // exact: c is a power of two
    const uint32_t own_row = (uint32_t)((tl >> 3) * 1024 + (tl & 7) * 128);    // panel_off(tl, .) without the column part
    // mirror-store address pieces that depend on this thread's column gi only (panel_off(row, gi) split by row bits)
    const uint32_t mir_base = (uint32_t)((gi >> 6) * 16384 + (gi & 7) * 2);
    uint32_t mir_x[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) mir_x[k] = (uint32_t)(k * 128 + (((((gi & 63) >> 3) ^ k)) << 4));

    for (int m = cluster_id; m < p.B; m += n_clusters) {
        const float* __restrict__ Hm = p.H + (size_t)m * N * N;
        float* __restrict__ Dm = p.D + (size_t)m * N * N;
        sp2_layer_stat_t* stats_m = (rank == 0) ? p.stats + (size_t)m * p.max_layers : nullptr;

        RT_MARK(5);
        // ------------------------------------------------------------------ load H (lower triangle, reading C22) into
        // the master region of TMEM; a1: Gershgorin bounds on the way (Alg. 1)
        if (p.auto_bounds) {
            for (int i = threadIdx.x; i < 1024; i += blockDim.x) (&sh->rcol[0][0])[i] = 0.f;
            __syncthreads();
        }
        if (warp < EW) {
            float Rrow = 0.f;
#pragma unroll 1
            for (int c = 0; c < NG; ++c) {
                if (!owns_block<NG>(g, c)) continue;
                const int j0 = 32 * c + CW * hf;              // first matrix column of this warp's part of the block
                float hv[CW];
                if (c > g) {
                    // block above the diagonal: entry (gi, j) is read as H(j, gi); lane = row already
#pragma unroll
                    for (int e = 0; e < CW; ++e)
                        hv[e] = (gi < N && j0 + e < N) ? __ldg(Hm + (size_t)(j0 + e) * N + gi) : 0.f;
                } else {
                    // coalesced row segments (32 / CW rows of CW per load), transposed through the staging tile
                    __syncwarp();
#pragma unroll 4
                    for (int r2 = 0; r2 < 32; r2 += 32 / CW) {
                        const int r = r2 + lane / CW, i = g * 32 + r, j = j0 + (lane & (CW - 1));
                        float v = 0.f;
                        if (i < N && j <= i) v = __ldg(Hm + (size_t)i * N + j);
                        stg[r * (CW + 1) + (lane & (CW - 1))] = v;
                    }
                    __syncwarp();
#pragma unroll
                    for (int e = 0; e < CW; ++e) hv[e] = stg[lane * (CW + 1) + e];
                }
                uint32_t hu[CW];
#pragma unroll
                for (int e = 0; e < CW; ++e) hu[e] = __float_as_uint(hv[e]);
                tmem_st_cw<CW>(t_S + (uint32_t)(32 * c), hu);
                if (p.auto_bounds) {
                    // |entry| adds to the radius of its row (this thread) and of its column (sum over the 32 rows)
                    __syncwarp();
#pragma unroll
                    for (int e = 0; e < CW; ++e) {
                        const int j = j0 + e;
                        const float a = (c == g && j >= gi) ? 0.f : fabsf(hv[e]);   // diagonal block: j < i only
                        if (c == g && j == gi) sh->dii[tl] = hv[e];
                        Rrow += a;
                        stg[lane * (CW + 1) + e] = a;
                    }
                    __syncwarp();
                    if (lane < CW) {
                        float colp = 0.f;
#pragma unroll 8
                        for (int r = 0; r < 32; ++r) colp += stg[r * (CW + 1) + lane];
                        sh->rcol[q][j0 + lane] = colp;      // each (row group, column) slot is written once
                    }
                }
            }
            tmem_st_wait();
            if (p.auto_bounds) sh->rrow[hf][tl] = Rrow;
        }
        double e0 = p.eps_min, e1 = p.eps_max;
        if (p.auto_bounds) {
            group_sync<CG>();
            float lo = INFINITY, hi = -INFINITY;
            if (warp < 4) {
                float R = 0.f;
                for (int w = 0; w < WPG; ++w) R += sh->rrow[w][tl];
                const float dii = (gi < N) ? sh->dii[tl] : 0.f;
                for (uint32_t r = 0; r < (uint32_t)CG; ++r)
                    for (int w = 0; w < 4; ++w)
                        R += (r == rank) ? sh->rcol[w][gi] : ld_cluster_f32(mapa_u32(smem_u32(&sh->rcol[w][gi]), r));
                if (gi < N) { lo = dii - R; hi = dii + R; }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, o));
                    hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, o));
                }
                if (lane == 0) { sh->mm[q][0] = lo; sh->mm[q][1] = hi; }
            }
            group_sync<CG>();
            lo = INFINITY; hi = -INFINITY;
            for (int w = 0; w < 4; ++w) {
                lo = fminf(lo, sh->mm[w][0]);
                hi = fmaxf(hi, sh->mm[w][1]);
                if (CG == 2) {
                    lo = fminf(lo, ld_cluster_f32(mapa_u32(smem_u32(&sh->mm[w][0]), rank ^ 1u)));
                    hi = fmaxf(hi, ld_cluster_f32(mapa_u32(smem_u32(&sh->mm[w][1]), rank ^ 1u)));
                }
            }
            e0 = (double)lo; e1 = (double)hi;
            group_sync<CG>();       // mm / rcol may be rewritten for the next matrix only after everyone has read
        }
        const bool bounds_ok = (e1 > e0) && isfinite(e0) && isfinite(e1);
        if (threadIdx.x == 0) {
            CtrlCore* c = &sh->ctrl;
            c->N_occ = (p.mode == MODE_GENERALIZED) ? 0 : (p.nocc_is_scalar ? p.N_occ[0] : p.N_occ[m]);
            c->eps_alt = p.eps_alt; c->tol = p.tol; c->eps_min = e0; c->eps_max = e1;
            c->N = N; c->mode = p.mode; c->max_layers = p.max_layers; c->auto_bounds = p.auto_bounds;
            c->n = 0; c->running = 0; c->stop_reason = 0; c->pending_stop = 0; c->sigma_prev = 0; c->sigma_prev2 = 0;
            c->error = bounds_ok ? 0 : SP2_ERR_BOUNDS_DEGENERATE; c->launches = 0;
            c->N_S = 0; c->fro2 = 0; c->iderr_prev = 0; c->iderr_prev2 = 0; c->nx_inflight = 0; c->kappa_q16 = p.kappa_q16;
            c->nonfinite = 0;
            c->accelerated = p.accelerated; c->acc_h = 1.0f; c->acc_l = 0.0f;
            c->homo = p.accelerated ? p.homo_lumo[2 * m] : 0.0;
            c->lumo = p.accelerated ? p.homo_lumo[2 * m + 1] : 0.0;
        }
        if (!bounds_ok) {           // uniform over the cluster (same e0, e1 everywhere)
            if (rank == 0 && threadIdx.x == 0) {
                p.status[m] = (isnan(e0) || isnan(e1)) ? SP2_ERR_NONFINITE : SP2_ERR_BOUNDS_DEGENERATE;
                p.n_layers[m] = 0;
                p.bounds[2 * m] = e0; p.bounds[2 * m + 1] = e1;
            }
            tc_fence_before();
            group_sync<CG>();
            tc_fence_after();
            continue;
        }
        __syncthreads();            // ctrl initialised before anyone reads it
        RT_MARK(6);

        // ------------------------------------------------------------------ the layers.  Pass 0 is a2: S_0 = W_0 H + B_0
        // (Alg. 1) = the generic update with th1 = 0, th2 = W_0, th3 = B_0 applied to the master (= H);
        // pass n >= 1 is S_n = th1 X_n / c^2 + th2 S_{n-1} + th3 I from layer n's accumulator.
        // The master in TMEM holds c S (c = 2^k of the split, reading C10: an exact rescale), so a layer reads
        //   c S_n = (th1 / c) (c^2 X_n) + th2 (c S_{n-1}) + c th3 I
        // and the split needs no multiply.  Traces are taken of S itself (the power-of-two factors come off exactly).
        float th1s = 0.f, th2 = (float)(-1.0 / (e1 - e0)) * cs, th3 = (float)(e1 / (e1 - e0)) * cs;
        bool use_acc = false;
        int iter = 0;
        while (true) {
            // Will the MMAs of the NEXT layer be issued right after this pass's barrier?  Decided from the control state
            // as the previous pass left it (the same for every thread of the cluster): not if this layer's own stop test
            // has already fired, nor when a fixed-depth network ends here.
            const bool issue_next = (sh->ctrl.pending_stop == SP2_STOP_NONE) &&
                                    !(p.mode == MODE_GENERALIZED && iter >= p.max_layers);
            RT_MARK(5);
            if (warp < EW) {
                if (use_acc) {
                    mbar_wait(&sh->mma_bar, (mma_uses - 1u) & 1u);
                    tc_fence_after();
                }
                RT_MARK(0);
                const bool use_S = (th2 != 0.f);
                long long trS = 0, fro2 = 0, trX = 0;       // 2^40 fixed point
                bool bad = false;                           // a non-finite (or absurdly large) value was seen
#pragma unroll 1
                for (int c = 0; c < NG; ++c) {
                    if (!owns_block<NG>(g, c)) continue;
                    const uint32_t tc = (uint32_t)(32 * c);
                    const int j0 = 32 * c + CW * hf;
                    uint32_t va[CW], vs[CW];
                    float sn[CW];
                    if (use_acc) tmem_ld_cw<CW>(t_acc + tc, va);
                    if (use_S && !(SP2_RES_EXP & 4)) tmem_ld_cw<CW>(t_S + tc, vs);
                    tmem_ld_wait();
                    if (use_acc && use_S) {
#pragma unroll
                        for (int e = 0; e < CW; ++e) sn[e] = fmaf(th1s, __uint_as_float(va[e]), th2 * __uint_as_float(vs[e]));
                    } else if (use_acc) {
#pragma unroll
                        for (int e = 0; e < CW; ++e) sn[e] = th1s * __uint_as_float(va[e]);
                    } else {
#pragma unroll
                        for (int e = 0; e < CW; ++e) sn[e] = th2 * __uint_as_float(vs[e]);
                    }
                    uint32_t hp[CW / 2], lp[CW / 2];
                    const uint32_t jr = (uint32_t)(j0 >> 7);                     // CTA that owns rows j0 .. j0 + CW - 1
                    // own row: columns j0 .. j0 + CW - 1 = CW / 8 16-byte pieces per matrix (swizzled chunk index ^ (tl & 7))
                    const uint32_t own0 = (uint32_t)((j0 >> 6) * 16384) + own_row + ((uint32_t)((((j0 & 63) >> 3)) ^ (tl & 7)) << 4);
                    const uint32_t own1 = (uint32_t)((j0 >> 6) * 16384) + own_row + ((uint32_t)((((j0 & 63) >> 3) + 1) ^ (tl & 7)) << 4);
                    // mirror (j, i): row j = j0 + e of CTA jr, column gi.  Byte offset inside the 128-row panel
                    // = mir_base + ((j0 & 127) / 8 + (e >> 3)) * 1024 + mir_x[e & 7]  (see panel_off)
                    const uint32_t mb = mir_base + (uint32_t)(((j0 & 127) >> 3) * 1024);
                    uint32_t bh[8], bl[8];
                    if (c != g) {
                        // ---- off-diagonal block: every entry is finalised here, no per-element predicate
#pragma unroll
                        for (int e = 0; e < CW; e += 2) split_scaled2(sn[e], sn[e + 1], hp[e >> 1], lp[e >> 1]);
                        float q0 = 0.f, q1 = 0.f, q2 = 0.f, q3 = 0.f;
#pragma unroll
                        for (int e = 0; e < CW; e += 4) {
                            q0 = fmaf(sn[e], sn[e], q0); q1 = fmaf(sn[e + 1], sn[e + 1], q1);
                            q2 = fmaf(sn[e + 2], sn[e + 2], q2); q3 = fmaf(sn[e + 3], sn[e + 3], q3);
                        }
                        const float qsum = ((q0 + q1) + (q2 + q3)) * inv2;   // FP32 over CW entries, fixed point across blocks
                        bad = bad || !(qsum <= 1.0e6f);
                        fro2 += 2 * to_fix(qsum);
                        if (!(SP2_RES_EXP & 4)) tmem_st_cw<CW>(t_S + tc, reinterpret_cast<const uint32_t(&)[CW]>(sn));   // FP32 master (c S)
                        if (!(SP2_RES_EXP & 8)) st_shared_v4(hi_addr + own0, hp[0], hp[1], hp[2], hp[3]);
                        if (!(SP2_RES_EXP & 8)) st_shared_v4(lo_addr + own0, lp[0], lp[1], lp[2], lp[3]);
                        if constexpr (CW == 16) {
                            st_shared_v4(hi_addr + own1, hp[CW / 2 - 4], hp[CW / 2 - 3], hp[CW / 2 - 2], hp[CW / 2 - 1]);
                            st_shared_v4(lo_addr + own1, lp[CW / 2 - 4], lp[CW / 2 - 3], lp[CW / 2 - 2], lp[CW / 2 - 1]);
                        }
                        if (CG == 2 && jr != rank) {
                            const uint32_t rh = mapa_u32(hi_addr, jr) + mb, rl = mapa_u32(lo_addr, jr) + mb;
#pragma unroll
                            for (int k = 0; k < 8; ++k) { bh[k] = rh + mir_x[k]; bl[k] = rl + mir_x[k]; }
                            mirror_cw<0, true, false, CW>(bh, bl, hp, lp, CW);
                        } else {
                            const uint32_t rh = hi_addr + mb, rl = lo_addr + mb;
#pragma unroll
                            for (int k = 0; k < 8; ++k) { bh[k] = rh + mir_x[k]; bl[k] = rl + mir_x[k]; }
                            mirror_cw<0, false, false, CW>(bh, bl, hp, lp, CW);
                        }
                    } else {
                        // ---- diagonal block: entries j <= i are authoritative; bias and traces on j == i.
                        // ed = this thread's diagonal column inside the half block (-1: it is in the other half);
                        // lim = number of strictly-lower columns (j < i) in this half
                        const int ed = ((lane / CW) == hf) ? (lane & (CW - 1)) : -1;
                        const int lim = lane - CW * hf;                           // e < lim  <=>  j < gi
                        const float bias = (gi < N) ? th3 : 0.f;
                        float vdiag = 0.f, xdiag = 0.f, qs = 0.f;
#pragma unroll
                        for (int e = 0; e < CW; ++e) {
                            if (e == ed) { sn[e] += bias; vdiag = sn[e]; xdiag = use_acc ? __uint_as_float(va[e]) : 0.f; }
                            if (e < lim) qs = fmaf(sn[e], sn[e], qs);
                        }
                        if (ed >= 0) {
                            const float sd = vdiag * inv_c;                        // the entry of S itself
                            bad = bad || !(fabsf(sd) <= 1.0e3f);
                            trS += to_fix(sd); fro2 += sq_fix(sd);
                            trX += to_fix(xdiag * inv2);
                        }
                        qs *= inv2;
                        bad = bad || !(qs <= 1.0e6f);
                        fro2 += 2 * to_fix(qs);
#pragma unroll
                        for (int e = 0; e < CW; e += 2) split_scaled2(sn[e], sn[e + 1], hp[e >> 1], lp[e >> 1]);
                        tmem_st_cw<CW>(t_S + tc, reinterpret_cast<const uint32_t(&)[CW]>(sn));   // entries j > i are never read back
                        // own row, all 16 columns at once; the entries above the diagonal (j > i) are then overwritten
                        // by the mirror stores of the rows that own them -- after the two warps of this row group have
                        // met, so that every such overwrite comes later
                        if (!(SP2_RES_EXP & 8)) st_shared_v4(hi_addr + own0, hp[0], hp[1], hp[2], hp[3]);
                        if (!(SP2_RES_EXP & 8)) st_shared_v4(lo_addr + own0, lp[0], lp[1], lp[2], lp[3]);
                        if constexpr (CW == 16) {
                            st_shared_v4(hi_addr + own1, hp[CW / 2 - 4], hp[CW / 2 - 3], hp[CW / 2 - 2], hp[CW / 2 - 1]);
                            st_shared_v4(lo_addr + own1, lp[CW / 2 - 4], lp[CW / 2 - 3], lp[CW / 2 - 2], lp[CW / 2 - 1]);
                        }
                        asm volatile("bar.sync %0, %1;\n" ::"r"(2 + q), "n"(32 * WPG) : "memory");
                        const uint32_t rh = hi_addr + mb, rl = lo_addr + mb;
#pragma unroll
                        for (int k = 0; k < 8; ++k) { bh[k] = rh + mir_x[k]; bl[k] = rl + mir_x[k]; }
                        mirror_cw<0, false, true, CW>(bh, bl, hp, lp, lim);
                    }
                }
                tmem_st_wait();
                RT_MARK(1);
                // ---- publish this warp's partial sums
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    trS += __shfl_xor_sync(0xffffffffu, trS, o);
                    fro2 += __shfl_xor_sync(0xffffffffu, fro2, o);
                    trX += __shfl_xor_sync(0xffffffffu, trX, o);
                }
                bad = __any_sync(0xffffffffu, bad);
                if (lane == 0) {
                    sh->part[iter & 1][warp][0] = trS;
                    sh->part[iter & 1][warp][1] = fro2;
                    sh->part[iter & 1][warp][2] = trX;
                    sh->part[iter & 1][warp][3] = bad ? 1 : 0;
                }
            }
            RT_MARK(2);
            // panels (generic-proxy writes, local and remote) -> visible to the tensor core (async proxy)
            asm volatile("fence.proxy.async;\n" ::: "memory");
            tc_fence_before();
            group_sync<CG>();
            tc_fence_after();
            RT_MARK(3);
            // ---- a4 of the NEXT layer, X = S^2 (Eq. 15): 3 MMAs per 16 columns of K, operands = the resident panels;
            // issued before the control step below has decided anything (it runs meanwhile)
            if (issue_next) {
                // one elected thread in warp-uniform control flow (elect_one: no R2UR loops around the MMAs)
                if (warp == C::MMA_WARP && rank == 0 && elect_one()) {
                    constexpr uint32_t idesc = umma_idesc_f16(128 * CG, NP);
#pragma unroll 1
                    for (int kb = 0; kb < C::KBLK; ++kb) {
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const uint64_t dh = umma_desc_sw128(hi_addr + kb * 16384 + k * 32);
                            const uint64_t dl = umma_desc_sw128(lo_addr + kb * 16384 + k * 32);
                            umma_f16<CG>(tmem_base, dh, dh, idesc, (kb | k) != 0);
                            umma_f16<CG>(tmem_base, dh, dl, idesc, 1u);
                            umma_f16<CG>(tmem_base, dl, dh, idesc, 1u);
                        }
                    }
                    if (CG == 1) umma_commit(&sh->mma_bar); else umma_commit_pair(&sh->mma_bar, 0x3);
                }
                ++mma_uses;
            }
            // ---- a8: control (Alg. 1), evaluated redundantly by both CTAs from identical sums
            // Lane l < 8 CG of warp 0 fetches the partial sums of epilogue warp (l & 7) of CTA (l >> 3) (own shared
            // memory or the peer's through DSMEM: all remote loads in flight at once), then a fixed xor-shuffle tree:
            // the same order in both CTAs, so both take identical decisions.
            if (warp == 0) {
                long long a = 0, b = 0, cX = 0, nf = 0;
                if (lane < EW * CG) {
                    const uint32_t r = (uint32_t)lane / EW;
                    const int w = lane & (EW - 1);
                    if (r == rank) {
                        a = sh->part[iter & 1][w][0]; b = sh->part[iter & 1][w][1]; cX = sh->part[iter & 1][w][2];
                        nf = sh->part[iter & 1][w][3];
                    } else {
                        const uint32_t base = mapa_u32(smem_u32(&sh->part[iter & 1][w][0]), r);
                        a = ld_cluster_s64(base); b = ld_cluster_s64(base + 8); cX = ld_cluster_s64(base + 16);
                        nf = ld_cluster_s64(base + 24);
                    }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {          // integer adds: exact, so both CTAs get identical sums
                    a += __shfl_xor_sync(0xffffffffu, a, o);
                    b += __shfl_xor_sync(0xffffffffu, b, o);
                    cX += __shfl_xor_sync(0xffffffffu, cX, o);
                    nf += __shfl_xor_sync(0xffffffffu, nf, o);
                }
                if (lane == 0) {
                    CtrlCore* c = &sh->ctrl;
                    if (iter == 0) {
                        c->N_S = a; c->fro2 = b; c->nonfinite = nf ? 1 : 0;       // N_S = Tr[S_0]
                        control_plan_next(c, stats_m, p.thetas);
                    } else {
                        control_finish_layer(c, stats_m, p.thetas, a, b, cX, nf != 0);
                    }
                }
            }
            __syncthreads();
            RT_MARK(4);
#ifdef SP2_RES_TIMING
            if (rt_on) g_res_timing[7 - 7] += 0;
#endif
            ++iter;
            if (!sh->ctrl.running) {
                if (issue_next) {                        // drain the speculative MMAs before anything is reused
                    mbar_wait(&sh->mma_bar, (mma_uses - 1u) & 1u);
                    tc_fence_after();
                }
                break;
            }
            th1s = sh->ctrl.theta[0] * inv_c; th2 = sh->ctrl.theta[1]; th3 = sh->ctrl.theta[2] * cs;
            use_acc = true;
        }

        // ------------------------------------------------------------------ output: D = S_n, both triangles
        RT_MARK(5);
        if (warp < EW) {
            const bool vec_ok = ((N & 3) == 0) && ((reinterpret_cast<uintptr_t>(Dm) & 15) == 0);
#pragma unroll 1
            for (int c = 0; c < NG; ++c) {
                if (!owns_block<NG>(g, c)) continue;
                const int j0 = 32 * c + CW * hf;
                uint32_t vs[CW];
                tmem_ld_cw<CW>(t_S + (uint32_t)(32 * c), vs);
                tmem_ld_wait();
                float v[CW];
#pragma unroll
                for (int e = 0; e < CW; ++e) v[e] = __uint_as_float(vs[e]) * inv_c;      // the master holds c S
                // mirrored position (j, gi): one row per instruction, coalesced across the warp
#pragma unroll
                for (int e = 0; e < CW; ++e) {
                    const int j = j0 + e;
                    if (gi < N && j < N && (c != g || j < gi)) Dm[(size_t)j * N + gi] = v[e];
                }
                // own position (gi, j): each lane writes a piece of its own row -- as 16-byte vectors where it can
                // (a scalar store per element costs the LSU 32 sectors per instruction for 4 bytes each)
                if (c != g && vec_ok && gi < N && j0 + CW <= N) {
                    float4* dst = reinterpret_cast<float4*>(Dm + (size_t)gi * N + j0);
#pragma unroll
                    for (int e4 = 0; e4 < CW / 4; ++e4) dst[e4] = make_float4(v[4 * e4], v[4 * e4 + 1], v[4 * e4 + 2], v[4 * e4 + 3]);
                } else {
#pragma unroll
                    for (int e = 0; e < CW; ++e) {
                        const int j = j0 + e;
                        if (gi < N && j < N && (c != g || j <= gi)) Dm[(size_t)gi * N + j] = v[e];
                    }
                }
            }
        }
        if (rank == 0 && threadIdx.x == 0) {
            const CtrlCore* c = &sh->ctrl;
            p.n_layers[m] = c->n;
            p.bounds[2 * m] = e0; p.bounds[2 * m + 1] = e1;
            int st = SP2_OK;
            if (c->error < 0) st = c->error;
            else if (c->mode == MODE_STANDARD && c->stop_reason == SP2_STOP_MAX_LAYERS) st = SP2_NOT_CONVERGED;
            p.status[m] = st;
        }
        tc_fence_before();
        group_sync<CG>();          // peer must be done reading this CTA's partial sums / panels before they are reused
        tc_fence_after();
        RT_MARK(7);
    }

#ifdef SP2_RES_TIMING
    if (rt_on) for (int i = 0; i < 8; ++i) g_res_timing[i] = (unsigned long long)rt_acc[i];
    if (threadIdx.x == 0 && blockIdx.x < 160) {
        unsigned long long g1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
        g_res_span[3 * blockIdx.x] = (unsigned long long)(clock64() - rt_c0);
        g_res_span[3 * blockIdx.x + 1] = rt_g0;
        g_res_span[3 * blockIdx.x + 2] = g1;
    }
#endif
    tc_fence_before();
    group_sync<CG>();
    if (warp == C::MMA_WARP) tmem_dealloc<CG>(tmem_base, C::TMEM_COLS);
}

using Res128 = ResCfg<128, 1, 16>;
using Res256 = ResCfg<256, 2, 8>;

template <class C>
static constexpr size_t res_smem() { return 2 * C::PANEL_BYTES + C::STAGE_FLOATS * 4 + sizeof(ResShared) + 1024 + 64; }

size_t resident_smem_bytes(int N) { return N <= 128 ? res_smem<Res128>() : res_smem<Res256>(); }

cudaError_t resident_kernel_setup() {
    cudaError_t e = cudaFuncSetAttribute(k_sp2_resident<Res128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)res_smem<Res128>());
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_sp2_resident<Res256>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)res_smem<Res256>());
}

template <class C>
static cudaError_t launch_res(const ResidentParams& p, int num_sms, cudaStream_t st) {
    int clusters = (C::CG == 2) ? num_sms / 2 : num_sms * 2;    // NP = 128 uses 256 TMEM columns: two CTAs per SM
    if (clusters > p.B) clusters = p.B;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(clusters * C::CG));
    cfg.blockDim = dim3(C::THREADS);
    cfg.dynamicSmemBytes = res_smem<C>();
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C::CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k_sp2_resident<C>, p);
}

#ifdef SP2_RES_TIMING
extern "C" void sp2_debug_resident_timing(unsigned long long out[8]) {
    cudaMemcpyFromSymbol(out, g_res_timing, 8 * sizeof(unsigned long long));
}
extern "C" void sp2_debug_resident_span(unsigned long long out[480]) {
    cudaMemcpyFromSymbol(out, g_res_span, 480 * sizeof(unsigned long long));
}
#endif

cudaError_t launch_resident(const ResidentParams& p, int num_sms, cudaStream_t st) {
    if (p.N <= 128) return launch_res<Res128>(p, num_sms, st);
    return launch_res<Res256>(p, num_sms, st);
}

}  // namespace sp2
