// Batched small-N path (row a10 of DESIGN.md; paper: "batching ... would most likely benefit the SP2 method for
// small N"): the WHOLE solve of one matrix (bounds, initial layer, every SP2 layer, control, output) in one
// CTA (N <= 128) or one 2-CTA cluster (N <= 256); a launch covers the whole batch, clusters loop over matrices.
//
// Residency: each CTA owns 128 rows.  Its FP16 hi/lo row panels live in shared memory in the UMMA K-major
// 128B-swizzled layout and are at the same time the A operand (its M rows) and its half of the B operand of a
// cta_group::2 MMA (M = 256, N = 256), so no operand ever moves.  The FP32 master S lives in the upper half of
// TMEM (columns NP..2NP-1, lane = row), the accumulator in the lower half.  Only the lower triangle (j <= i) is
// finalised; each value is written to (i,j) and mirrored to (j,i) in the panels (through distributed shared
// memory when row j belongs to the peer CTA), which keeps S exactly symmetric (an antisymmetric rounding
// residue would be amplified by the 2S - S^2 branch).
#include "sp2_kernels.h"
#include "sp2_ptx.cuh"

namespace sp2 {

template <int NP_, int CG_>
struct ResCfg {
    static constexpr int NP = NP_, CG = CG_;
    static constexpr int KBLK = NP / 64;
    static constexpr int PANEL_BYTES = KBLK * 16384;      // 128 rows x NP fp16
    static constexpr int TMEM_COLS = 2 * NP;
    // warps 0-7: rows / epilogue (warp w owns TMEM lanes 32 (w % 4) .. +31 and every second 32-column chunk of them:
    // two warps per scheduler hide each other's latencies and halve the longest chunk list), warp 8: MMA + TMEM alloc
    static constexpr int THREADS = 288;
    static constexpr int MMA_WARP = 8;
    static constexpr int STAGE_FLOATS = 8 * 32 * 33;
};

struct ResShared {
    uint64_t mma_bar;
    uint32_t tmem_slot;
    uint32_t pad0;
    double part[2][8][4];        // [iteration parity][warp][trS, fro2, trX, -]
    float rrow[2][128];          // Gershgorin: per chunk-half row sums of the strictly-lower entries
    float dii[128];              // Gershgorin: diagonal entries
    float rcol[4][256];          // Gershgorin: per-warp column sums of the strictly-lower triangle (this CTA's rows)
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

// Which 32-column chunks does the warp owning rows [row0, row0 + 31] finalise?  Every unordered pair {i, j} exactly
// once.  Plain rule: the lower triangle (c0 <= row0).  With two CTAs that leaves CTA 1 (rows 128-255) 26 chunk tasks
// and CTA 0 ten, so the block rows 192-255 x columns 0-127 is handed to CTA 0, which finalises it from its own
// accumulator's transposed copy (rows 0-127, columns 192-255: the MMA computes the full square): 18 tasks each,
// at most 3 per warp instead of 4.  Returns -1 not handled, 0 all 32 x 32 entries (off-diagonal), 1 diagonal chunk.
template <int CG>
__device__ __forceinline__ int chunk_kind(int row0, int c0) {
    if (CG == 2) {
        if (row0 < 128 && c0 >= 192) return 0;
        if (row0 >= 192 && c0 < 128) return -1;
    }
    if (c0 > row0) return -1;
    return c0 == row0 ? 1 : 0;
}

template <int CG>
__device__ __forceinline__ void group_sync() {
    if (CG == 2) cluster_sync_all(); else __syncthreads();
}

// Load the 32 x 32 block H[row0 + r][c0 + l] (lower-triangle entries only, zero elsewhere / outside N) coalesced,
// transpose it through `stg` so that lane `l` ends up with its own row's 32 values.
__device__ __forceinline__ void load_block_rows(const float* __restrict__ Hm, int N, int row0, int c0, float* stg,
                                                int lane, float (&vals)[32]) {
    __syncwarp();
#pragma unroll 8
    for (int r = 0; r < 32; ++r) {
        const int i = row0 + r, j = c0 + lane;
        float v = 0.f;
        if (i < N && j <= i) v = __ldg(Hm + (size_t)i * N + j);
        stg[r * 33 + lane] = v;
    }
    __syncwarp();
#pragma unroll
    for (int c = 0; c < 32; ++c) vals[c] = stg[lane * 33 + c];
}

template <class C>
__global__ void __launch_bounds__(C::THREADS, 1) k_sp2_resident(const ResidentParams p) {
    constexpr int NP = C::NP, CG = C::CG;
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
    uint32_t mma_phase = 0;

    const int q = warp & 3;
    const int hf = (warp >> 2) & 1;               // which half of the 32-column chunks this warp takes
    const int tl = q * 32 + lane;                  // row inside this CTA's panel (TMEM lane)
    const int gi = (int)rank * 128 + tl;           // global row
    const int row0 = (int)rank * 128 + q * 32;     // first row of this warp
    float* stg = stage + (warp & 7) * (32 * 33);
    const uint32_t t_acc = tmem_base + ((uint32_t)(q * 32) << 16);
    const uint32_t t_S = t_acc + NP;
    const float cs = p.scale, inv2 = p.inv_scale2;
    // mirror-store address pieces that depend on this thread's column gi only (panel_off(row, gi) split by row bits)
    const uint32_t mir_base = (uint32_t)((gi >> 6) * 16384 + (gi & 7) * 2);
    uint32_t mir_x[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) mir_x[k] = (uint32_t)(k * 128 + (((((gi & 63) >> 3) ^ k)) << 4));

    for (int m = cluster_id; m < p.B; m += n_clusters) {
        const float* __restrict__ Hm = p.H + (size_t)m * N * N;
        float* __restrict__ Dm = p.D + (size_t)m * N * N;
        sp2_layer_stat_t* stats_m = (rank == 0) ? p.stats + (size_t)m * p.max_layers : nullptr;

        // ------------------------------------------------------------------ a1: Gershgorin bounds (Alg. 1)
        double e0 = p.eps_min, e1 = p.eps_max;
        if (p.auto_bounds) {
            for (int i = threadIdx.x; i < 1024; i += blockDim.x) (&sh->rcol[0][0])[i] = 0.f;
            __syncthreads();
            float Rrow = 0.f;
            if (warp < 8) {
                for (int c0 = 0; c0 < NP; c0 += 32) {
                    const int kind = chunk_kind<CG>(row0, c0);
                    if (kind < 0 || ((c0 >> 5) & 1) != hf) continue;
                    __syncwarp();
                    float colp = 0.f;
                    if (c0 > row0) {
                        // transposed block: entry (gi, c0 + c) is read as H(c0 + c, gi) (lower triangle, reading C22);
                        // lane = row already, the column sums go through the staging tile
#pragma unroll 8
                        for (int c = 0; c < 32; ++c) {
                            const int j = c0 + c;
                            float v = 0.f;
                            if (gi < N && j < N) v = fabsf(__ldg(Hm + (size_t)j * N + gi));
                            Rrow += v;
                            stg[lane * 33 + c] = v;
                        }
                        __syncwarp();
#pragma unroll 8
                        for (int r = 0; r < 32; ++r) colp += stg[r * 33 + lane];
                        sh->rcol[q][c0 + lane] = colp;
                        continue;
                    }
                    // column partial sums in the load layout (lane = column), row sums after the transpose
#pragma unroll 8
                    for (int r = 0; r < 32; ++r) {
                        const int i = row0 + r, j = c0 + lane;
                        float v = 0.f;
                        if (i < N && j <= i) v = __ldg(Hm + (size_t)i * N + j);
                        if (j < i) colp += fabsf(v);
                        stg[r * 33 + lane] = v;
                    }
                    __syncwarp();
                    sh->rcol[q][c0 + lane] = colp;      // each (warp, column) slot is written once: deterministic
#pragma unroll
                    for (int c = 0; c < 32; ++c) {
                        const float v = stg[lane * 33 + c];
                        const int j = c0 + c;
                        if (j < gi) Rrow += fabsf(v);
                        if (j == gi) sh->dii[tl] = v;
                    }
                }
                sh->rrow[hf][tl] = Rrow;
            }
            group_sync<CG>();
            float lo = INFINITY, hi = -INFINITY;
            if (warp < 4) {
                float R = sh->rrow[0][tl] + sh->rrow[1][tl];
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
            c->N_occ = (p.mode == MODE_GENERALIZED) ? 0.0 : (p.nocc_is_scalar ? p.N_occ[0] : p.N_occ[m]);
            c->eps_alt = p.eps_alt; c->tol = p.tol; c->eps_min = e0; c->eps_max = e1;
            c->N = N; c->mode = p.mode; c->max_layers = p.max_layers; c->auto_bounds = p.auto_bounds;
            c->n = 0; c->running = 0; c->stop_reason = 0; c->pending_stop = 0; c->sigma_prev = 0; c->sigma_prev2 = 0;
            c->error = bounds_ok ? 0 : SP2_ERR_BOUNDS_DEGENERATE; c->launches = 0;
            c->N_S = 0; c->fro2 = 0; c->iderr_prev = 0; c->iderr_prev2 = 0; c->nx_inflight = 0; c->noise_kappa = p.noise_kappa;
            c->accelerated = p.accelerated; c->acc_h = 1.0; c->acc_l = 0.0;
            c->homo = p.accelerated ? p.homo_lumo[2 * m] : 0.0;
            c->lumo = p.accelerated ? p.homo_lumo[2 * m + 1] : 0.0;
        }
        if (!bounds_ok) {           // uniform over the cluster (same e0, e1 everywhere)
            if (rank == 0 && threadIdx.x == 0) {
                p.status[m] = SP2_ERR_BOUNDS_DEGENERATE; p.n_layers[m] = 0;
                p.bounds[2 * m] = e0; p.bounds[2 * m + 1] = e1;
            }
            group_sync<CG>();
            continue;
        }

        // ------------------------------------------------------------------ a2: S_0, first split, Tr S_0, ||S_0||_F^2
        const float w0 = (float)(-1.0 / (e1 - e0)), b0 = (float)(e1 / (e1 - e0));
        double trS = 0.0, fro2 = 0.0, trX = 0.0;
        float th1s = 0.f, th2 = 0.f, th3 = 0.f;
        int iter = 0;
        bool first = true;
        while (true) {
            if (warp < 8) {
                // ---- finalise the lower-triangle part of this thread's row: chunk by chunk
                for (int c0 = 0; c0 < NP; c0 += 32) {
                    const int kind = chunk_kind<CG>(row0, c0);
                    if (kind < 0 || ((c0 >> 5) & 1) != hf) continue;
                    const bool upper = (c0 > row0);             // transposed block (columns beyond the rows)
                    float sn[32];
                    if (first) {
                        float hv[32];
                        if (upper) {
#pragma unroll 8
                            for (int c = 0; c < 32; ++c)
                                hv[c] = (gi < N && c0 + c < N) ? __ldg(Hm + (size_t)(c0 + c) * N + gi) : 0.f;
                        } else {
                            load_block_rows(Hm, N, row0, c0, stg, lane, hv);
                        }
#pragma unroll
                        for (int c = 0; c < 32; ++c) {
                            const int j = c0 + c;
                            float s = 0.f;
                            if (gi < N && (upper ? j < N : j <= gi)) { s = w0 * hv[c]; if (j == gi) s += b0; }
                            sn[c] = s;
                        }
                    } else {
                        uint32_t va[32], vs[32];
                        tmem_ld_32x32(t_acc + (uint32_t)c0, va);
                        tmem_ld_32x32(t_S + (uint32_t)c0, vs);
                        tmem_ld_wait();
#pragma unroll
                        for (int c = 0; c < 32; ++c) {
                            const int j = c0 + c;
                            const float x = __uint_as_float(va[c]);
                            float val = fmaf(th1s, x, th2 * __uint_as_float(vs[c]));
                            if (j == gi) {
                                if (gi < N) val += th3;
                                trX += (double)(x * inv2);
                            }
                            sn[c] = val;
                        }
                    }
                    uint32_t so[32];
                    uint32_t hp[16], lp[16];
                    // squares of the strictly-lower entries: FP32 over one chunk (4 partial sums), FP64 across chunks;
                    // FP64 per element only on the diagonal (the FP64 pipe is narrow)
                    float q0 = 0.f, q1 = 0.f, q2 = 0.f, q3 = 0.f;
#pragma unroll
                    for (int c = 0; c < 32; ++c) {
                        const int j = c0 + c;
                        so[c] = __float_as_uint(sn[c]);
                        if ((c & 1) == 0) split_hi_lo2(sn[c], sn[c + 1], cs, hp[c >> 1], lp[c >> 1]);
                        const float sq = (upper || j < gi) ? sn[c] * sn[c] : 0.f;
                        if ((c & 3) == 0) q0 += sq; else if ((c & 3) == 1) q1 += sq;
                        else if ((c & 3) == 2) q2 += sq; else q3 += sq;
                        if (j == gi) {
                            const double vd = (double)sn[c];
                            trS += vd; fro2 += vd * vd;
                        }
                    }
                    fro2 += 2.0 * (double)((q0 + q1) + (q2 + q3));
                    tmem_st_32x32(t_S + (uint32_t)c0, so);      // FP32 master (entries j > i are never read)
                    const bool below = (kind == 0);             // every entry of the chunk is off-diagonal and handled here
                    const uint32_t jr = (uint32_t)(c0 >> 7);    // CTA that owns rows c0..c0+31
                    if (below) {
#pragma unroll
                        for (int g = 0; g < 4; ++g) {           // own row: four 16-byte pieces per matrix
                            const uint32_t off = panel_off(tl, c0 + 8 * g);
                            *reinterpret_cast<uint4*>(hiP + off) = make_uint4(hp[4 * g], hp[4 * g + 1], hp[4 * g + 2], hp[4 * g + 3]);
                            *reinterpret_cast<uint4*>(loP + off) = make_uint4(lp[4 * g], lp[4 * g + 1], lp[4 * g + 2], lp[4 * g + 3]);
                        }
                    }
                    // mirror (j, i): row j = c0 + c of CTA jr, column gi.  Byte offset inside the 128-row panel
                    // = mir_base + (c >> 3) * 1024 + mir_x[c & 7]  (see panel_off): one add per element
                    const uint32_t mb = mir_base + (uint32_t)(((c0 & 127) >> 3) * 1024);
                    if (below) {                                // every j < gi: straight-line stores
                        if (CG == 2 && jr != rank) {
                            const uint32_t rh = mapa_u32(hi_addr, jr) + mb, rl = mapa_u32(lo_addr, jr) + mb;
#pragma unroll
                            for (int c = 0; c < 32; ++c) {
                                const uint32_t off = (uint32_t)((c >> 3) * 1024) + mir_x[c & 7];
                                st_cluster_u16(rh + off, (unsigned short)(hp[c >> 1] >> (16 * (c & 1))));
                                st_cluster_u16(rl + off, (unsigned short)(lp[c >> 1] >> (16 * (c & 1))));
                            }
                        } else {
#pragma unroll
                            for (int c = 0; c < 32; ++c) {
                                const uint32_t off = mb + (uint32_t)((c >> 3) * 1024) + mir_x[c & 7];
                                *reinterpret_cast<unsigned short*>(hiP + off) = (unsigned short)(hp[c >> 1] >> (16 * (c & 1)));
                                *reinterpret_cast<unsigned short*>(loP + off) = (unsigned short)(lp[c >> 1] >> (16 * (c & 1)));
                            }
                        }
                    } else {                                    // diagonal chunk (rows and columns of this CTA)
#pragma unroll
                        for (int c = 0; c < 32; ++c) {
                            const int j = c0 + c;
                            const unsigned short hb = (unsigned short)(hp[c >> 1] >> (16 * (c & 1)));
                            const unsigned short lb = (unsigned short)(lp[c >> 1] >> (16 * (c & 1)));
                            if (j <= gi) {                      // own entries one by one
                                const uint32_t off = panel_off(tl, j);
                                *reinterpret_cast<unsigned short*>(hiP + off) = hb;
                                *reinterpret_cast<unsigned short*>(loP + off) = lb;
                            }
                            if (j < gi) {
                                const uint32_t off = mb + (uint32_t)((c >> 3) * 1024) + mir_x[c & 7];
                                *reinterpret_cast<unsigned short*>(hiP + off) = hb;
                                *reinterpret_cast<unsigned short*>(loP + off) = lb;
                            }
                        }
                    }
                }
                tmem_st_wait();
                // ---- publish this warp's partial sums
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    trS += __shfl_xor_sync(0xffffffffu, trS, o);
                    fro2 += __shfl_xor_sync(0xffffffffu, fro2, o);
                    trX += __shfl_xor_sync(0xffffffffu, trX, o);
                }
                if (lane == 0) {
                    sh->part[iter & 1][warp][0] = trS;
                    sh->part[iter & 1][warp][1] = fro2;
                    sh->part[iter & 1][warp][2] = trX;
                }
            }
            // panels (generic-proxy writes, local and remote) -> visible to the tensor core (async proxy)
            asm volatile("fence.proxy.async;\n" ::: "memory");
            tc_fence_before();
            group_sync<CG>();
            tc_fence_after();
            // ---- a8: control (Alg. 1), evaluated redundantly by both CTAs from identical sums
            // Lane l < 8 CG of warp 0 fetches the partial sums of epilogue warp (l & 7) of CTA (l >> 3) (own shared
            // memory or the peer's through DSMEM: all remote loads in flight at once), then a fixed xor-shuffle tree:
            // the same order in both CTAs, so both take identical decisions.
            if (warp == 0) {
                double a = 0.0, b = 0.0, cX = 0.0;
                if (lane < 8 * CG) {
                    const uint32_t r = (uint32_t)lane >> 3;
                    const int w = lane & 7;
                    if (r == rank) {
                        a = sh->part[iter & 1][w][0]; b = sh->part[iter & 1][w][1]; cX = sh->part[iter & 1][w][2];
                    } else {
                        const uint32_t base = mapa_u32(smem_u32(&sh->part[iter & 1][w][0]), r);
                        a = ld_cluster_f64(base); b = ld_cluster_f64(base + 8); cX = ld_cluster_f64(base + 16);
                    }
                }
#pragma unroll
                for (int o = 8; o > 0; o >>= 1) {
                    a += __shfl_xor_sync(0xffffffffu, a, o);
                    b += __shfl_xor_sync(0xffffffffu, b, o);
                    cX += __shfl_xor_sync(0xffffffffu, cX, o);
                }
                if (lane == 0) {
                    CtrlCore* c = &sh->ctrl;
                    if (first) {
                        c->N_S = a; c->fro2 = b;         // N_S = Tr[S_0]
                        control_plan_next(c, stats_m, p.thetas);
                    } else {
                        control_finish_layer(c, stats_m, p.thetas, a, b, cX);
                    }
                }
            }
            __syncthreads();
            first = false;
            ++iter;
            if (!sh->ctrl.running) break;
            th1s = sh->ctrl.theta[0] * inv2; th2 = sh->ctrl.theta[1]; th3 = sh->ctrl.theta[2];
            trS = fro2 = trX = 0.0;
            // ---- a4: X = S^2 (Eq. 15): 3 MMAs per 16 columns of K, operands = the resident panels
            if (warp == C::MMA_WARP && rank == 0 && lane == 0) {
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
            __syncwarp();
            mbar_wait(&sh->mma_bar, mma_phase);
            mma_phase ^= 1u;
            tc_fence_after();
        }

        // ------------------------------------------------------------------ output: D = S_n, both triangles
        if (warp < 8) {
            for (int c0 = 0; c0 < NP; c0 += 32) {
                const int kind = chunk_kind<CG>(row0, c0);
                if (kind < 0 || ((c0 >> 5) & 1) != hf) continue;
                uint32_t vs[32];
                tmem_ld_32x32(t_S + (uint32_t)c0, vs);
                tmem_ld_wait();
#pragma unroll
                for (int c = 0; c < 32; ++c) {
                    const int j = c0 + c;
                    if (gi < N && (c0 > row0 ? j < N : j <= gi)) {
                        const float v = __uint_as_float(vs[c]);
                        Dm[(size_t)j * N + gi] = v;      // mirrored position: coalesced across the warp
                        Dm[(size_t)gi * N + j] = v;
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
    }

    tc_fence_before();
    group_sync<CG>();
    if (warp == C::MMA_WARP) tmem_dealloc<CG>(tmem_base, C::TMEM_COLS);
}

using Res128 = ResCfg<128, 1>;
using Res256 = ResCfg<256, 2>;

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

cudaError_t launch_resident(const ResidentParams& p, int num_sms, cudaStream_t st) {
    if (p.N <= 128) return launch_res<Res128>(p, num_sms, st);
    return launch_res<Res256>(p, num_sms, st);
}

}  // namespace sp2
