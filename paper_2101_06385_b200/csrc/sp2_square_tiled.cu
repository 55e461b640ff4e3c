// Fused symmetric-square layer of the SP2 network (rows a4-a8 of DESIGN.md) for sm_100a.
//
// One launch = one layer of Alg. 1 with Alg. 2 as the activation:
//   acc(I,J) = sum_k  hi[I,k] hi[J,k] + hi[I,k] lo[J,k] + lo[I,k] hi[J,k]       (Eq. 15; X symmetric so the
//                                                                              transpose term is lo[I,:] . hi[J,:])
//   S_n      = th1 acc / c^2 + th2 S_{n-1} + th3 I                              (Alg. 1's W_n, B_n; Eq. 17)
//   epilogue: Tr S_n, ||S_n||_F^2 (= next layer's N_X), Tr X_n as 2^40 fixed-point integers; next layer's hi/lo
//   (Eqs. 12-13);
//   last CTA: sigma_{n+1}, IdErr_{n+1}, stop tests (control_finish_layer).
// Only lower-triangle tiles (I >= J) are computed; every hi/lo value is also stored at its mirrored position, so the
// operands stay exactly symmetric and the next layer can read full row panels as K-major operands.  Of the FP32
// master only the mirrored (upper-triangle) copy is kept current outside the diagonal chunks: that is the copy the
// epilogue reads back (coalesced), and k_copy_sym mirrors the final result once.
//
// Structure: persistent CTAs (or CTA pairs), static round-robin over a host-ordered supertile list;
// warp 0 = TMA producer, warp 1 = tcgen05.mma issuer (+ TMEM alloc), both issuing through elect.sync; warps 2.. =
// epilogue (TMEM -> registers -> global; two warps per TMEM lane quarter in the plain instantiations).  Two TMEM
// accumulator buffers overlap the epilogue with the next tile's MMAs and let the two rounds of an epoch walk K
// together (K-interleave, ki_range below).
#include "sp2_kernels.h"
#include "sp2_ptx.cuh"

namespace sp2 {

template <int BN_, int CG_, bool ENH_ = false, bool MIX_ = false, bool SP_ = false, int EW_ = 8>
struct TileCfg {
    // SP: blocked-sparse variant for matrices with decay (reading C28): 128 x 128 blocks of S_{n-1}
    // whose Frobenius norm is <= tau count as zero -- their K-blocks are neither loaded nor multiplied.
    static constexpr bool SP = SP_;
    // MIX: the epilogue also accumulates the output mix M += c_n S_n (Eq. 18) in one more FP32 matrix.
    static constexpr bool MIX = MIX_;
    // ENH: enhanced accumulation ("single precision with double accumulation") for the refinement layers:
    // the tensor core accumulates only p.enh_kc K-blocks at a time; the chunk sums are added into a running FP32 pair
    // (two-sum) kept in two more TMEM regions, so the truncating FP32 accumulation never runs over the whole K.
    static constexpr bool ENH = ENH_;
    static constexpr int BN = BN_;                 // accumulator columns = supertile edge
    static constexpr int CG = CG_;                 // CTAs cooperating on one MMA (cta_group)
    static constexpr int BM = 128;                 // accumulator rows per CTA (TMEM lanes)
    static constexpr int BK = 64;                  // K per pipeline stage (one 128-byte swizzle row of FP16)
    static constexpr int BNL = BN / CG;            // B-operand rows this CTA loads
    static constexpr int A_BYTES = BM * BK * 2;
    static constexpr int B_BYTES = BNL * BK * 2;
    static constexpr int STAGE_BYTES = 2 * A_BYTES + 2 * B_BYTES;   // hi and lo of both panels
    static constexpr int STAGES = (STAGE_BYTES > 65536) ? 2 : 3;
    static constexpr int SUB = (BN / BM) / CG;     // 128-row work items per supertile per CTA slot
    // CAT (128 x 128 single-CTA tiles): the hi and lo tiles of the B rows lie one behind the other in a stage, so ONE MMA
    // with N = 256 over both gives [X0 X0 | X0 X1] in a 256-column accumulator; a second one with N = 128 adds
    // (X0 X1)^T = X1 X0 to the left half, and the epilogue adds the two halves.  Same tensor-pipe time as three N = 128
    // MMAs (128 + 64 cycles per K = 16), but two instructions instead of three for the issuing thread, whose own time
    // is not hidden at this tile size (tests/cuda/mma_rate.cu: 916 against 1009 cycles per stage of 768), and the chain
    // of truncating adds behind the dominant term of an entry is a third shorter.
    static constexpr bool CAT = (BN_ == 128) && (CG_ == 1) && !ENH_;
    static constexpr int ACC_COLS = CAT ? 2 * BN : BN;       // TMEM columns of one accumulator buffer
    static constexpr int TMEM_COLS = ENH ? 4 * BN : 2 * ACC_COLS;   // two accumulator buffers (+ running hi, lo)
    static_assert(TMEM_COLS <= 512, "TMEM has 512 columns");
    static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*align*/ + 256 /*barriers*/;
    // warp 0 = TMA producer, warp 1 = MMA issuer, then EPI_WARPS epilogue warps: EPI_WARPS / 4 per TMEM lane quarter,
    // taking alternate 32-column chunks of their 32 rows
    static constexpr int EPI_WARPS = EW_;
    static constexpr int THREADS = 64 + 32 * EPI_WARPS;
};

// Entries of the block-norm tables: low 62 bits = squared Frobenius norm in 2^48 fixed point; top 2 bits = for how many
// consecutive layers the block has been WRITTEN as exact zeros (saturating at 3): after two such layers both ping-pong
// operand pairs and the master hold zeros there, and a tile that would again be zero is not touched at all.
constexpr unsigned long long kBnNormMask = (1ull << 62) - 1ull;
// Blocked-sparse variant: which 128-wide K-blocks of tile (I, J) survive the truncation?  Bit kk says that both
// S'_{I,kk} and S'_{J,kk} are kept (diagonal blocks always are).  bn = squared block norms of S_{n-1} in 2^48 fixed
// point, nb x nb, symmetric.  One ballot per 32 blocks (nb <= 128).
__device__ __forceinline__ void sparse_kmask(const unsigned long long* __restrict__ bn, int nb, int I, int J,
                                             unsigned long long tau2, int lane, uint32_t (&m)[4]) {
#pragma unroll
    for (int t = 0; t < 4; ++t) {
        const int kk = 32 * t + lane;
        bool act = false;
        if (kk < nb) {
            const bool a = (kk == I) || (__ldcg(bn + (size_t)I * nb + kk) & kBnNormMask) > tau2;
            const bool b = (kk == J) || (__ldcg(bn + (size_t)J * nb + kk) & kBnNormMask) > tau2;
            act = a && b;
        }
        m[t] = __ballot_sync(0xffffffffu, act);
    }
}
__device__ __forceinline__ bool sparse_bit(const uint32_t (&m)[4], int kk) {
    const uint32_t word = (kk < 32) ? m[0] : (kk < 64) ? m[1] : (kk < 96) ? m[2] : m[3];
    return ((word >> (kk & 31)) & 1u) != 0u;
}

// Grid-wide layer barrier of the persistent mode: wait until `target` layers of the solve have been applied (the CTA
// that runs the control step publishes ctrl->n with release semantics), make the other CTAs' stores visible to this
// thread's generic and async (TMA) accesses, and tell whether another layer follows.  Bounded spin (a grid
// that is not co-resident cannot be launched in this mode -- cooperative launch -- so a time-out is a bug: trap).
__device__ __forceinline__ bool layer_barrier_one(Ctrl* ctrl, int target) {      // per calling thread
    unsigned int spins = 0;
    int gen;
    do {
        asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(gen) : "l"(&ctrl->layer_gen) : "memory");
        if (gen >= target) break;
        __nanosleep(32);
        if (++spins > (1u << 25)) __trap();
    } while (true);
    __threadfence();                                      // also drops this SM's stale L1 lines
    asm volatile("fence.proxy.async;\n" ::: "memory");
    return *((volatile int*)&ctrl->running) != 0;
}
// Whole warp: EVERY lane does the acquire load and both fences itself.  Acquire semantics and proxy fences are
// per-thread; a value passed on by __shfl_sync orders nothing for the receiving lanes, and the lane that issues the next
// layer's TMA loads is whichever one elect.sync picks.  (The 32 polls of one address are one L2 request.)
__device__ __forceinline__ bool layer_barrier(Ctrl* ctrl, int target, int lane) {
    (void)lane;
    int run = layer_barrier_one(ctrl, target) ? 1 : 0;
    run = __shfl_sync(0xffffffffu, run, 0);               // warp-uniform by construction (running is published before
    return run != 0;                                      // layer_gen); the shuffle only keeps the branch convergent
}


// K-interleave of two consecutive rounds (an EPOCH): a CTA (pair) holds two accumulators in TMEM, so it can walk K
// for its tile of round 2e (accumulator 0) and its tile of round 2e+1 (accumulator 1) in alternating chunks of
// K-blocks instead of one tile after the other.  All CTAs do so in lockstep (round sync at every chunk), which makes
// the 2 x n_slots tiles of an epoch share their operand panels through L2: a panel is fetched from HBM once per
// epoch, not once per round.  The chunks at both ends of K are longer (ki_edge K-blocks) than the ones in between
// (ki_mid): the epilogue of the first tile runs under the second tile's last chunk, the epilogue of the second one
// under the next epoch's first chunk.  Per tile the K order is unchanged (monotonic), so results do not depend on
// the chunking.  Chunk c of nchunks covers K-blocks [kb0, kb1).
__device__ __forceinline__ int ki_nchunks(int KB, int edge, int mid) {
    // a short K is not interleaved (one chunk = one tile after the other): the first tile's epilogue would no longer
    // fit under the second tile's last chunk (measured at N = 3072, 128 x 128 tiles: 3 % slower with two chunks of 24)
    if (edge <= 0 || mid <= 0 || KB < 2 * edge) return 1;
    if (KB == 2 * edge) return 2;
    return 2 + (KB - 2 * edge + mid - 1) / mid;
}
__device__ __forceinline__ void ki_range(int c, int nchunks, int KB, int edge, int mid, int& kb0, int& kb1) {
    if (nchunks == 1) { kb0 = 0; kb1 = KB; return; }
    if (nchunks == 2) { kb0 = c == 0 ? 0 : KB / 2; kb1 = c == 0 ? KB / 2 : KB; return; }
    if (c == 0) { kb0 = 0; kb1 = edge; return; }
    if (c == nchunks - 1) { kb0 = KB - edge; kb1 = KB; return; }
    kb0 = edge + (c - 1) * mid;
    kb1 = kb0 + mid;
    if (kb1 > KB - edge) kb1 = KB - edge;
}

#ifdef SP2_LAYER_TIMING
// experiment builds only: per CTA {globaltimer at entry, after setup, first accumulator ready, last epilogue done, exit}
__device__ unsigned long long g_layer_timing[160 * 8];
extern "C" void sp2_debug_layer_timing(unsigned long long* out) { cudaMemcpyFromSymbol(out, g_layer_timing, 160 * 8 * 8); }
#define LT_MARK(i) do { if (blockIdx.x < 160) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); g_layer_timing[blockIdx.x * 8 + (i)] = t_; } } while (0)
#define LT_ADD(i, v) do { if (blockIdx.x < 160) g_layer_timing[blockIdx.x * 8 + (i)] += (unsigned long long)(v); } while (0)
#define LT_CLK() clock64()
#define LT_ZERO(i) do { if (blockIdx.x < 160) g_layer_timing[blockIdx.x * 8 + (i)] = 0ull; } while (0)
#else
#define LT_MARK(i) do { } while (0)
#define LT_ADD(i, v) do { } while (0)
#define LT_CLK() 0ll
#define LT_ZERO(i) do { } while (0)
#endif

template <class C>
__global__ void __launch_bounds__(C::THREADS, 1)
k_sp2_layer(const __grid_constant__ CUtensorMap tm_hi0, const __grid_constant__ CUtensorMap tm_lo0,
            const __grid_constant__ CUtensorMap tm_hi1, const __grid_constant__ CUtensorMap tm_lo1,
            const LayerParams p) {
    constexpr int BN = C::BN, CG = C::CG, BM = C::BM, BK = C::BK, STAGES = C::STAGES;
    Ctrl* ctrl = p.ctrl;
    // Device-side loop control: a layer launched after convergence does nothing (all CTAs agree: the flag only
    // changes at the very end of a layer kernel).
    if (*((volatile int*)&ctrl->running) == 0) {
        if (p.cond_handle != 0 && blockIdx.x == 0 && threadIdx.x == 0) cudaGraphSetConditional(p.cond_handle, 0);
        return;
    }

    if (threadIdx.x == 64) { LT_MARK(0); LT_ZERO(5); LT_ZERO(6); LT_ZERO(7); }
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * C::STAGE_BYTES);
    uint64_t* full_bar = bars;                       // [STAGES]
    uint64_t* empty_bar = bars + STAGES;             // [STAGES]
    uint64_t* tfull_bar = bars + 2 * STAGES;         // [2]
    uint64_t* tempty_bar = bars + 2 * STAGES + 2;    // [2]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * STAGES + 4);
    __shared__ fx_t red[8][4];
    __shared__ unsigned long long red48[2][8];       // SP: per-warp sums of squares of the tile in flight (2^48 fixed point)

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const uint32_t rank = (CG == 2) ? cluster_ctarank() : 0u;
    const int slot = blockIdx.x / CG;
    const int nslots = gridDim.x / CG;
    const int n_work = p.n_items;
    const int KB = p.Np / BK;

    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tm_hi0);
        tma_prefetch_desc(&tm_lo0);
        if (p.persist) { tma_prefetch_desc(&tm_hi1); tma_prefetch_desc(&tm_lo1); }
    }
    // Persistent mode (p.persist): this launch runs layer after layer until the control stops the solve; the CTAs meet
    // at a grid-wide barrier after each layer (released by the CTA that ran the control step).  Layer l of the launch
    // reads the operand pair (l & 1) and writes the other one.  n_at_entry: layers applied before this launch.
    const int n_at_entry = *((volatile int*)&ctrl->n);
    if (warp == 1) {
        if (lane == 0) {
            for (int s = 0; s < STAGES; ++s) {
                mbar_init(&full_bar[s], 1);           // leader's arrive.expect_tx only; the peer's bytes are counted too
                mbar_init(&empty_bar[s], 1);
            }
            for (int b = 0; b < 2; ++b) {
                mbar_init(&tfull_bar[b], 1);
                mbar_init(&tempty_bar[b], C::EPI_WARPS * CG);
            }
            fence_barrier_init();
        }
        __syncwarp();
        tmem_alloc<CG>(tmem_slot, C::TMEM_COLS);
        tmem_relinquish<CG>();
    }
    tc_fence_before();
    if (CG == 2) cluster_sync_all(); else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *((volatile uint32_t*)tmem_slot);
    if (threadIdx.x == 64) LT_MARK(1);

    if (warp == 0 && C::SP) {
        // =============================== TMA producer, blocked-sparse: the whole warp finds the surviving K-blocks of a
        // tile (ballots), one lane loads them
        int s = 0;
        uint32_t ph = 0;
        const uint64_t pol = l2_policy_evict_last();
        const unsigned long long tau2 = ctrl->tau2_fx48;
        for (int layer = 0;; ++layer) {
        const CUtensorMap* tmh = (layer & 1) ? &tm_hi1 : &tm_hi0;
        const CUtensorMap* tml = (layer & 1) ? &tm_lo1 : &tm_lo0;
        const unsigned long long* bn_cur = (layer & 1) ? p.bn_next : p.bn_cur;
        for (int w = slot; w < n_work; w += nslots) {
            const WorkItem wi = p.items[w];
            uint32_t m[4];
            sparse_kmask(bn_cur, p.nb, wi.I, wi.J, tau2, lane, m);
            if (elect_one()) {
                const int m0 = wi.I * BN, n0 = wi.J * BN;
                for (int kk = 0; kk < p.nb; ++kk) {
                    if (!sparse_bit(m, kk)) continue;
#pragma unroll 1
                    for (int half = 0; half < 2; ++half) {
                        mbar_wait(&empty_bar[s], ph ^ 1u);
                        uint8_t* st = smem + s * C::STAGE_BYTES;
                        const int k0 = kk * 128 + half * BK;
                        mbar_arrive_expect_tx(&full_bar[s], C::STAGE_BYTES);
                        tma_load_2d_hint(st, tmh, &full_bar[s], k0, m0, pol);
                        tma_load_2d_hint(st + C::A_BYTES, tml, &full_bar[s], k0, m0, pol);
                        tma_load_2d_hint(st + 2 * C::A_BYTES, tmh, &full_bar[s], k0, n0, pol);
                        tma_load_2d_hint(st + 2 * C::A_BYTES + C::B_BYTES, tml, &full_bar[s], k0, n0, pol);
                        if (++s == STAGES) { s = 0; ph ^= 1u; }
                    }
                }
            }
            __syncwarp();
        }
        if (!p.persist || !layer_barrier(ctrl, n_at_entry + layer + 1, lane)) break;
        }
    } else if (warp == 0) {
        // =============================== TMA producer: the whole warp walks the loops (warp-uniform control flow), one
        // elected lane issues (elect_one: no R2UR loops around the TMA instructions)
        {
            int s = 0;
            uint32_t ph = 0;
            const uint64_t pol = l2_policy_evict_last();     // operand panels: reused by the other CTAs of the wave
            // Round sync: the CTAs of a round share row panels through L2 only while they walk K together.  Nothing
            // else keeps them together (each runs its tiles back to back), so every producer checks in at each sync
            // point (round boundary; with the K-interleave every chunk boundary) and goes on when all have (bounded
            // spin: never a hang, at worst no sync).  The counter is monotonic over a solve (every CTA checks in
            // exactly n_sync times per layer), so the targets of layer n + 1 start at n n_sync gridDim.x and a late
            // check-in of the previous layer can never be lost to a reset.
            const int n_rounds = (n_work + nslots - 1) / nslots;
            const bool kint = !C::ENH && p.ki_edge > 0;
            const int nchunks = kint ? ki_nchunks(KB, p.ki_edge, p.ki_mid) : 1;
            const int n_epochs = (n_rounds + 1) >> 1;
            const unsigned int n_sync = kint ? (unsigned int)(n_epochs * nchunks - 1) : (unsigned int)(n_rounds - 1);
            auto sync_point = [&](unsigned int q, bool wait) {      // q = 1 .. n_sync within the layer
                if (lane == 0) {
                    atomicAdd(&ctrl->round_counter, 1u);
                    if (wait && *((volatile unsigned int*)&ctrl->round_sync_broken) == 0u) {
                        const unsigned int target = q * gridDim.x;
                        unsigned int spins = 0;
                        while (*((volatile unsigned int*)&ctrl->round_counter) < target && ++spins < p.round_spins)
                            __nanosleep(64);
                        // timed out: the grid is not co-resident (shared GPU); the sync is only an optimisation, so
                        // give it up for the rest of this solve instead of paying the timeout at every boundary
                        if (spins >= p.round_spins) ctrl->round_sync_broken = 1u;
                    }
                }
                __syncwarp();
            };
            for (int layer = 0;; ++layer) {
            const CUtensorMap* tmh = (layer & 1) ? &tm_hi1 : &tm_hi0;
            const CUtensorMap* tml = (layer & 1) ? &tm_lo1 : &tm_lo0;
            const unsigned int base = (unsigned int)(n_at_entry + layer) * n_sync;
            auto load_stage = [&](int k0, int m0, int n0) {
                mbar_wait(&empty_bar[s], ph ^ 1u);
                uint8_t* st = smem + s * C::STAGE_BYTES;
                if (!elect_one()) {
                } else if (CG == 1) {
                    mbar_arrive_expect_tx(&full_bar[s], C::STAGE_BYTES);
                    tma_load_2d_hint(st, tmh, &full_bar[s], k0, m0, pol);
                    tma_load_2d_hint(st + C::A_BYTES, tml, &full_bar[s], k0, m0, pol);
#pragma unroll
                    for (int h = 0; h < C::BNL / 128; ++h) {
                        tma_load_2d_hint(st + 2 * C::A_BYTES + h * 16384, tmh, &full_bar[s], k0, n0 + h * 128, pol);
                        tma_load_2d_hint(st + 2 * C::A_BYTES + C::B_BYTES + h * 16384, tml, &full_bar[s], k0,
                                         n0 + h * 128, pol);
                    }
                } else {
                    // both CTAs' loads complete_tx on the leader's barrier; only the leader arrives (a peer
                    // load landing first just leaves the transaction count negative until the expect_tx)
                    if (rank == 0) mbar_arrive_expect_tx(&full_bar[s], 2 * C::STAGE_BYTES);
                    tma_load_2d_pair_hint(st, tmh, &full_bar[s], k0, m0, pol);
                    tma_load_2d_pair_hint(st + C::A_BYTES, tml, &full_bar[s], k0, m0, pol);
#pragma unroll
                    for (int h = 0; h < C::BNL / 128; ++h) {
                        tma_load_2d_pair_hint(st + 2 * C::A_BYTES + h * 16384, tmh, &full_bar[s], k0, n0 + h * 128,
                                              pol);
                        tma_load_2d_pair_hint(st + 2 * C::A_BYTES + C::B_BYTES + h * 16384, tml, &full_bar[s], k0,
                                              n0 + h * 128, pol);
                    }
                }
                __syncwarp();
                if (++s == STAGES) { s = 0; ph ^= 1u; }
            };
            if (kint) {
                for (int e = 0; e < n_epochs; ++e) {
                    int m0[2] = {0, 0}, n0[2] = {0, 0};
                    bool has[2];
#pragma unroll
                    for (int t = 0; t < 2; ++t) {
                        const int w = slot + (2 * e + t) * nslots;
                        has[t] = w < n_work;
                        if (has[t]) {
                            const WorkItem wi = p.items[w];
                            m0[t] = wi.I * BN + (wi.sub * CG + (int)rank) * BM;
                            n0[t] = wi.J * BN + wi.col0 + (int)rank * (wi.ncols / CG);
                        }
                    }
                    // odd epochs walk K backwards: the panels shared with the previous epoch (same band) are still in
                    // L2 for the K-blocks that epoch finished with
                    const bool back = (e & 1) != 0;
                    for (int c = 0; c < nchunks; ++c) {
                        const int q = e * nchunks + c;
                        if (p.round_sync && q > 0) sync_point(base + (unsigned int)q, has[0]);
                        int kb0, kb1;
                        ki_range(back ? nchunks - 1 - c : c, nchunks, KB, p.ki_edge, p.ki_mid, kb0, kb1);
#pragma unroll
                        for (int t = 0; t < 2; ++t) {
                            if (!has[t]) continue;
                            for (int i = 0; i < kb1 - kb0; ++i)
                                load_stage((back ? kb1 - 1 - i : kb0 + i) * BK, m0[t], n0[t]);
                        }
                    }
                }
            } else {
                int round = 0;
                for (int w = slot; ; w += nslots, ++round) {
                    if (p.round_sync && round > 0 && round < n_rounds) sync_point(base + (unsigned int)round, w < n_work);
                    if (w >= n_work) break;
                    const WorkItem wi = p.items[w];
                    const int m0 = wi.I * BN + (wi.sub * CG + (int)rank) * BM;                 // A rows of this CTA
                    // B rows this CTA loads: its share of the item's ncols columns (always a full 128-row box per load:
                    // for a narrow tail item the rows beyond ncols / CG are loaded but not used by the MMA)
                    const int n0 = wi.J * BN + wi.col0 + (int)rank * (wi.ncols / CG);
                    // the K direction alternates per PAIR of rounds, as with the K-interleave (so that switching the
                    // interleave off leaves every tile's summation order, hence every bit of the result, unchanged);
                    // the enhanced-accumulation layers have no interleave and alternate per round
                    const bool back = C::ENH ? ((round & 1) != 0) : (((round >> 1) & 1) != 0);
                    for (int kb = 0; kb < KB; ++kb) load_stage((back ? (KB - 1 - kb) : kb) * BK, m0, n0);
                }
            }
            if (!p.persist || !layer_barrier(ctrl, n_at_entry + layer + 1, lane)) break;
            }
        }
        __syncwarp();     // reconverge before the .aligned cluster barrier of the teardown
    } else if (warp == 1 && C::SP) {
        // =============================== MMA issuer, blocked-sparse: the same K-block list as the producer
        int s = 0;
        uint32_t ph = 0;
        int it = 0;
        const unsigned long long tau2 = ctrl->tau2_fx48;
        constexpr uint32_t idesc = umma_idesc_f16(BM, BN);
        for (int layer = 0;; ++layer) {
        const unsigned long long* bn_cur = (layer & 1) ? p.bn_next : p.bn_cur;
        for (int w = slot; w < n_work; w += nslots, ++it) {
            const WorkItem wi = p.items[w];
            uint32_t m[4];
            sparse_kmask(bn_cur, p.nb, wi.I, wi.J, tau2, lane, m);
            const int buf = it & 1;
            mbar_wait(&tempty_bar[buf], ((uint32_t)(it >> 1) & 1u) ^ 1u);
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + (uint32_t)(buf * C::ACC_COLS);
            bool fresh = true;                                  // the tile's first MMA overwrites the accumulator
            for (int kk = 0; kk < p.nb; ++kk) {
                if (!sparse_bit(m, kk)) continue;
#pragma unroll 1
                for (int half = 0; half < 2; ++half) {
                    mbar_wait(&full_bar[s], ph);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint64_t dst = umma_desc_sw128(smem_u32(smem)) + (uint64_t)((uint32_t)s * (uint32_t)(C::STAGE_BYTES >> 4));
#pragma unroll
                        for (int k = 0; k < BK / 16; ++k) {
                            const uint64_t dah = dst + (uint64_t)(2 * k);
                            const uint64_t dal = dst + (uint64_t)((C::A_BYTES >> 4) + 2 * k);
                            const uint64_t dbh = dst + (uint64_t)(((2 * C::A_BYTES) >> 4) + 2 * k);
                            // [X0 X0 | X0 X1] with one N = 256 MMA over the adjacent hi and lo tiles of the B rows, then
                            // X1 X0 into the left half (TileCfg::CAT)
                            umma_f16<1>(d_tmem, dah, dbh, umma_idesc_f16(BM, 2 * BN), (fresh && k == 0) ? 0u : 1u);
                            umma_f16<1>(d_tmem, dal, dbh, idesc, 1u);
                        }
                        umma_commit(&empty_bar[s]);
                    }
                    __syncwarp();
                    fresh = false;
                    if (++s == STAGES) { s = 0; ph ^= 1u; }
                }
            }
            if (elect_one()) {
                umma_commit(&tfull_bar[buf]);                   // also when nothing was issued: arrives at once
                atomicAdd(&ctrl->work_active, (unsigned long long)(__popc(m[0]) + __popc(m[1]) + __popc(m[2]) + __popc(m[3])));
                atomicAdd(&ctrl->work_dense, (unsigned long long)p.nb);
            }
            __syncwarp();
        }
        if (!p.persist || !layer_barrier(ctrl, n_at_entry + layer + 1, lane)) break;
        }
    } else if (warp == 1) {
        // =============================== MMA issuer: ONE elected thread of the leader CTA runs the whole loop.  What it
        // executes between the last MMA of a stage and the first of the next one is not hidden by the tensor pipe (the
        // pipe does not queue MMAs far ahead: tests/cuda/mma_rate.cu), so that stretch is kept short: no per-stage
        // elect / warp barrier, and a descriptor is ONE add to a base descriptor (the address field of a 1024-byte
        // aligned stage advances by bytes >> 4 without carries into the other fields).
        if (rank == 0 && elect_one()) {
            int s = 0;
            uint32_t ph = 0;
            int it = 0;                                   // accumulator uses so far (one per item; per chunk if ENH)
            const uint64_t desc0 = umma_desc_sw128(smem_u32(smem));
            // one pipeline stage: wait for the operands, 3 MMAs per K = 16 into d_tmem, release the stage; `first`: the
            // tile's (or ENH chunk's) first stage overwrites the accumulator; `last`: signal the epilogue
            // The wait for the NEXT stage's operands sits in front of the current stage's last K-step (its latency is then
            // covered by that K-step's MMAs instead of lying between two stages); `have`: this stage's wait is done.
            const int my_stages = (slot < n_work ? (n_work - slot + nslots - 1) / nslots : 0) * KB;   // per layer
            int issued = 0;
            bool have = false;
            auto mma_stage = [&](uint32_t d_tmem, uint32_t idesc, bool first, bool last, int buf) {
                if (!have) {
                    mbar_wait(&full_bar[s], ph);
                    tc_fence_after();
                }
                {
                    const uint64_t dst = desc0 + (uint64_t)((uint32_t)s * (uint32_t)(C::STAGE_BYTES >> 4));
#pragma unroll
                    for (int k = 0; k < BK / 16; ++k) {
                        if (k == BK / 16 - 1) {
                            have = (++issued < my_stages);
                            if (have) {
                                const int s1 = (s + 1 == STAGES) ? 0 : s + 1;
                                mbar_wait(&full_bar[s1], (s + 1 == STAGES) ? (ph ^ 1u) : ph);
                                tc_fence_after();
                            }
                        }
                        const uint64_t dah = dst + (uint64_t)(2 * k);
                        const uint64_t dal = dst + (uint64_t)((C::A_BYTES >> 4) + 2 * k);
                        const uint64_t dbh = dst + (uint64_t)(((2 * C::A_BYTES) >> 4) + 2 * k);
                        const uint64_t dbl = dst + (uint64_t)(((2 * C::A_BYTES + C::B_BYTES) >> 4) + 2 * k);
                        if (C::CAT) {
                            // B_hi and B_lo are adjacent 128-row tiles: [X0 X0 | X0 X1] in one N = 256 MMA (whatever the
                            // item's ncols: a strip's unused columns are computed and ignored), then X1 X0 on the left
                            umma_f16<CG>(d_tmem, dah, dbh, umma_idesc_f16(BM, 2 * BN), (!first || k != 0) ? 1u : 0u);
                            umma_f16<CG>(d_tmem, dal, dbh, umma_idesc_f16(BM, BN), 1u);
                            (void)dbl;
                        } else {
                            umma_f16<CG>(d_tmem, dah, dbh, idesc, (!first || k != 0) ? 1u : 0u);      // X0 X0
                            umma_f16<CG>(d_tmem, dah, dbl, idesc, 1u);                                // X0 X1
                            umma_f16<CG>(d_tmem, dal, dbh, idesc, 1u);                                // (X0 X1)^T
                        }
                    }
                    if (CG == 1) umma_commit(&empty_bar[s]); else umma_commit_pair(&empty_bar[s], 0x3);
                    if (last) {
                        if (CG == 1) umma_commit(&tfull_bar[buf]); else umma_commit_pair(&tfull_bar[buf], 0x3);
                    }
                }
                if (++s == STAGES) { s = 0; ph ^= 1u; }
            };
            const bool kint = !C::ENH && p.ki_edge > 0;
            const int n_rounds = (n_work + nslots - 1) / nslots;
            for (int layer = 0;; ++layer) {
            issued = 0;
            have = false;
            if (kint) {
                // K-interleave: the tiles of rounds 2e and 2e + 1 advance through K in alternating chunks (see ki_range);
                // the order of (epoch, chunk, tile, K-block) is the producer's
                const int nchunks = ki_nchunks(KB, p.ki_edge, p.ki_mid);
                const int n_epochs = (n_rounds + 1) >> 1;
                for (int e = 0; e < n_epochs; ++e) {
                    bool has[2];
                    uint32_t idesc[2] = {0u, 0u};
#pragma unroll
                    for (int t = 0; t < 2; ++t) {
                        const int w = slot + (2 * e + t) * nslots;
                        has[t] = w < n_work;
                        if (has[t]) idesc[t] = umma_idesc_f16(BM * CG, p.items[w].ncols);
                    }
                    const bool back = (e & 1) != 0;
                    for (int c = 0; c < nchunks; ++c) {
                        int kb0, kb1;
                        ki_range(back ? nchunks - 1 - c : c, nchunks, KB, p.ki_edge, p.ki_mid, kb0, kb1);
#pragma unroll
                        for (int t = 0; t < 2; ++t) {
                            if (!has[t]) continue;
                            const int itt = it + t;
                            const int buf = itt & 1;
                            if (c == 0) {                               // epilogue has drained this accumulator
                                const long long t0_ = LT_CLK();
                                mbar_wait(&tempty_bar[buf], ((uint32_t)(itt >> 1) & 1u) ^ 1u);
                                LT_ADD(6, LT_CLK() - t0_);
                                tc_fence_after();
                            }
                            const uint32_t d_tmem = tmem_base + (uint32_t)(buf * C::ACC_COLS);
                            for (int i = 0; i < kb1 - kb0; ++i)
                                mma_stage(d_tmem, idesc[t], c == 0 && i == 0, c == nchunks - 1 && i == kb1 - kb0 - 1, buf);
                        }
                    }
                    it += (has[0] ? 1 : 0) + (has[1] ? 1 : 0);
                }
            } else {
                for (int w = slot; w < n_work; w += nslots) {
                    const uint32_t idesc = umma_idesc_f16(BM * CG, p.items[w].ncols);   // N = 256, or 128 / 64 in the tail
                    const int KC = p.enh_kc;                  // K-blocks per accumulation chunk (ENH)
                    const int nch = C::ENH ? (KB + KC - 1) / KC : 1;
                    for (int ch = 0; ch < nch; ++ch, ++it) {
                        const int buf = it & 1;
                        const uint32_t use = (uint32_t)(it >> 1);
                        const int kb0 = C::ENH ? ch * KC : 0;
                        const int kb1 = C::ENH ? (kb0 + KC < KB ? kb0 + KC : KB) : KB;
                        const long long t0_ = LT_CLK();
                        mbar_wait(&tempty_bar[buf], (use & 1u) ^ 1u);   // epilogue has drained this accumulator
                        LT_ADD(6, LT_CLK() - t0_);
                        tc_fence_after();
                        const uint32_t d_tmem = tmem_base + (uint32_t)(buf * C::ACC_COLS);
                        for (int kb = kb0; kb < kb1; ++kb) mma_stage(d_tmem, idesc, kb == kb0, kb == kb1 - 1, buf);
                    }
                }
            }
            if (!p.persist || !layer_barrier_one(ctrl, n_at_entry + layer + 1)) break;
            }
        }
        __syncwarp();     // reconverge before the .aligned barrier / tcgen05.dealloc of the teardown
    } else {
        // =============================== epilogue warps (TMEM lane quarter = warp % 4)
        const int q = warp & 3;
        const int ew = warp - 2;                            // epilogue warp index
        const int part = ew >> 2;                           // which of the alternate chunks of its rows this warp takes
        constexpr int NPART = C::EPI_WARPS / 4;
        const int rl = q * 32 + lane;                       // accumulator row (TMEM lane) of this thread
        int it = 0;                                         // accumulator uses so far (same count as the MMA warp)
        for (int layer = 0;; ++layer) {
        const float th1 = ((volatile float*)ctrl->theta)[0];
        const float th1s = th1 * p.inv_scale2;
        const float th2 = ((volatile float*)ctrl->theta)[1];
        const float th3 = ((volatile float*)ctrl->theta)[2];
        const float cN = ((volatile float*)ctrl->theta)[3];   // weight of S_n in the output mix (MIX only)
        float* __restrict__ M = p.mix;
        const float cs = p.scale;
        const float inv2 = p.inv_scale2;
        const long long ld = p.ld, ldf = p.ldf;
        float* __restrict__ S = p.S;
        // odd layers of a persistent launch go the other way between the two operand pairs
        __half* __restrict__ HO = (layer & 1) ? p.hi_in : p.hi_out;
        __half* __restrict__ LO = (layer & 1) ? p.lo_in : p.lo_out;
        unsigned long long* __restrict__ Rcur = (layer & 1) ? p.rowsq_next : p.rowsq_cur;
        unsigned long long* __restrict__ Rnext = (layer & 1) ? p.rowsq_cur : p.rowsq_next;
        const unsigned long long* __restrict__ bn_cur = (layer & 1) ? p.bn_next : p.bn_cur;
        unsigned long long* __restrict__ bn_next = (layer & 1) ? const_cast<unsigned long long*>(p.bn_cur) : p.bn_next;
        // No FP64 anywhere in the kernel (an isolated FP64 instruction pays ~170 cycles to wake the datapath, see
        // sp2_control.cuh): the traces are 2^40 fixed-point integers.  Off-diagonal squares are summed in FP32 over one
        // 32-element chunk (4 independent partial sums, |error| <= ~2^-22 of a sum of ~1e-3) and converted once per
        // chunk (exact); the diagonal chunk (one per 128 rows of a diagonal supertile) converts per element, squares
        // as exact FP32 pairs.
        fx_t trS = 0, off2 = 0, dg2 = 0, trX = 0;           // ||S_n||_F^2 = 2 off2 + dg2
        bool bad = false;                                   // a non-finite (or out-of-range) value went into a trace
        const int nch = C::ENH ? (KB + p.enh_kc - 1) / p.enh_kc : 1;
        const uint32_t lane_off = (uint32_t)(q * 32) << 16;
        for (int w = slot; w < n_work; w += nslots, ++it) {
            const WorkItem wi = p.items[w];
            const int m0 = wi.I * BN + (wi.sub * CG + (int)rank) * BM;
            const int n0 = wi.J * BN + wi.col0;
            const int ncols = wi.ncols;
            // blocked-sparse: is the accumulator empty (no surviving K-block), and does S_{n-1}'s own block count as zero?
            bool sp_empty = false, sp_zero_in = false;
            int sp_zc = 0;
            const bool sp_offdiag = C::SP && (wi.I != wi.J);
            fx_t tile40 = 0;                                 // the tile's sum of squares, as it goes into N_X if kept
            unsigned long long tile48 = 0;                   // the same in 2^48 fixed point, for the comparison with tau^2
            if (C::SP) {
                uint32_t m[4];
                sparse_kmask(bn_cur, p.nb, wi.I, wi.J, ctrl->tau2_fx48, lane, m);
                sp_empty = ((m[0] | m[1] | m[2] | m[3]) == 0u);
                if (sp_offdiag) {
                    const unsigned long long cur = __ldcg(bn_cur + (size_t)wi.I * p.nb + wi.J);
                    sp_zero_in = !((cur & kBnNormMask) > ctrl->tau2_fx48);
                    sp_zc = (int)(cur >> 62);
                }
            }
            // the output tile is exactly zero (no surviving product, own block counts as zero; the bias touches diagonal
            // tiles only) -- and if the last two layers already wrote zeros here, there is nothing to do
            const bool sp_zero_out = sp_offdiag && sp_empty && sp_zero_in;
            const bool sp_skip = sp_zero_out && sp_zc >= 2;
            const int gi = m0 + rl;
            const int gi_wmin = m0 + q * 32, gi_wmax = gi_wmin + 31;
            fx_t rowacc = 0;                                // sum_j S_n(gi, j)^2 over the own entries (j <= gi) of this tile
            if (C::ENH) {
                // all chunks but the last: fold the chunk sum into the running FP32 pair (two-sum, error-free)
                const uint32_t t_rh = tmem_base + (uint32_t)(2 * BN) + lane_off, t_rl = t_rh + (uint32_t)BN;
                for (int ch = 0; ch < nch - 1; ++ch, ++it) {
                    const int fbuf = it & 1;
                    mbar_wait(&tfull_bar[fbuf], (uint32_t)(it >> 1) & 1u);
                    tc_fence_after();
                    const uint32_t t_acc = tmem_base + (uint32_t)(fbuf * BN) + lane_off;
#pragma unroll 1
                    for (int c0 = 0; c0 < ncols; c0 += 32) {
                        if (n0 + c0 > gi_wmax) break;
                        if (NPART > 1 && ((c0 >> 5) % NPART) != part) continue;
                        uint32_t a[32], rh[32], rlo[32];
                        tmem_ld_32x32(t_acc + (uint32_t)c0, a);
                        if (ch > 0) {
                            tmem_ld_32x32(t_rh + (uint32_t)c0, rh);
                            tmem_ld_32x32(t_rl + (uint32_t)c0, rlo);
                        }
                        tmem_ld_wait();
                        if (ch == 0) {
#pragma unroll
                            for (int c = 0; c < 32; ++c) { rh[c] = a[c]; rlo[c] = 0u; }
                        } else {
#pragma unroll
                            for (int c = 0; c < 32; ++c) {
                                const float x = __uint_as_float(rh[c]), y = __uint_as_float(a[c]);
                                const float sm = x + y;
                                const float bb = sm - x;
                                const float err = (x - (sm - bb)) + (y - bb);
                                rh[c] = __float_as_uint(sm);
                                rlo[c] = __float_as_uint(__uint_as_float(rlo[c]) + err);
                            }
                        }
                        tmem_st_32x32(t_rh + (uint32_t)c0, rh);
                        tmem_st_32x32(t_rl + (uint32_t)c0, rlo);
                    }
                    tmem_st_wait();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) {
                        if (CG == 1) mbar_arrive(&tempty_bar[fbuf]); else mbar_arrive_cluster(&tempty_bar[fbuf], 0);
                    }
                }
            }
            const int buf = it & 1;
            const uint32_t use = (uint32_t)(it >> 1);
            mbar_wait(&tfull_bar[buf], use & 1u);
            tc_fence_after();
            if (threadIdx.x == 64 && w == slot) LT_MARK(2);
            const long long te0_ = LT_CLK();
            const uint32_t taddr = tmem_base + (uint32_t)(buf * C::ACC_COLS) + lane_off;
            unsigned short* HOu = reinterpret_cast<unsigned short*>(HO);
            unsigned short* LOu = reinterpret_cast<unsigned short*>(LO);
#pragma unroll 1
            for (int c0 = 0; c0 < (sp_skip ? 0 : ncols); c0 += 32) {
                const int gj0 = n0 + c0;
                if (gj0 > gi_wmax) break;                   // rest of the row block lies above the diagonal
                if (NPART > 1 && ((c0 >> 5) % NPART) != part) continue;
                uint32_t v[32];
                float so[32];
                if (C::SP && sp_empty) {
#pragma unroll
                    for (int c = 0; c < 32; ++c) v[c] = 0u;
                } else {
                    tmem_ld_32x32(taddr + (uint32_t)c0, v);
                    if (C::CAT) {                           // X0 X1 lies 128 columns to the right of X0 X0 + X1 X0
                        uint32_t v2[32];
                        tmem_ld_32x32(taddr + (uint32_t)(BN + c0), v2);
                        tmem_ld_wait();
#pragma unroll
                        for (int c = 0; c < 32; ++c) v[c] = __float_as_uint(__uint_as_float(v[c]) + __uint_as_float(v2[c]));
                    }
                }
                if (C::ENH && nch > 1) {
                    // last chunk: total = running pair + this chunk, rounded once to FP32
                    uint32_t rh[32], rlo[32];
                    tmem_ld_32x32(tmem_base + (uint32_t)(2 * BN) + lane_off + (uint32_t)c0, rh);
                    tmem_ld_32x32(tmem_base + (uint32_t)(3 * BN) + lane_off + (uint32_t)c0, rlo);
                    tmem_ld_wait();
#pragma unroll
                    for (int c = 0; c < 32; ++c) {
                        const float x = __uint_as_float(rh[c]), y = __uint_as_float(v[c]);
                        const float sm = x + y;
                        const float bb = sm - x;
                        const float err = (x - (sm - bb)) + (y - bb);
                        v[c] = __float_as_uint(sm + (err + __uint_as_float(rlo[c])));
                    }
                }
                const bool below = (gj0 + 31 <= gi_wmin);   // whole 32x32 chunk strictly in the lower triangle
                // S_{n-1}: read at the mirrored position (S is exactly symmetric) -> coalesced across the warp.  In a
                // diagonal chunk only the entries gj <= gi are used; the others (which a neighbouring lane rewrites
                // further down) are not even loaded.
                float mo[C::MIX ? 32 : 1];
                if (C::SP && sp_zero_in) {
#pragma unroll
                    for (int c = 0; c < 32; ++c) so[c] = 0.f;
                } else if (below) {
#pragma unroll
                    for (int c = 0; c < 32; ++c) so[c] = __ldcs(S + (long long)(gj0 + c) * ld + gi);
                    if (C::MIX) {
#pragma unroll
                        for (int c = 0; c < 32; ++c) mo[C::MIX ? c : 0] = __ldcs(M + (long long)(gj0 + c) * ld + gi);
                    }
                } else {
#pragma unroll
                    for (int c = 0; c < 32; ++c) so[c] = (gj0 + c <= gi) ? __ldcs(S + (long long)(gj0 + c) * ld + gi) : 0.f;
                    if (C::MIX) {
#pragma unroll
                        for (int c = 0; c < 32; ++c)
                            mo[C::MIX ? c : 0] = (gj0 + c <= gi) ? __ldcs(M + (long long)(gj0 + c) * ld + gi) : 0.f;
                    }
                }
                if (below) {
                    tmem_ld_wait();
                    float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
                    __half* __restrict__ rowH = HO + (long long)gi * ldf + gj0;
                    __half* __restrict__ rowL = LO + (long long)gi * ldf + gj0;
                    uint32_t hq[4], lq[4];                  // the previous group's pairs (own rows leave as 32-byte stores)
#pragma unroll
                    for (int g = 0; g < 4; ++g) {           // 8 columns at a time: values leave registers early
                        uint32_t hp[4], lp[4];              // FP16 pairs (even column in the low half)
                        float vals[8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) vals[e] = fmaf(th1s, __uint_as_float(v[8 * g + e]), th2 * so[8 * g + e]);
#pragma unroll
                        for (int e = 0; e < 8; e += 2) split_hi_lo2(vals[e], vals[e + 1], cs, hp[e >> 1], lp[e >> 1]);
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            const int c = 8 * g + e;
                            const float val = vals[e];
                            const uint32_t hb = (hp[e >> 1] >> (16 * (e & 1))) & 0xffffu;
                            const uint32_t lb = (lp[e >> 1] >> (16 * (e & 1))) & 0xffffu;
                            const float sq = val * val;
                            so[c] = sq;                     // column sums below: square of the mirrored entry
                            if ((e & 3) == 0) a0 += sq; else if ((e & 3) == 1) a1 += sq;
                            else if ((e & 3) == 2) a2 += sq; else a3 += sq;
                            // mirrored position: one 128-byte (FP32) / 64-byte (FP16) warp store per column
                            __stcs(S + (long long)(gj0 + c) * ld + gi, val);
                            if (C::MIX) {
                                const float mv = fmaf(cN, val, mo[C::MIX ? c : 0]);
                                mo[C::MIX ? c : 0] = mv;
                                __stcs(M + (long long)(gj0 + c) * ld + gi, mv);
                            }
                            // (pairing two columns into one 32-bit store per lane through a lane exchange was tried:
                            // slower, 38.9 -> 44.2 us per layer at N = 2048)
                            const long long o = (long long)(gj0 + c) * ldf + gi;
                            __stcs(HOu + o, (unsigned short)hb);
                            __stcs(LOu + o, (unsigned short)lb);
                        }
                        // own position: 32 contiguous bytes of each FP16 operand per thread per two groups (the FP32 master
                        // is not written here: only its mirrored copy is ever read back; k_copy_sym mirrors the result)
                        if (C::MIX) {
                            float4* rowM = reinterpret_cast<float4*>(M + (long long)gi * ld + gj0);
                            const int b8 = C::MIX ? 8 * g : 0;
                            st_cs_v8(rowM + 2 * g, __float_as_uint(mo[b8]), __float_as_uint(mo[b8 + (C::MIX ? 1 : 0)]),
                                     __float_as_uint(mo[b8 + (C::MIX ? 2 : 0)]), __float_as_uint(mo[b8 + (C::MIX ? 3 : 0)]),
                                     __float_as_uint(mo[b8 + (C::MIX ? 4 : 0)]), __float_as_uint(mo[b8 + (C::MIX ? 5 : 0)]),
                                     __float_as_uint(mo[b8 + (C::MIX ? 6 : 0)]), __float_as_uint(mo[b8 + (C::MIX ? 7 : 0)]));
                        }
                        if (g & 1) {
                            st_cs_v8(reinterpret_cast<uint4*>(rowH) + (g - 1), hq[0], hq[1], hq[2], hq[3], hp[0], hp[1], hp[2], hp[3]);
                            st_cs_v8(reinterpret_cast<uint4*>(rowL) + (g - 1), lq[0], lq[1], lq[2], lq[3], lp[0], lp[1], lp[2], lp[3]);
                        } else {
#pragma unroll
                            for (int e = 0; e < 4; ++e) { hq[e] = hp[e]; lq[e] = lp[e]; }
                        }
                    }
                    const float sdf = (a0 + a1) + (a2 + a3);
                    bad = bad || !(sdf <= 1.0e6f);
                    const fx_t sd = fx_from_float(sdf);
                    if (sp_offdiag) { tile40 += sd; tile48 += (unsigned long long)__float2ll_rn(sdf * 281474976710656.0f); }
                    else off2 += sd;
                    rowacc += sd;
                } else {
                    // diagonal chunk: only gj <= gi is authoritative (exact symmetry inside the tile).  Exact diagonal
                    // of X_n: diag(S_{n-1}^2)_i = sum_j S_{n-1}(i,j)^2, accumulated while S_{n-1} was written
                    float xdiag = 0.f;
                    if (Rcur != nullptr) {
                        xdiag = (float)(long long)__ldcg(Rcur + gi) * kRowSqInvF;   // one rounding, as through FP64; L2 (atomics)
                        Rcur[gi] = 0ull;                    // this buffer is the accumulator of the layer after next
                    }
                    tmem_ld_wait();
                    fx_t sq_own = 0;
                    // Off-diagonal squares (gj < gi) are summed in FP32 and converted once, as in the chunks below the
                    // diagonal; the diagonal element is converted exactly.  Own rows leave as vectors, sixteen columns at
                    // a time (a 4-byte store per lane and row costs the LSU 32 sectors per instruction).  The entries
                    // above the diagonal (gj > gi) written here are this thread's own rounding of a value that belongs to
                    // row gj; after the warp barrier the mirror stores of the rows that own them overwrite them (exact
                    // symmetry inside the tile).
                    float q0 = 0.f, q1 = 0.f, q2 = 0.f, q3 = 0.f;
                    float4* rowS = reinterpret_cast<float4*>(S + (long long)gi * ld + gj0);
                    uint4* rowH = reinterpret_cast<uint4*>(HO + (long long)gi * ldf + gj0);
                    uint4* rowL = reinterpret_cast<uint4*>(LO + (long long)gi * ldf + gj0);
#pragma unroll
                    for (int half = 0; half < 2; ++half) {
                        uint32_t hp[8], lp[8];              // FP16 pairs of sixteen columns (even column in the low half)
#pragma unroll
                        for (int cc = 0; cc < 16; ++cc) {
                            const int c = 16 * half + cc;
                            const int gj = gj0 + c;
                            const float x = __uint_as_float(v[c]);
                            const bool on_diag = (gj == gi);
                            float val = fmaf(th1s, x, th2 * so[c]);
                            if (on_diag) {
                                if (Rcur != nullptr) val = fmaf(th1, xdiag, th2 * so[c]);
                                if (gi < p.N) val += th3;
                                const fx_t v2 = fx_square(val);
                                sq_own += v2;
                                dg2 += v2; trS += fx_from_float(val); trX += fx_from_float(x * inv2);
                            }
                            __half h, l;
                            split_hi_lo(val, cs, h, l);
                            const uint32_t hb = __half_as_ushort(h), lb = __half_as_ushort(l);
                            if (cc & 1) { hp[cc >> 1] |= hb << 16; lp[cc >> 1] |= lb << 16; }
                            else { hp[cc >> 1] = hb; lp[cc >> 1] = lb; }
                            if (gj <= gi) bad = bad || !(fabsf(val) <= 1.0e3f);
                            const float sq = (gj < gi) ? val * val : 0.f;
                            so[c] = sq;
                            if ((cc & 3) == 0) q0 += sq; else if ((cc & 3) == 1) q1 += sq;
                            else if ((cc & 3) == 2) q2 += sq; else q3 += sq;
                            v[c] = __float_as_uint(val);
                            if (C::MIX) mo[C::MIX ? c : 0] = fmaf(cN, val, mo[C::MIX ? c : 0]);
                        }
                        st_cs_v8(rowS + 4 * half, v[16 * half], v[16 * half + 1], v[16 * half + 2], v[16 * half + 3],
                                 v[16 * half + 4], v[16 * half + 5], v[16 * half + 6], v[16 * half + 7]);
                        st_cs_v8(rowS + 4 * half + 2, v[16 * half + 8], v[16 * half + 9], v[16 * half + 10], v[16 * half + 11],
                                 v[16 * half + 12], v[16 * half + 13], v[16 * half + 14], v[16 * half + 15]);
                        st_cs_v8(rowH + 2 * half, hp[0], hp[1], hp[2], hp[3], hp[4], hp[5], hp[6], hp[7]);
                        st_cs_v8(rowL + 2 * half, lp[0], lp[1], lp[2], lp[3], lp[4], lp[5], lp[6], lp[7]);
                    }
                    if (C::MIX) {
                        float4* rowM = reinterpret_cast<float4*>(M + (long long)gi * ld + gj0);
#pragma unroll
                        for (int g = 0; g < 8; ++g)
                            rowM[g] = make_float4(mo[C::MIX ? 4 * g : 0], mo[C::MIX ? 4 * g + 1 : 0],
                                                  mo[C::MIX ? 4 * g + 2 : 0], mo[C::MIX ? 4 * g + 3 : 0]);
                    }
                    {
                        const float sdf = (q0 + q1) + (q2 + q3);
                        bad = bad || !(sdf <= 1.0e6f);
                        const fx_t sd = fx_from_float(sdf);
                        off2 += sd;
                        sq_own += sd;
                    }
                    __syncwarp();
#pragma unroll
                    for (int c = 0; c < 32; ++c) {
                        const int gj = gj0 + c;
                        if (gj < gi) {                      // mirrored position: coalesced across the warp
                            const float val = __uint_as_float(v[c]);
                            __half h, l;
                            split_hi_lo(val, cs, h, l);     // the same bits as in the own row
                            const long long o = (long long)gj * ldf + gi;
                            S[(long long)gj * ld + gi] = val;
                            HOu[o] = __half_as_ushort(h);
                            LOu[o] = __half_as_ushort(l);
                            if (C::MIX) M[(long long)gj * ld + gi] = mo[C::MIX ? c : 0];
                        }
                    }
                    rowacc += sq_own;
                }
                if (Rnext != nullptr) {
                    // sum over the warp's 32 rows of so[c] for every column c: butterfly transpose-reduce, lane c
                    // ends with column c's sum (31 shuffles), then one fixed-point atomic per column.
#pragma unroll
                    for (int sft = 16; sft >= 1; sft >>= 1) {
                        const bool up = (lane & sft) != 0;
#pragma unroll
                        for (int i = 0; i < sft; ++i) {
                            const float send = up ? so[i] : so[i + sft];
                            const float keep = up ? so[i + sft] : so[i];
                            so[i] = keep + __shfl_xor_sync(0xffffffffu, send, sft);
                        }
                    }
                    if (so[0] != 0.f) atomicAdd(Rnext + gj0 + lane, rowsq_fix(so[0]));
                }
            }
            if (Rnext != nullptr && rowacc != 0) atomicAdd(Rnext + gi, (unsigned long long)(rowacc << (kRowSqBits - kFxBits)));
            // all tcgen05.ld of this accumulator have completed (tmem_ld_wait above): hand it back to the MMA warp
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                if (CG == 1) mbar_arrive(&tempty_bar[buf]); else mbar_arrive_cluster(&tempty_bar[buf], 0);
            }
            if (threadIdx.x == 64) LT_ADD(5, LT_CLK() - te0_);
            if (sp_zero_out) {
                if (warp == 2 && lane == 0) {
                    const unsigned long long v = (unsigned long long)(sp_zc < 3 ? sp_zc + 1 : 3) << 62;
                    bn_next[(size_t)wi.I * p.nb + wi.J] = v;
                    bn_next[(size_t)wi.J * p.nb + wi.I] = v;
                }
            } else if (sp_offdiag) {
                // the block's squared Frobenius norm decides whether the NEXT layer sees it, and -- now -- whether it
                // counts in N_X = ||S'_n||_F^2 (the oracle squares the truncated matrix)
                for (int o = 16; o > 0; o >>= 1) tile48 += __shfl_xor_sync(0xffffffffu, tile48, o);
                const int par = it & 1;
                if (lane == 0) red48[par][ew] = tile48;
                asm volatile("bar.sync 1, %0;\n" ::"n"(32 * C::EPI_WARPS) : "memory");
                unsigned long long tot = 0;
#pragma unroll
                for (int i = 0; i < C::EPI_WARPS; ++i) tot += red48[par][i];
                if (tot > ctrl->tau2_fx48) off2 += tile40;
                if (warp == 2 && lane == 0) {
                    const unsigned long long v = tot < kBnNormMask ? tot : kBnNormMask;
                    bn_next[(size_t)wi.I * p.nb + wi.J] = v;
                    bn_next[(size_t)wi.J * p.nb + wi.I] = v;
                }
            }
        }
        if (threadIdx.x == 64) LT_MARK(3);
        // ---- block partials -> ctrl -> last CTA runs the control step (integer adds: exact, any order)
        fx_t fro2 = 2 * off2 + dg2;
        for (int o = 16; o > 0; o >>= 1) {
            trS += __shfl_xor_sync(0xffffffffu, trS, o);
            fro2 += __shfl_xor_sync(0xffffffffu, fro2, o);
            trX += __shfl_xor_sync(0xffffffffu, trX, o);
        }
        bad = __any_sync(0xffffffffu, bad);
        if (lane == 0) { red[ew][0] = trS; red[ew][1] = fro2; red[ew][2] = trX; red[ew][3] = bad ? 1 : 0; }
        asm volatile("bar.sync 1, %0;\n" ::"n"(32 * C::EPI_WARPS) : "memory");     // the epilogue warps only
        if (warp == 2) {
            unsigned int done = 0;
            if (lane == 0) {
                fx_t a = 0, b = 0, c = 0, f = 0;
                for (int i = 0; i < C::EPI_WARPS; ++i) { a += red[i][0]; b += red[i][1]; c += red[i][2]; f += red[i][3]; }
                ctrl->ipartial[blockIdx.x][0] = a;
                ctrl->ipartial[blockIdx.x][1] = b;
                ctrl->ipartial[blockIdx.x][2] = c;
                ctrl->ipartial[blockIdx.x][3] = f;
                asm volatile("fence.proxy.async;\n" ::: "memory");     // persistent mode: other CTAs TMA-load what was stored
                __threadfence();
                done = atomicAdd(&ctrl->done_counter, 1u);
            }
            done = __shfl_sync(0xffffffffu, done, 0);
            if (done == gridDim.x - 1) {
                // last CTA: sum the per-CTA partials and run the control step of Alg. 1
                __threadfence();
                fx_t a = 0, b = 0, c = 0, f = 0;
                // L2 loads (the partials were written by other SMs), 32-byte vectors, all of a lane's loads in flight
                // before the first add
                for (unsigned int i0 = lane; i0 < gridDim.x; i0 += 128) {
                    longlong4 v[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const unsigned int i = i0 + 32u * u;
                        v[u] = make_longlong4(0, 0, 0, 0);
                        if (i < gridDim.x) {
                            const longlong2 lo = __ldcg(reinterpret_cast<const longlong2*>(ctrl->ipartial[i]));
                            const longlong2 hi = __ldcg(reinterpret_cast<const longlong2*>(ctrl->ipartial[i]) + 1);
                            v[u] = make_longlong4(lo.x, lo.y, hi.x, hi.y);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) { a += v[u].x; b += v[u].y; c += v[u].z; f += v[u].w; }
                }
                for (int o = 16; o > 0; o >>= 1) {
                    a += __shfl_xor_sync(0xffffffffu, a, o);
                    b += __shfl_xor_sync(0xffffffffu, b, o);
                    c += __shfl_xor_sync(0xffffffffu, c, o);
                    f += __shfl_xor_sync(0xffffffffu, f, o);
                }
                if (lane == 0) {
                    control_finish_layer(ctrl, p.stats, p.thetas, a, b, c, f != 0);
                    __threadfence();
                    if (p.cond_handle != 0) cudaGraphSetConditional(p.cond_handle, ctrl->running ? 1u : 0u);
                    if (p.persist)       // release the grid: layer n_at_entry + layer + 1 of the solve is applied
                        asm volatile("st.release.gpu.global.s32 [%0], %1;\n" ::"l"(&ctrl->layer_gen), "r"(ctrl->n) : "memory");
                }
            }
        }
        if (!p.persist) break;
        // this thread's stores of the layer (S, the operand pair, row sums) must be ordered before the next layer's
        // TMA loads of other CTAs: they are released through the done counter above; here the warp just waits
        if (!layer_barrier(ctrl, n_at_entry + layer + 1, lane)) break;
        }
    }

    // ---- teardown
    tc_fence_before();
    if (CG == 2) cluster_sync_all(); else __syncthreads();
    if (warp == 1) tmem_dealloc<CG>(tmem_base, C::TMEM_COLS);
    if (threadIdx.x == 64) LT_MARK(4);
}

using Cfg128 = TileCfg<128, 1>;
using Cfg256 = TileCfg<256, 1>;
using Cfg256P = TileCfg<256, 2>;
// eight epilogue warps for the plain and the blocked-sparse layers (their epilogue is exposed at small N); four for the
// enhanced-accumulation and output-mix instantiations, whose chunk code needs the registers (measured: no gain from eight)
using Cfg128E = TileCfg<128, 1, true, false, false, 4>;
using Cfg128M = TileCfg<128, 1, false, true, false, 4>;
using Cfg256PM = TileCfg<256, 2, false, true, false, 4>;
using Cfg128S = TileCfg<128, 1, false, false, true>;

int tile_super_edge(int cfg) { return (cfg == TILE_128x128 || cfg == TILE_128x128_ENH) ? 128 : 256; }
int tile_subs(int cfg) { return cfg == TILE_128x256 ? Cfg256::SUB : 1; }
int tile_cta_group(int cfg) { return cfg == TILE_256x256_PAIR ? 2 : 1; }
int layer_slots(int cfg, int n_items, int num_sms) {
    const int cg = tile_cta_group(cfg);
    int slots = num_sms / cg;
    if (slots > n_items) slots = n_items;
    if (slots * cg > kMaxPartials) slots = kMaxPartials / cg;
    return slots;
}
size_t tile_smem_bytes(int cfg) {
    return cfg == TILE_128x128 ? Cfg128::SMEM_BYTES : cfg == TILE_128x128_ENH ? Cfg128E::SMEM_BYTES :
           cfg == TILE_128x256 ? Cfg256::SMEM_BYTES : Cfg256P::SMEM_BYTES;
}

cudaError_t layer_kernel_setup(int cfg) {
    switch (cfg) {
        case TILE_128x128:
            return cudaFuncSetAttribute(k_sp2_layer<Cfg128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        Cfg128::SMEM_BYTES);
        case TILE_128x256:
            return cudaFuncSetAttribute(k_sp2_layer<Cfg256>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        Cfg256::SMEM_BYTES);
        case TILE_256x256_PAIR:
            return cudaFuncSetAttribute(k_sp2_layer<Cfg256P>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        Cfg256P::SMEM_BYTES);
        case TILE_128x128_ENH: {
            cudaError_t e = cudaFuncSetAttribute(k_sp2_layer<Cfg128E>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                 Cfg128E::SMEM_BYTES);
            if (e != cudaSuccess) return e;
            // the output-mix instantiations (generalized network with Eq. 18's sum) ride along
            e = cudaFuncSetAttribute(k_sp2_layer<Cfg128M>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     Cfg128M::SMEM_BYTES);
            if (e != cudaSuccess) return e;
            e = cudaFuncSetAttribute(k_sp2_layer<Cfg128S>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     Cfg128S::SMEM_BYTES);
            if (e != cudaSuccess) return e;
            return cudaFuncSetAttribute(k_sp2_layer<Cfg256PM>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        Cfg256PM::SMEM_BYTES);
        }
    }
    return cudaErrorInvalidValue;
}

template <class C>
static cudaError_t launch_cfg(const CUtensorMap& tm_hi, const CUtensorMap& tm_lo, const CUtensorMap& tm_hi1,
                              const CUtensorMap& tm_lo1, const LayerParams& p, int num_sms, cudaStream_t st) {
    (void)num_sms;
    const int slots = p.n_slots;          // chosen by the host together with the item list (layer_slots)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(slots * C::CG));
    cfg.blockDim = dim3(C::THREADS);
    cfg.dynamicSmemBytes = C::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = C::CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (p.persist) {                      // the grid barrier between layers needs every CTA resident: cooperative launch
        attr[1].id = cudaLaunchAttributeCooperative;
        attr[1].val.cooperative = 1;
        cfg.numAttrs = 2;
    }
    return cudaLaunchKernelEx(&cfg, k_sp2_layer<C>, tm_hi, tm_lo, tm_hi1, tm_lo1, p);
}

cudaError_t launch_layer(int cfg, const CUtensorMap& tm_hi, const CUtensorMap& tm_lo, const CUtensorMap& tm_hi1,
                         const CUtensorMap& tm_lo1, const LayerParams& p, int num_sms, cudaStream_t st) {
    if (p.bn_cur != nullptr) {           // blocked-sparse variant: 128x128 tiles only
        if (cfg == TILE_128x128 && p.mix == nullptr) return launch_cfg<Cfg128S>(tm_hi, tm_lo, tm_hi1, tm_lo1, p, num_sms, st);
        return cudaErrorInvalidValue;
    }
    if (p.mix != nullptr) {              // output mix: 128x128 or pair tiles only
        if (cfg == TILE_128x128) return launch_cfg<Cfg128M>(tm_hi, tm_lo, tm_hi1, tm_lo1, p, num_sms, st);
        if (cfg == TILE_256x256_PAIR) return launch_cfg<Cfg256PM>(tm_hi, tm_lo, tm_hi1, tm_lo1, p, num_sms, st);
        return cudaErrorInvalidValue;
    }
    switch (cfg) {
        case TILE_128x128: return launch_cfg<Cfg128>(tm_hi, tm_lo, tm_hi1, tm_lo1, p, num_sms, st);
        case TILE_128x256: return launch_cfg<Cfg256>(tm_hi, tm_lo, tm_hi1, tm_lo1, p, num_sms, st);
        case TILE_256x256_PAIR: return launch_cfg<Cfg256P>(tm_hi, tm_lo, tm_hi1, tm_lo1, p, num_sms, st);
        case TILE_128x128_ENH: return launch_cfg<Cfg128E>(tm_hi, tm_lo, tm_hi1, tm_lo1, p, num_sms, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace sp2
