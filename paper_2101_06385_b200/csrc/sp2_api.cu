// C ABI of libsp2b200.so (include/sp2_b200.h): handle / workspace lifecycle, TMA tensor maps, the CUDA graph
// that holds the device-side layer loop, and the solve entry points.
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <mutex>
#include <tuple>
#include <vector>

#include "sp2_kernels.h"

using namespace sp2;

static thread_local char g_cuda_err[512] = "";

static sp2_status_t cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
    return SP2_ERR_CUDA;
}
#define CK(call)                                              \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct LoopGraph {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
};

struct sp2_handle_s {
    int N_max = 0, batch_max = 0, max_layers = 0;
    int Np_max = 0;
    int num_sms = 0, device = 0;
    // single-matrix workspace
    float* S = nullptr;
    __half* hl[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};   // [ping-pong][hi, lo]
    float* gpart = nullptr;         // Gershgorin: per-tile row / column sums (gershgorin_part_floats)
    double* diag = nullptr;
    unsigned long long* rowsq[2] = {nullptr, nullptr};   // fixed-point row sums of squares of S (ping-pong)
    Ctrl* ctrl = nullptr;
    sp2_layer_stat_t* stats_dev = nullptr;
    float* thetas_dev = nullptr;
    WorkItem* items_dev[2] = {nullptr, nullptr};   // [0] solves, [1] refinement layers (different tile config)
    int items_cap = 0;
    // batched workspace
    sp2_layer_stat_t* bstats_dev = nullptr;
    int* bnl_dev = nullptr;
    int* bstatus_dev = nullptr;
    double* bbounds_dev = nullptr;
    long long* bnocc_dev = nullptr;        // per-matrix N_occ, 2^40 fixed point
    long long* bnocc_host = nullptr;
    double* bhl_dev = nullptr;      // [batch][2] HOMO / LUMO estimates of the accelerated batched solve
    // pinned host mirrors of the batched outputs (a device -> pageable copy is staged and slow: 2.9 MB of statistics
    // for 1024 matrices cost ~1 ms, a fifth of the whole batched solve)
    sp2_layer_stat_t* bstats_host = nullptr;
    int* bnl_host = nullptr;        // [batch] layers, then [batch] status
    double* bbounds_host = nullptr;
    // pinned host mirrors
    Ctrl* ctrl_host = nullptr;
    sp2_layer_stat_t* stats_host = nullptr;
    float* thetas_host = nullptr;          // pinned; what is uploaded (FP32, the epilogue's type)
    double* bounds_host = nullptr;
    // host staging for the *_host entry point
    float* stage_H = nullptr;
    float* stage_D = nullptr;
    size_t stage_elems = 0;
    cudaEvent_t host_ev[4] = {nullptr, nullptr, nullptr, nullptr};   // H2D start, solve start, D2H start, end
    float host_ms[3] = {0.f, 0.f, 0.f};
    double host_bytes[2] = {0.0, 0.0};   // bytes the last sp2_density_matrix_host call copied: host -> device, device -> host
    PFN_encodeTiled encode = nullptr;
    // (N, Np, cfg, scale_log2, exact_diag | mix << 1 | sparse << 2 | enh_kc << 3): everything a captured launch bakes in
    std::map<std::tuple<int, int, int, int, int>, LoopGraph> graphs;
    int items_key_np[2] = {-1, -1}, items_key_cfg[2] = {-1, -1}, items_key_split[2] = {-1, -1};
    int n_items[2] = {0, 0}, n_slots[2] = {0, 0};
    float* mix = nullptr;           // output mix M = sum_i c_i S_i (Eq. 18), allocated on first use
    unsigned long long* bn[2] = {nullptr, nullptr};   // blocked-sparse variant: squared block norms (ping-pong), on first use
    double sparse_work[2] = {0.0, 0.0};               // K-blocks multiplied / a dense solve's, last sparse solve
    double* obs_dev = nullptr;      // [6] observables of sp2_refine_energy
    double* obs_host = nullptr;
    int tail_split = 1;
    int last_launches = 0;
    int round_sync = 1;
    unsigned int round_spins = 1u << 16;
    int ki_edge = 32, ki_mid = 32;   // K-interleave chunking (performance only; SP2_K_INTERLEAVE=edge[:mid], 0 = off)
    cudaStream_t cap_stream = nullptr;
};

static int round_up(int x, int m) { return (x + m - 1) / m * m; }

static size_t ctrl_header_bytes() { return sizeof(CtrlCore); }

extern "C" const char* sp2_status_string(sp2_status_t s) {
    switch (s) {
        case SP2_OK: return "SP2_OK";
        case SP2_NOT_CONVERGED: return "SP2_NOT_CONVERGED";
        case SP2_ERR_INVALID_ARG: return "SP2_ERR_INVALID_ARG";
        case SP2_ERR_BOUNDS_DEGENERATE: return "SP2_ERR_BOUNDS_DEGENERATE";
        case SP2_ERR_NONFINITE: return "SP2_ERR_NONFINITE";
        case SP2_ERR_WORKSPACE: return "SP2_ERR_WORKSPACE";
        case SP2_ERR_CUDA: return "SP2_ERR_CUDA";
        case SP2_ERR_UNSUPPORTED_N: return "SP2_ERR_UNSUPPORTED_N";
    }
    return "SP2_UNKNOWN";
}
extern "C" const char* sp2_last_cuda_error(void) { return g_cuda_err; }
extern "C" const char* sp2_version(void) { return "sp2b200 0.1 (sm_100a)"; }

extern "C" void sp2_default_opts(sp2_opts_t* o) {
    if (!o) return;
    o->auto_bounds = 1;
    o->eps_min = 0.0;
    o->eps_max = 0.0;
    o->tol = 0.0;
    o->max_layers = 120;
    o->eps_alt = 0.0;
    o->fp16_scale_log2 = -1;
    o->control = 0;
    o->tile_config = 0;
    o->exact_diag = 1;
    o->accelerated = 0;
    o->homo = 0.0;
    o->lumo = 0.0;
    o->noise_kappa = -1.0;
    o->enh_kc = 0;
    o->trunc_tau = 0.0;
}

static double opt_kappa(const sp2_opts_t& o) { return o.noise_kappa < 0.0 ? 0.125 : o.noise_kappa; }
// kappa as a 16.16 fixed-point factor for the integer control step (sp2_control.cuh); 0 disables the test
static int opt_kappa_q16(const sp2_opts_t& o) {
    const double k = opt_kappa(o);
    if (!(k > 0.0)) return 0;
    const double q = k * 65536.0 + 0.5;
    return q >= 2147483647.0 ? 2147483647 : (q < 1.0 ? 1 : (int)q);
}
// fixed-point image of a host double, saturated well inside the 64-bit range
static fx_t to_fx(double x) {
    if (!(x == x)) return 0;
    if (x > 4.0e6) x = 4.0e6;
    if (x < -4.0e6) x = -4.0e6;
    return fx_from_double_host(x);
}
static void stats_to_double(sp2_layer_stat_t* st, int n) {       // the device writes raw fixed-point integers
    for (int i = 0; i < n; ++i) {
        fx_t v[4];
        memcpy(&v[0], &st[i].trace_S, 8); memcpy(&v[1], &st[i].trace_X, 8);
        memcpy(&v[2], &st[i].trace_X_diag, 8); memcpy(&v[3], &st[i].iderr, 8);
        st[i].trace_S = fx_to_double(v[0]); st[i].trace_X = fx_to_double(v[1]);
        st[i].trace_X_diag = fx_to_double(v[2]); st[i].iderr = fx_to_double(v[3]);
    }
}
static int opt_enh_kc(const sp2_opts_t* o) { return (o && o->enh_kc > 0) ? o->enh_kc : 4; }

extern "C" size_t sp2_workspace_bytes(int N_max, int batch_max, int max_layers) {
    if (N_max < 1 || max_layers < 1) return 0;
    const size_t Np = (size_t)round_up(N_max, 256);
    size_t b = Np * (size_t)ws_ld_f32((int)Np) * 4 + 4 * Np * (size_t)ws_ld_f16((int)Np) * 2;   // S + two hi/lo pairs
    b += gershgorin_part_floats((int)Np) * 4;                 // Gershgorin per-tile sums
    b += 3 * Np * sizeof(double);                             // diagonal, two row-sum vectors
    b += sizeof(Ctrl) + (size_t)max_layers * (sizeof(sp2_layer_stat_t) + kThetaStride * sizeof(double));
    b += 2 * ((Np / 128) * (Np / 128 + 1) / 2 + 1024) * sizeof(WorkItem);
    b += (size_t)(batch_max > 0 ? batch_max : 1) *
         ((size_t)max_layers * sizeof(sp2_layer_stat_t) + 2 * sizeof(int) + 5 * sizeof(double));
    return b;
}

// Allocations made on first use (see the header): the output-mix matrix, the two staging matrices of the host entry
// point at N = N_max, the block norms of the blocked-sparse variant.
extern "C" size_t sp2_workspace_bytes_lazy(int N_max) {
    if (N_max < 1) return 0;
    const size_t Np = (size_t)round_up(N_max, 256);
    const size_t nb = Np / 128;
    return Np * (size_t)ws_ld_f32((int)Np) * 4 + 2 * (size_t)N_max * (size_t)N_max * 4 + 2 * nb * nb * sizeof(double);
}

extern "C" sp2_status_t sp2_destroy(sp2_handle_t h) {
    if (!h) return SP2_ERR_INVALID_ARG;
    for (auto& kv : h->graphs) {
        if (kv.second.exec) cudaGraphExecDestroy(kv.second.exec);
        if (kv.second.graph) cudaGraphDestroy(kv.second.graph);
    }
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    for (int i = 0; i < 4; ++i) if (h->host_ev[i]) cudaEventDestroy(h->host_ev[i]);
    cudaFree(h->S);
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) cudaFree(h->hl[a][b]);
    cudaFree(h->rowsq[0]); cudaFree(h->rowsq[1]);
    cudaFree(h->gpart); cudaFree(h->diag); cudaFree(h->ctrl); cudaFree(h->stats_dev); cudaFree(h->thetas_dev);
    cudaFree(h->items_dev[0]); cudaFree(h->items_dev[1]); cudaFree(h->obs_dev); cudaFree(h->mix); cudaFree(h->bn[0]); cudaFree(h->bn[1]); cudaFreeHost(h->obs_host); cudaFree(h->bstats_dev); cudaFree(h->bnl_dev); cudaFree(h->bstatus_dev);
    cudaFree(h->bbounds_dev); cudaFree(h->bnocc_dev); cudaFree(h->bhl_dev);
    cudaFreeHost(h->ctrl_host); cudaFreeHost(h->stats_host); cudaFreeHost(h->thetas_host);
    cudaFreeHost(h->bounds_host); cudaFree(h->stage_H); cudaFree(h->stage_D);
    cudaFreeHost(h->bstats_host); cudaFreeHost(h->bnl_host); cudaFreeHost(h->bbounds_host); cudaFreeHost(h->bnocc_host);
    delete h;
    return SP2_OK;
}

extern "C" sp2_status_t sp2_create(sp2_handle_t* out, int N_max, int batch_max, int max_layers) {
    if (!out || N_max < 1 || batch_max < 0 || max_layers < 1 || max_layers > 4096) return SP2_ERR_INVALID_ARG;
    int dev = 0;
    CK(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "device is sm_%d%d; this library is built for sm_100a only", prop.major,
                 prop.minor);
        return SP2_ERR_CUDA;
    }
    sp2_handle_s* h = new sp2_handle_s();
    h->N_max = N_max; h->batch_max = batch_max; h->max_layers = max_layers;
    // performance toggles only (results are bit-identical for any setting)
    if (const char* e = getenv("SP2_TAIL_SPLIT")) h->tail_split = atoi(e);
    if (const char* e = getenv("SP2_ROUND_SYNC")) h->round_sync = atoi(e);
    if (const char* e = getenv("SP2_K_INTERLEAVE")) {
        int a = 0, b = 0;
        const int n = sscanf(e, "%d:%d", &a, &b);
        if (n >= 1) { h->ki_edge = a < 0 ? 0 : a; h->ki_mid = (n >= 2 && b > 0) ? b : h->ki_edge; }
    }
    if (const char* e = getenv("SP2_ROUND_SYNC_SPINS")) { const long v = atol(e); h->round_spins = v < 1 ? 1u : (unsigned int)v; }
    h->Np_max = round_up(N_max, 256);
    h->num_sms = prop.multiProcessorCount; h->device = dev;
    const size_t Np = (size_t)h->Np_max;
    sp2_status_t st = SP2_OK;
    auto A = [&](void** p, size_t bytes) {
        if (st != SP2_OK) return;
        cudaError_t e = cudaMalloc(p, bytes);
        if (e != cudaSuccess) st = cuda_fail(e, "cudaMalloc(workspace)");
    };
    A((void**)&h->S, Np * (size_t)ws_ld_f32(h->Np_max) * 4);
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) A((void**)&h->hl[a][b], Np * (size_t)ws_ld_f16(h->Np_max) * 2);
    A((void**)&h->gpart, gershgorin_part_floats(h->Np_max) * sizeof(float));
    A((void**)&h->diag, Np * sizeof(double));
    A((void**)&h->rowsq[0], Np * sizeof(unsigned long long));
    A((void**)&h->rowsq[1], Np * sizeof(unsigned long long));
    A((void**)&h->ctrl, sizeof(Ctrl));
    A((void**)&h->stats_dev, (size_t)max_layers * sizeof(sp2_layer_stat_t));
    A((void**)&h->thetas_dev, (size_t)max_layers * kThetaStride * sizeof(float));
    h->items_cap = (int)((Np / 128) * (Np / 128 + 1) / 2) + 1024;
    A((void**)&h->items_dev[0], (size_t)h->items_cap * sizeof(WorkItem));
    A((void**)&h->items_dev[1], (size_t)h->items_cap * sizeof(WorkItem));
    A((void**)&h->obs_dev, 8 * sizeof(double));
    {   // at least one slot: single matrices of N <= 256 are solved by the resident kernel too
        const size_t bm = (size_t)(batch_max > 0 ? batch_max : 1);
        A((void**)&h->bstats_dev, bm * max_layers * sizeof(sp2_layer_stat_t));
        A((void**)&h->bnl_dev, bm * sizeof(int));
        A((void**)&h->bstatus_dev, bm * sizeof(int));
        A((void**)&h->bbounds_dev, bm * 2 * sizeof(double));
        A((void**)&h->bnocc_dev, bm * sizeof(long long));
        A((void**)&h->bhl_dev, bm * 2 * sizeof(double));
    }
    auto AH = [&](void** p, size_t bytes) {
        if (st != SP2_OK) return;
        cudaError_t e = cudaMallocHost(p, bytes);
        if (e != cudaSuccess) st = cuda_fail(e, "cudaMallocHost");
    };
    AH((void**)&h->ctrl_host, sizeof(Ctrl));
    AH((void**)&h->stats_host, (size_t)max_layers * sizeof(sp2_layer_stat_t));
    AH((void**)&h->thetas_host, (size_t)max_layers * kThetaStride * sizeof(float));
    AH((void**)&h->bounds_host, 2 * sizeof(double));
    AH((void**)&h->obs_host, 8 * sizeof(double));
    {
        const size_t bm = (size_t)(batch_max > 0 ? batch_max : 1);
        AH((void**)&h->bstats_host, bm * max_layers * sizeof(sp2_layer_stat_t));
        AH((void**)&h->bnl_host, bm * 2 * sizeof(int));
        AH((void**)&h->bbounds_host, bm * 2 * sizeof(double));
        AH((void**)&h->bnocc_host, bm * sizeof(long long));
    }
    if (st == SP2_OK) {
        cudaError_t e = cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) st = cuda_fail(e, "cudaStreamCreate");
    }
    if (st == SP2_OK) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
        if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn)
            st = cuda_fail(e == cudaSuccess ? cudaErrorUnknown : e, "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled)");
        h->encode = (PFN_encodeTiled)fn;
    }
    for (int cfg = TILE_128x128; cfg <= TILE_128x128_ENH && st == SP2_OK; ++cfg) {
        cudaError_t e = layer_kernel_setup(cfg);
        if (e != cudaSuccess) st = cuda_fail(e, "cudaFuncSetAttribute(layer kernel)");
    }
    if (st == SP2_OK) {
        cudaError_t e = resident_kernel_setup();
        if (e != cudaSuccess) st = cuda_fail(e, "cudaFuncSetAttribute(resident kernel)");
    }
    if (st != SP2_OK) { sp2_destroy(h); return st; }
    *out = h;
    return SP2_OK;
}

// K-major FP16 operand map: Np x Np row-major (leading dimension ws_ld_f16), box = 64 (K) x 128 (rows),
// 128-byte swizzle.
static sp2_status_t make_tmap(sp2_handle_s* h, CUtensorMap* tm, void* base, int Np) {
    cuuint64_t gdim[2] = {(cuuint64_t)Np, (cuuint64_t)Np};
    cuuint64_t gstr[1] = {(cuuint64_t)ws_ld_f16(Np) * 2};
    cuuint32_t box[2] = {64, 128};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = h->encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, base, gdim, gstr, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled failed: %d", (int)r);
        return SP2_ERR_CUDA;
    }
    return SP2_OK;
}

// Band plan of the work list: the lower triangle of the nt x nt supertile grid is cut into bands of supertile rows,
// [b_0 = 0, b_1), [b_1, b_2), ..., and the list walks each band column by column.  The `per` consecutive items of an
// epoch (two rounds of n_slots tiles, walked through K together: see ki_range in sp2_square_tiled.cu) then form a
// rectangle of ~r x c supertiles that touches r + c row panels, and every panel an epoch touches is fetched from HBM
// once.  The number of items in front of a band that starts at row a is a (a + 1) / 2 whatever the bands before it,
// so the cost of a band (distinct panels per epoch, summed over the epochs that intersect it) depends on (a, b) only
// and the best boundaries follow from a shortest-path recursion over b.  Bands are at most hmax rows high (the
// panels of one round of an epoch, r + c / 2, must stay inside the L2 window).  N = 16384, pair tiles (nt = 64,
// per = 148, hmax = 17): 336 panel loads per layer against 506 for fixed bands of 8 walked round by round.
static std::vector<int> plan_bands(int nt, int per, int hmax) {
    std::vector<long long> best((size_t)nt + 1, -1);
    std::vector<int> prev((size_t)nt + 1, -1);
    std::vector<int> seen((size_t)nt, -1);
    best[0] = 0;
    for (int b = 1; b <= nt; ++b)
        for (int a = (b > hmax ? b - hmax : 0); a < b; ++a) {
            if (best[(size_t)a] < 0) continue;
            long long idx = (long long)a * (a + 1) / 2, cost = 0, cur = -1;
            for (int j = 0; j < b; ++j)
                for (int i = (j > a ? j : a); i < b; ++i, ++idx) {
                    const long long e = idx / per;
                    if (e != cur) { cur = e; std::fill(seen.begin(), seen.end(), -1); }
                    if (seen[(size_t)i] < 0) { seen[(size_t)i] = 1; ++cost; }
                    if (seen[(size_t)j] < 0) { seen[(size_t)j] = 1; ++cost; }
                }
            const long long c = best[(size_t)a] + cost;
            if (best[(size_t)b] < 0 || c < best[(size_t)b]) { best[(size_t)b] = c; prev[(size_t)b] = a; }
        }
    std::vector<int> bounds;
    for (int b = nt; b > 0; b = prev[(size_t)b]) bounds.push_back(b);
    bounds.push_back(0);
    std::reverse(bounds.begin(), bounds.end());
    return bounds;
}

// Work list of a layer (launch order).  Supertiles of the lower triangle in bands of supertile rows (plan_bands),
// column-major inside a band, so that the CTAs of one epoch (2 n_slots consecutive items run in K-lockstep) share few
// row panels (L2 reuse of the operands).  If the last round is partial and short enough, its items are cut into
// 2 or 4 column strips each (ncols = E/2, E/4 >= 64): more CTAs share the tail and it ends sooner.
static void build_work_list(int nt, int band, int edge, int subs, int cta_group, int num_sms, int tail_split,
                            std::vector<WorkItem>& out, int* n_slots) {
    out.clear();
    std::vector<int> bounds;
    if (band > 0) {
        for (int i0 = 0; i0 < nt; i0 += band) bounds.push_back(i0);
        bounds.push_back(nt);
    } else {
        int sl = num_sms / cta_group;
        if (sl * cta_group > kMaxPartials) sl = kMaxPartials / cta_group;
        const int per_tiles = (2 * sl) / subs > 0 ? (2 * sl) / subs : 1;
        bounds = plan_bands(nt, per_tiles, 17);      // measured at N = 16384: 12: 9.65, 14: 9.63, 17: 9.61 ms per layer
    }
    for (size_t bi = 0; bi + 1 < bounds.size(); ++bi) {
        const int i0 = bounds[bi], i1 = bounds[bi + 1];
        for (int j = 0; j < i1; ++j)
            for (int i = (j > i0 ? j : i0); i < i1; ++i)
                for (int sub = 0; sub < subs; ++sub) {
                    WorkItem w = {};
                    w.I = (short)i; w.J = (short)j; w.sub = (short)sub; w.col0 = 0; w.ncols = (short)edge;
                    out.push_back(w);
                }
    }
    int slots = num_sms / cta_group;
    if (slots > (int)out.size()) slots = (int)out.size();
    if (slots * cta_group > kMaxPartials) slots = kMaxPartials / cta_group;
    *n_slots = slots;
    const int n = (int)out.size();
    const int r = n % slots;
    if (!tail_split || n <= slots || r == 0) return;
    int f = 1;
    while (f < 4 && r * (2 * f) <= slots && edge / (2 * f) >= 64) f *= 2;
    if (f == 1) return;
    std::vector<WorkItem> tail(out.end() - r, out.end());
    out.resize((size_t)(n - r));
    for (int q = 0; q < f; ++q)
        for (const WorkItem& t : tail) {
            WorkItem w = t;
            w.ncols = (short)(edge / f);
            w.col0 = (short)(q * (edge / f));
            out.push_back(w);
        }
}

static int choose_tile_config(int N, int requested, int num_sms) {
    if (requested >= TILE_128x128 && requested <= TILE_128x128_ENH) return requested;
    const int n128 = round_up(N, 128) / 128;
    const long long t128 = (long long)n128 * (n128 + 1) / 2;
    // 128 x 128 single-CTA tiles up to ~1.75 rounds of them (N <= 2816 on 148 SMs), 256 x 256 pair tiles above: at
    // 128 x 128 a pipeline stage is 768 cycles of tensor-pipe time and what the issuing thread does between two stages is
    // exposed (measured ~1100 cycles per stage in the kernel, tests/cuda/mma_rate.cu), so small tiles only pay while they
    // put more SMs to work.  Measured us per layer, tile 1 / tile 3: N = 2048: 47.8 / 68.9, 2304: 66.7 / 71.7,
    // 2560: 71.7 / 76.6, 2816: 82.8 / 82.5, 3072: 113.0 / 106.9, 3584: 159.5 / 151.1, 4096: 227.5 / 198.7.
    if (4 * t128 > 7LL * num_sms) return TILE_256x256_PAIR;
    return TILE_128x128;
}

struct Problem {
    int N, Np, cfg, scale_log2, n_items, n_slots, exact_diag, list, mix, enh_kc, sparse;
    float scale, inv_scale2;
};

static sp2_status_t prepare_problem(sp2_handle_s* h, int N, const sp2_opts_t* o, Problem* pb, cudaStream_t st,
                                    int forced_cfg = 0) {
    pb->N = N;
    pb->cfg = forced_cfg ? forced_cfg : choose_tile_config(N, o ? o->tile_config : 0, h->num_sms);
    pb->list = (pb->cfg == TILE_128x128_ENH) ? 1 : 0;   // the enhanced-accumulation layers keep their own work list
    pb->mix = 0;
    pb->sparse = (o && o->trunc_tau > 0.0) ? 1 : 0;
    if (pb->sparse) {                                      // 128 x 128 tiles, no strips: a block = a tile
        if (forced_cfg || (o->tile_config != TILE_AUTO && o->tile_config != TILE_128x128)) return SP2_ERR_INVALID_ARG;
        pb->cfg = TILE_128x128;
    }
    const int L = pb->list;
    const int edge = tile_super_edge(pb->cfg);
    pb->Np = round_up(N, edge);
    if (pb->Np > h->Np_max) return SP2_ERR_WORKSPACE;
    int k = o ? o->fp16_scale_log2 : -1;
    if (k < 0) k = 13;
    if (k > 14) return SP2_ERR_INVALID_ARG;
    pb->scale_log2 = k;
    pb->exact_diag = (o && o->exact_diag == 0) ? 0 : 1;
    if (pb->sparse) pb->exact_diag = 0;      // the diagonal of X comes from the (masked) tensor-core products
    pb->enh_kc = opt_enh_kc(o);
    pb->scale = ldexpf(1.0f, k);
    pb->inv_scale2 = ldexpf(1.0f, -2 * k);
    const int nt = pb->Np / edge;
    // planned bands (plan_bands) for the plain layers; the enhanced-accumulation layers (no K-interleave) keep fixed ones
    const int band = (pb->cfg == TILE_128x128_ENH) ? 12 : 0;
    const int split = pb->sparse ? 0 : h->tail_split;
    if (h->items_key_np[L] != pb->Np || h->items_key_cfg[L] != pb->cfg || h->items_key_split[L] != split) {
        std::vector<WorkItem> list;
        int slots = 0;
        build_work_list(nt, band, edge, tile_subs(pb->cfg), tile_cta_group(pb->cfg), h->num_sms, split, list,
                        &slots);
        if ((int)list.size() > h->items_cap) return SP2_ERR_WORKSPACE;
        // synchronous small copy: happens only when the problem shape changes
        CK(cudaMemcpyAsync(h->items_dev[L], list.data(), list.size() * sizeof(WorkItem), cudaMemcpyHostToDevice, st));
        CK(cudaStreamSynchronize(st));
        h->items_key_np[L] = pb->Np; h->items_key_cfg[L] = pb->cfg; h->items_key_split[L] = split;
        h->n_items[L] = (int)list.size();
        h->n_slots[L] = slots;
    }
    pb->n_items = h->n_items[L];
    pb->n_slots = h->n_slots[L];
    return SP2_OK;
}

static LayerParams layer_params(sp2_handle_s* h, const Problem& pb, int parity, unsigned long long cond) {
    LayerParams p;
    p.ctrl = h->ctrl; p.stats = h->stats_dev; p.thetas = h->thetas_dev; p.S = h->S;
    p.mix = pb.mix ? h->mix : nullptr;
    p.hi_out = h->hl[parity ^ 1][0]; p.lo_out = h->hl[parity ^ 1][1];
    p.hi_in = h->hl[parity][0]; p.lo_in = h->hl[parity][1];
    p.persist = 0;
    p.rowsq_cur = pb.exact_diag ? h->rowsq[parity] : nullptr;
    p.rowsq_next = pb.exact_diag ? h->rowsq[parity ^ 1] : nullptr;
    p.items = h->items_dev[pb.list]; p.ld = ws_ld_f32(pb.Np); p.ldf = ws_ld_f16(pb.Np); p.N = pb.N; p.Np = pb.Np;
    p.n_items = pb.n_items; p.n_slots = pb.n_slots;
    p.bn_cur = pb.sparse ? h->bn[parity] : nullptr; p.bn_next = pb.sparse ? h->bn[parity ^ 1] : nullptr;
    p.nb = pb.Np / 128;
    p.scale = pb.scale; p.inv_scale2 = pb.inv_scale2; p.cond_handle = cond; p.round_sync = h->round_sync; p.round_spins = h->round_spins; p.enh_kc = pb.enh_kc;
    p.ki_edge = h->ki_edge; p.ki_mid = h->ki_mid;
    return p;
}

// persist = 1: ONE launch runs every layer of the solve (grid barrier between layers, cooperative launch).
static sp2_status_t launch_one_layer(sp2_handle_s* h, const Problem& pb, int parity, unsigned long long cond,
                                     cudaStream_t st, int persist = 0) {
    CUtensorMap tm_hi, tm_lo, tm_hi1, tm_lo1;
    sp2_status_t s = make_tmap(h, &tm_hi, h->hl[parity][0], pb.Np);
    if (s != SP2_OK) return s;
    s = make_tmap(h, &tm_lo, h->hl[parity][1], pb.Np);
    if (s != SP2_OK) return s;
    s = make_tmap(h, &tm_hi1, h->hl[parity ^ 1][0], pb.Np);
    if (s != SP2_OK) return s;
    s = make_tmap(h, &tm_lo1, h->hl[parity ^ 1][1], pb.Np);
    if (s != SP2_OK) return s;
    LayerParams p = layer_params(h, pb, parity, cond);
    p.persist = persist;
    CK(launch_layer(pb.cfg, tm_hi, tm_lo, tm_hi1, tm_lo1, p, h->num_sms, st));
    return SP2_OK;
}

// WHILE(ctrl->running) { layer(ping -> pong); layer(pong -> ping); } as a CUDA graph with a conditional node; the
// condition is set on the device by the last CTA of each layer kernel (cudaGraphSetConditional).
static sp2_status_t get_loop_graph(sp2_handle_s* h, const Problem& pb, LoopGraph** out) {
    auto key = std::make_tuple(pb.N, pb.Np, pb.cfg, pb.scale_log2, pb.exact_diag | (pb.mix << 1) | (pb.sparse << 2) | (pb.enh_kc << 3));
    auto it = h->graphs.find(key);
    if (it != h->graphs.end()) { *out = &it->second; return SP2_OK; }
    if (h->graphs.size() >= 16) {            // bounded cache: start over rather than grow without limit
        for (auto& kv : h->graphs) {
            if (kv.second.exec) cudaGraphExecDestroy(kv.second.exec);
            if (kv.second.graph) cudaGraphDestroy(kv.second.graph);
        }
        h->graphs.clear();
    }
    LoopGraph lg;
    CK(cudaGraphCreate(&lg.graph, 0));
    cudaGraphConditionalHandle handle;
    CK(cudaGraphConditionalHandleCreate(&handle, lg.graph, 1, cudaGraphCondAssignDefault));
    cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = handle;
    np.conditional.type = cudaGraphCondTypeWhile;
    np.conditional.size = 1;
    cudaGraphNode_t node;
    CK(cudaGraphAddNode(&node, lg.graph, nullptr, 0, &np));
    cudaGraph_t body = np.conditional.phGraph_out[0];
    CK(cudaStreamBeginCaptureToGraph(h->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
    sp2_status_t s = launch_one_layer(h, pb, 0, (unsigned long long)handle, h->cap_stream);
    if (s == SP2_OK) s = launch_one_layer(h, pb, 1, (unsigned long long)handle, h->cap_stream);
    cudaGraph_t captured = nullptr;
    cudaError_t e = cudaStreamEndCapture(h->cap_stream, &captured);
    if (s != SP2_OK) { cudaGraphDestroy(lg.graph); return s; }
    if (e != cudaSuccess) { cudaGraphDestroy(lg.graph); return cuda_fail(e, "cudaStreamEndCapture"); }
    e = cudaGraphInstantiate(&lg.exec, lg.graph, 0);
    if (e != cudaSuccess) { cudaGraphDestroy(lg.graph); return cuda_fail(e, "cudaGraphInstantiate"); }
    auto ins = h->graphs.emplace(key, lg);
    *out = &ins.first->second;
    return SP2_OK;
}

// A handle belongs to the device that was current at sp2_create (its workspace and graphs live there).
static sp2_status_t check_device(sp2_handle_s* h) {
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev != h->device) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "handle was created on device %d, current device is %d", h->device, dev);
        return SP2_ERR_INVALID_ARG;
    }
    return SP2_OK;
}

static sp2_status_t check_common(sp2_handle_s* h, const void* in, int N, int ldin, const void* outp, int ldout) {
    if (!h || !in || !outp || N < 1 || ldin < N || ldout < N) return SP2_ERR_INVALID_ARG;
    if (N > h->N_max) return SP2_ERR_WORKSPACE;
    return check_device(h);
}

// Shared body of the single-matrix solves.  mode = MODE_STANDARD or MODE_GENERALIZED (thetas already in
// h->thetas_host[0..3L)).
static sp2_status_t solve_single(sp2_handle_s* h, const float* H_dev, int N, int ldh, double N_occ, int mode,
                                 const sp2_opts_t* o, float* D_dev, int ldd, sp2_layer_stat_t* stats_out,
                                 int* n_layers_out, double bounds_out[2], cudaStream_t st, bool mix = false,
                                 double c0 = 0.0, double mix_diag = 1.0) {
    Problem pb;
    sp2_status_t s = prepare_problem(h, N, o, &pb, st);
    if (s != SP2_OK) return s;
    if (mix) {
        // the mix epilogue exists for tile configurations 1 and 3 only
        if (pb.cfg == TILE_128x256 || pb.cfg == TILE_128x128_ENH) return SP2_ERR_INVALID_ARG;
        if (!h->mix) CK(cudaMalloc((void**)&h->mix, (size_t)h->Np_max * (size_t)ws_ld_f32(h->Np_max) * 4));
        pb.mix = 1;
        if (pb.sparse) return SP2_ERR_INVALID_ARG;
    }
    const int nb = pb.Np / 128;
    if (pb.sparse) {
        if (nb > 128 || !isfinite(o->trunc_tau)) return SP2_ERR_INVALID_ARG;      // the K-block masks hold 128 bits
        const size_t nbm = (size_t)(h->Np_max / 128);
        for (int a = 0; a < 2; ++a)
            if (!h->bn[a]) CK(cudaMalloc((void**)&h->bn[a], nbm * nbm * sizeof(unsigned long long)));
        CK(cudaMemsetAsync(h->bn[0], 0, (size_t)nb * nb * sizeof(unsigned long long), st));
        CK(cudaMemsetAsync(h->bn[1], 0, (size_t)nb * nb * sizeof(unsigned long long), st));
    }
    const int max_layers = o->max_layers;
    // ---- control block
    Ctrl* c = h->ctrl_host;
    memset(c, 0, ctrl_header_bytes());
    c->N_occ = to_fx(N_occ); c->eps_alt = to_fx(o->eps_alt); c->tol = (o->tol > 0.0) ? (to_fx(o->tol) > 0 ? to_fx(o->tol) : 1) : 0;
    c->eps_min = o->eps_min; c->eps_max = o->eps_max;
    c->N = N; c->mode = mode; c->max_layers = max_layers; c->auto_bounds = o->auto_bounds;
    c->kappa_q16 = opt_kappa_q16(*o);
    if (pb.sparse) {
        const double t2 = o->trunc_tau * o->trunc_tau * 281474976710656.0;     // 2^48
        c->tau2_fx48 = t2 >= 9.0e18 ? 9000000000000000000ull : (unsigned long long)llrint(t2);
    }
    c->accelerated = (mode == MODE_STANDARD && o->accelerated) ? 1 : 0;
    c->homo = o->homo; c->lumo = o->lumo;
    CK(cudaMemcpyAsync(h->ctrl, c, ctrl_header_bytes(), cudaMemcpyHostToDevice, st));
    if (mode == MODE_GENERALIZED)
        CK(cudaMemcpyAsync(h->thetas_dev, h->thetas_host, (size_t)max_layers * kThetaStride * sizeof(float),
                           cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(h->stats_dev, 0, (size_t)max_layers * sizeof(sp2_layer_stat_t), st));
    // ---- padding rows/columns of S_0 are zero (inert: eigenvalue 0 is a fixed point of both branches)
    const size_t ldS = (size_t)ws_ld_f32(pb.Np), ldF = (size_t)ws_ld_f16(pb.Np);
    if (pb.Np != N) {
        CK(cudaMemsetAsync(h->S, 0, (size_t)pb.Np * ldS * 4, st));
        if (pb.mix) CK(cudaMemsetAsync(h->mix, 0, (size_t)pb.Np * ldS * 4, st));
        CK(cudaMemsetAsync(h->hl[0][0], 0, (size_t)pb.Np * ldF * 2, st));
        CK(cudaMemsetAsync(h->hl[0][1], 0, (size_t)pb.Np * ldF * 2, st));
    }
    // ---- a1: bounds, a2: initial affine layer + first split + first control step
    if (o->auto_bounds) CK(launch_gershgorin(H_dev, N, ldh, h->gpart, h->diag, h->ctrl, h->num_sms, st));
    if (pb.exact_diag) {
        CK(cudaMemsetAsync(h->rowsq[0], 0, (size_t)pb.Np * sizeof(unsigned long long), st));
        CK(cudaMemsetAsync(h->rowsq[1], 0, (size_t)pb.Np * sizeof(unsigned long long), st));
    }
    CK(launch_affine_split(H_dev, N, ldh, h->S, h->hl[0][0], h->hl[0][1], (long long)ldS, (long long)ldF, pb.scale, h->ctrl, h->stats_dev,
                           h->thetas_dev, pb.exact_diag ? h->rowsq[0] : nullptr, pb.mix ? h->mix : nullptr, (float)c0,
                           pb.sparse ? h->bn[0] : nullptr, nb, h->num_sms, st));
    // ---- a4-a8: the layer loop
    if (o->control == 0) {
        LoopGraph* lg = nullptr;
        s = get_loop_graph(h, pb, &lg);
        if (s != SP2_OK) return s;
        CK(cudaGraphLaunch(lg->exec, st));
    } else if (o->control == 1) {
        for (int n = 0; n < max_layers; ++n) {
            CK(cudaMemcpyAsync(&h->ctrl_host->running, &h->ctrl->running, sizeof(int), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            if (!h->ctrl_host->running) break;
            s = launch_one_layer(h, pb, n & 1, 0, st);
            if (s != SP2_OK) return s;
        }
    } else if (o->control == 3) {
        s = launch_one_layer(h, pb, 0, 0, st, 1);       // persistent: the layer loop runs inside one cooperative launch
        if (s != SP2_OK) return s;
    } else {
        for (int n = 0; n < max_layers; ++n) {
            s = launch_one_layer(h, pb, n & 1, 0, st);
            if (s != SP2_OK) return s;
        }
    }
    // ---- results
    if (pb.mix)      // F = d I - M  (Eq. 18 in the library's variables, see generalized_impl)
        CK(launch_one_minus(h->mix, (long long)ldS, D_dev, ldd, N, (float)mix_diag, h->num_sms, st));
    else
        CK(launch_copy_sym(h->S, (long long)ldS, D_dev, ldd, N, h->num_sms, st));
    CK(cudaMemcpyAsync(h->ctrl_host, h->ctrl, ctrl_header_bytes(), cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(h->stats_host, h->stats_dev, (size_t)max_layers * sizeof(sp2_layer_stat_t),
                       cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    c = h->ctrl_host;
    h->last_launches = c->launches + 1;      // + the copy-out kernel (k_copy_sym / k_one_minus)
    h->sparse_work[0] = (double)c->work_active; h->sparse_work[1] = (double)c->work_dense;
    if (bounds_out) { bounds_out[0] = c->eps_min; bounds_out[1] = c->eps_max; }
    if (n_layers_out) *n_layers_out = c->n;
    if (stats_out) {
        const int ns = c->n < max_layers ? c->n : max_layers;
        memcpy(stats_out, h->stats_host, (size_t)ns * sizeof(sp2_layer_stat_t));
        stats_to_double(stats_out, ns);
    }
    if (c->error < 0) return (sp2_status_t)c->error;
    if (c->running) return SP2_ERR_CUDA;     // loop ended while the device still wanted layers: should not happen
    if (mode == MODE_STANDARD && c->stop_reason == SP2_STOP_MAX_LAYERS) return SP2_NOT_CONVERGED;
    return SP2_OK;
}

static sp2_status_t resident_solve(sp2_handle_s* h, const float* H_dev, int N, int B, const double* N_occ,
                                   int nocc_is_scalar, const sp2_opts_t& o, float* D_dev, sp2_layer_stat_t* stats_host,
                                   int* n_layers, int* status_out, double* bounds_out, cudaStream_t st, int mode,
                                   const double* homo_lumo);

extern "C" sp2_status_t sp2_density_matrix(sp2_handle_t h, const float* H_dev, int N, int ldh, double N_occ,
                                           const sp2_opts_t* opts, float* D_dev, int ldd,
                                           sp2_layer_stat_t* stats_host, int* n_layers, double bounds_out[2],
                                           void* stream) {
    sp2_status_t s = check_common(h, H_dev, N, ldh, D_dev, ldd);
    if (s != SP2_OK) return s;
    sp2_opts_t o;
    if (opts) o = *opts; else sp2_default_opts(&o);
    if (!(N_occ >= 0.0 && N_occ <= (double)N)) return SP2_ERR_INVALID_ARG;
    if (o.max_layers < 1 || o.max_layers > h->max_layers) return SP2_ERR_INVALID_ARG;
    if (!o.auto_bounds) {
        if (!isfinite(o.eps_min) || !isfinite(o.eps_max)) return SP2_ERR_INVALID_ARG;
        if (!(o.eps_max > o.eps_min)) return SP2_ERR_BOUNDS_DEGENERATE;
    }
    if (o.accelerated) {
        if (!isfinite(o.homo) || !isfinite(o.lumo) || !(o.lumo > o.homo)) return SP2_ERR_INVALID_ARG;
        if (!o.auto_bounds && !(o.eps_min <= o.homo && o.lumo <= o.eps_max)) return SP2_ERR_INVALID_ARG;
    }
    if (N <= 256 && o.tile_config == TILE_AUTO && o.control == 0 && !o.accelerated && !(o.trunc_tau > 0.0) && ldh == N &&
        ldd == N) {
        // small N: the whole solve in ONE launch of the resident kernel (matrix on chip across all layers) instead of
        // one kernel per layer.  (exact_diag does not apply there: the diagonal comes from the tensor core.)
        int nl = 0;
        sp2_status_t s2 = resident_solve(h, H_dev, N, 1, &N_occ, 1, o, D_dev, stats_host, &nl, nullptr, bounds_out,
                                         (cudaStream_t)stream, MODE_STANDARD, nullptr);
        if (n_layers) *n_layers = nl;
        return s2;
    }
    return solve_single(h, H_dev, N, ldh, N_occ, MODE_STANDARD, &o, D_dev, ldd, stats_host, n_layers, bounds_out,
                        (cudaStream_t)stream);
}

extern "C" sp2_status_t sp2_density_matrix_host(sp2_handle_t h, const float* H_host, int N, int ldh, double N_occ,
                                                const sp2_opts_t* opts, float* D_host, int ldd,
                                                sp2_layer_stat_t* stats_host, int* n_layers, double bounds_out[2],
                                                void* stream) {
    sp2_status_t s = check_common(h, H_host, N, ldh, D_host, ldd);
    if (s != SP2_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t elems = (size_t)N * N;
    if (h->stage_elems < elems) {
        cudaFree(h->stage_H); cudaFree(h->stage_D);
        h->stage_H = h->stage_D = nullptr; h->stage_elems = 0;
        CK(cudaMalloc((void**)&h->stage_H, elems * 4));
        CK(cudaMalloc((void**)&h->stage_D, elems * 4));
        h->stage_elems = elems;
    }
    for (int i = 0; i < 4; ++i)
        if (!h->host_ev[i]) CK(cudaEventCreate(&h->host_ev[i]));
    CK(cudaEventRecord(h->host_ev[0], st));
    // Only the LOWER triangle of H is ever read (header, "Conventions"), so only it crosses the bus: row bands of
    // kHostBand rows, each copied up to its last row's diagonal element.  Band edges are multiples of the 64 x 64 tiles the
    // HBM kernels walk, so every element of a tile they touch has been written; the staging matrix above the bands keeps
    // whatever it held and is never read.  Halves the host -> device time at large N (16384: 1 GiB -> 0.51 GiB).
    constexpr int kHostBand = 256;
    double h2d_bytes = 0.0;
    if (N <= 4 * kHostBand) {
        CK(cudaMemcpy2DAsync(h->stage_H, (size_t)N * 4, H_host, (size_t)ldh * 4, (size_t)N * 4, (size_t)N,
                             cudaMemcpyHostToDevice, st));
        h2d_bytes = (double)elems * 4.0;
    } else {
        for (int r0 = 0; r0 < N; r0 += kHostBand) {
            const int r1 = r0 + kHostBand < N ? r0 + kHostBand : N;
            CK(cudaMemcpy2DAsync(h->stage_H + (size_t)r0 * N, (size_t)N * 4, H_host + (size_t)r0 * ldh, (size_t)ldh * 4,
                                 (size_t)r1 * 4, (size_t)(r1 - r0), cudaMemcpyHostToDevice, st));
            h2d_bytes += (double)r1 * 4.0 * (double)(r1 - r0);
        }
    }
    h->host_bytes[0] = h2d_bytes; h->host_bytes[1] = (double)elems * 4.0;
    CK(cudaEventRecord(h->host_ev[1], st));
    s = sp2_density_matrix(h, h->stage_H, N, N, N_occ, opts, h->stage_D, N, stats_host, n_layers, bounds_out, stream);
    if (s < 0) return s;
    CK(cudaEventRecord(h->host_ev[2], st));
    CK(cudaMemcpy2DAsync(D_host, (size_t)ldd * 4, h->stage_D, (size_t)N * 4, (size_t)N * 4, (size_t)N,
                         cudaMemcpyDeviceToHost, st));
    CK(cudaEventRecord(h->host_ev[3], st));
    CK(cudaStreamSynchronize(st));
    for (int i = 0; i < 3; ++i) CK(cudaEventElapsedTime(&h->host_ms[i], h->host_ev[i], h->host_ev[i + 1]));
    return s;
}

// NEXT-1: final refinement f_final (Eq. 16) as two layers with enhanced accumulation, plus Tr[D H].
extern "C" sp2_status_t sp2_refine_energy(sp2_handle_t h, const float* S_dev, int N, int lds, int last_sigma,
                                          const float* H_dev, int ldh, const sp2_opts_t* opts, float* D_dev, int ldd,
                                          sp2_refine_result_t* result, void* stream) {
    sp2_status_t s = check_common(h, S_dev, N, lds, D_dev, ldd);
    if (s != SP2_OK) return s;
    if (!H_dev || ldh < N || !result || (last_sigma != 1 && last_sigma != -1)) return SP2_ERR_INVALID_ARG;
    if (h->max_layers < 2) return SP2_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    Problem pb;
    sp2_opts_t ro;
    sp2_default_opts(&ro);
    if (opts) { ro.fp16_scale_log2 = opts->fp16_scale_log2; ro.enh_kc = opts->enh_kc; }
    s = prepare_problem(h, N, &ro, &pb, st, TILE_128x128_ENH);
    if (s != SP2_OK) return s;
    pb.exact_diag = 1;                               // diag(X) from row sums of squares (reading C24), as in the solve
    // Reading C15: continue the alternation from the last applied sign.
    //   last sigma = -1: X = S^2, then 2X - X^2  ->  2 S^2 - S^4 ;   last sigma = +1: T = 2S - S^2, then T^2.
    float* th = h->thetas_host;
    memset(th, 0, 2 * kThetaStride * sizeof(float));
    if (last_sigma < 0) { th[0] = 1; th[kThetaStride] = -1; th[kThetaStride + 1] = 2; }
    else                { th[0] = -1; th[1] = 2; th[kThetaStride] = 1; }
    Ctrl* c = h->ctrl_host;
    memset(c, 0, ctrl_header_bytes());
    c->N = N; c->mode = MODE_GENERALIZED; c->max_layers = 2;
    CK(cudaMemcpyAsync(h->ctrl, c, ctrl_header_bytes(), cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(h->thetas_dev, th, 2 * kThetaStride * sizeof(float), cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(h->stats_dev, 0, 2 * sizeof(sp2_layer_stat_t), st));
    const size_t ldS = (size_t)ws_ld_f32(pb.Np), ldF = (size_t)ws_ld_f16(pb.Np);
    if (pb.Np != N) CK(cudaMemsetAsync(h->S, 0, (size_t)pb.Np * ldS * 4, st));
    CK(cudaMemcpy2DAsync(h->S, ldS * 4, S_dev, (size_t)lds * 4, (size_t)N * 4, (size_t)N, cudaMemcpyDeviceToDevice, st));
    // observables of the input, and the plan of layer 1 (thetas[0])
    CK(cudaMemsetAsync(h->rowsq[0], 0, (size_t)pb.Np * sizeof(unsigned long long), st));
    CK(cudaMemsetAsync(h->rowsq[1], 0, (size_t)pb.Np * sizeof(unsigned long long), st));
    CK(launch_energy_traces(h->S, (long long)ldS, H_dev, ldh, N, h->ctrl, h->obs_dev, 1, h->stats_dev, h->thetas_dev,
                            h->rowsq[0], h->num_sms, st));
    CK(launch_split(h->S, pb.Np, (long long)ldS, h->hl[0][0], h->hl[0][1], (long long)ldF, pb.scale, h->num_sms, st));
    s = launch_one_layer(h, pb, 0, 0, st);
    if (s == SP2_OK) s = launch_one_layer(h, pb, 1, 0, st);
    if (s != SP2_OK) return s;
    CK(launch_copy_sym(h->S, (long long)ldS, D_dev, ldd, N, h->num_sms, st));
    CK(launch_energy_traces(D_dev, ldd, H_dev, ldh, N, h->ctrl, h->obs_dev + 3, 0, nullptr, nullptr, nullptr,
                            h->num_sms, st));
    CK(cudaMemcpyAsync(h->obs_host, h->obs_dev, 6 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(h->ctrl_host, h->ctrl, ctrl_header_bytes(), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    const double* o = h->obs_host;
    result->energy_in = o[0]; result->trace_in = o[1]; result->iderr_in = o[1] - o[2];
    result->energy_out = o[3]; result->trace_out = o[4]; result->iderr_out = o[4] - o[5];
    h->last_launches = h->ctrl_host->launches + 2;   // device-counted: 2 layers + 2 k_energy_traces; + split, copy-out
    if (h->ctrl_host->error < 0) return (sp2_status_t)h->ctrl_host->error;
    if (h->ctrl_host->n != 2) return SP2_ERR_CUDA;
    if (!isfinite(o[3]) || !isfinite(o[4]) || !isfinite(o[5])) return SP2_ERR_NONFINITE;
    return SP2_OK;
}

// Shared body of sp2_generalized / sp2_generalized_mix: c_host == nullptr -> output X_L = S_L, else F = I - sum c_i S_i.
static sp2_status_t generalized_impl(sp2_handle_t h, const float* H_dev, int N, int ldh, const double* theta_host,
                                     const double* c_host, int L, double eps_min, double eps_max,
                                     const sp2_opts_t* opts, float* out_dev, int ldo, sp2_layer_stat_t* stats_host,
                                     void* stream) {
    sp2_status_t s = check_common(h, H_dev, N, ldh, out_dev, ldo);
    if (s != SP2_OK) return s;
    if (!theta_host || L < 1 || L > h->max_layers) return SP2_ERR_INVALID_ARG;
    sp2_opts_t o;
    if (opts) o = *opts; else sp2_default_opts(&o);
    o.max_layers = L;
    o.tol = 0.0;
    o.eps_alt = 0.0;
    o.auto_bounds = !(eps_max > eps_min);
    o.eps_min = eps_min; o.eps_max = eps_max;
    if (!o.auto_bounds && (!isfinite(eps_min) || !isfinite(eps_max))) return SP2_ERR_INVALID_ARG;
    for (int n = 0; n < L; ++n) {
        for (int k = 0; k < 3; ++k) {
            if (!isfinite(theta_host[3 * n + k])) return SP2_ERR_INVALID_ARG;
            h->thetas_host[kThetaStride * n + k] = (float)theta_host[3 * n + k];
        }
        const double cn = c_host ? c_host[n + 1] : 0.0;      // weight of the output of layer n+1
        if (!isfinite(cn)) return SP2_ERR_INVALID_ARG;
        h->thetas_host[kThetaStride * n + 3] = (float)cn;
    }
    double c0 = 0.0, diag_const = 1.0;
    if (c_host) {
        if (!isfinite(c_host[0])) return SP2_ERR_INVALID_ARG;
        // Eq. 17 starts from eps_0 = the rescaled H in NATURAL order (reading C26), the library's S_0 is the
        // reversed one (Alg. 1): eps_0 = I - S_0.  Substituting into layer 1 and into the sum (exact algebra):
        //   eps_1 = th1 S_0^2 - (2 th1 + th2) S_0 + (th1 + th2 + th3) I
        //   F~ = I - sum c_i eps_i = (1 - c_0) I - [ (-c_0) S_0 + sum_{i>=1} c_i eps_i ]
        const double t1 = theta_host[0], t2 = theta_host[1], t3 = theta_host[2];
        h->thetas_host[0] = (float)t1;
        h->thetas_host[1] = (float)(-(2.0 * t1 + t2));
        h->thetas_host[2] = (float)(t1 + t2 + t3);
        c0 = -c_host[0];
        diag_const = 1.0 - c_host[0];
    }
    int nl = 0;
    return solve_single(h, H_dev, N, ldh, 0.0, MODE_GENERALIZED, &o, out_dev, ldo, stats_host, &nl, nullptr,
                        (cudaStream_t)stream, c_host != nullptr, c0, diag_const);
}

extern "C" sp2_status_t sp2_generalized(sp2_handle_t h, const float* H_dev, int N, int ldh, const double* theta_host,
                                        int L, double eps_min, double eps_max, const sp2_opts_t* opts, float* X_L_dev,
                                        int ldx, sp2_layer_stat_t* stats_host, void* stream) {
    return generalized_impl(h, H_dev, N, ldh, theta_host, nullptr, L, eps_min, eps_max, opts, X_L_dev, ldx, stats_host,
                            stream);
}

// NEXT-2: the optimised finite-temperature expansion F~(H) = I - sum_{i=0..L} c_i S_i (Eqs. 17-18).
extern "C" sp2_status_t sp2_generalized_mix(sp2_handle_t h, const float* H_dev, int N, int ldh,
                                            const double* theta_host, const double* c_host, int L, double eps_min,
                                            double eps_max, const sp2_opts_t* opts, float* F_dev, int ldf,
                                            sp2_layer_stat_t* stats_host, void* stream) {
    if (!c_host) return SP2_ERR_INVALID_ARG;
    return generalized_impl(h, H_dev, N, ldh, theta_host, c_host, L, eps_min, eps_max, opts, F_dev, ldf, stats_host,
                            stream);
}

extern "C" sp2_status_t sp2_generalized_wb(sp2_handle_t h, const float* H_dev, int N, int ldh, const int* sigma,
                                           const double* weights, const double* biases, int L, double eps_min,
                                           double eps_max, const sp2_opts_t* opts, float* X_L_dev, int ldx,
                                           sp2_layer_stat_t* stats_host, void* stream) {
    if (!h || !weights || !biases || L < 1 || L > h->max_layers) return SP2_ERR_INVALID_ARG;
    std::vector<double> th((size_t)3 * L);
    for (int n = 0; n < L; ++n) {
        const int sg = sigma ? sigma[n] : 1;
        if (sg != 1 && sg != -1) return SP2_ERR_INVALID_ARG;
        th[3 * n + 0] = weights[n] * sg;           // theta_1 = w sigma
        th[3 * n + 1] = weights[n] * (1 - sg);     // theta_2 = w (1 - sigma)
        th[3 * n + 2] = biases[n];                 // theta_3 = b
    }
    return sp2_generalized(h, H_dev, N, ldh, th.data(), L, eps_min, eps_max, opts, X_L_dev, ldx, stats_host, stream);
}

// Shared body of the batched calls and of small single matrices: B contiguous N x N problems, one resident-kernel
// launch.  mode = MODE_STANDARD (Alg. 1, optionally with the accelerated weights and per-matrix estimates
// homo_lumo[B][2]) or MODE_GENERALIZED (L = o.max_layers layers with the thetas already in h->thetas_host).
static sp2_status_t resident_solve(sp2_handle_s* h, const float* H_dev, int N, int B, const double* N_occ,
                                   int nocc_is_scalar, const sp2_opts_t& o, float* D_dev, sp2_layer_stat_t* stats_host,
                                   int* n_layers, int* status_out, double* bounds_out /*[B][2] or NULL*/,
                                   cudaStream_t st, int mode, const double* homo_lumo) {
    int k = o.fp16_scale_log2;
    if (k < 0) k = 13;
    if (k > 14) return SP2_ERR_INVALID_ARG;
    if (N_occ) {
        const int nn = nocc_is_scalar ? 1 : B;
        for (int i = 0; i < nn; ++i) h->bnocc_host[i] = to_fx(N_occ[i]);
        CK(cudaMemcpyAsync(h->bnocc_dev, h->bnocc_host, (size_t)nn * sizeof(long long), cudaMemcpyHostToDevice, st));
    }
    if (homo_lumo) CK(cudaMemcpyAsync(h->bhl_dev, homo_lumo, (size_t)B * 2 * sizeof(double), cudaMemcpyHostToDevice, st));
    if (mode == MODE_GENERALIZED)
        CK(cudaMemcpyAsync(h->thetas_dev, h->thetas_host, (size_t)o.max_layers * kThetaStride * sizeof(float),
                           cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(h->bstats_dev, 0, (size_t)B * o.max_layers * sizeof(sp2_layer_stat_t), st));
    ResidentParams p;
    memset(&p, 0, sizeof(p));
    p.H = H_dev; p.D = D_dev; p.N_occ = h->bnocc_dev; p.nocc_is_scalar = nocc_is_scalar; p.N = N; p.B = B;
    p.auto_bounds = o.auto_bounds; p.eps_min = o.eps_min; p.eps_max = o.eps_max;
    p.tol = (o.tol > 0.0) ? (to_fx(o.tol) > 0 ? to_fx(o.tol) : 1) : 0; p.eps_alt = to_fx(o.eps_alt);
    p.max_layers = o.max_layers; p.mode = mode; p.thetas = (mode == MODE_GENERALIZED) ? h->thetas_dev : nullptr;
    p.kappa_q16 = opt_kappa_q16(o);
    p.accelerated = (mode == MODE_STANDARD && homo_lumo) ? 1 : 0;
    p.homo_lumo = h->bhl_dev;
    p.scale = ldexpf(1.0f, k); p.inv_scale2 = ldexpf(1.0f, -2 * k);
    p.stats = h->bstats_dev; p.n_layers = h->bnl_dev; p.status = h->bstatus_dev; p.bounds = h->bbounds_dev;
    CK(launch_resident(p, h->num_sms, st));
    int* nl = h->bnl_host;
    int* stt = h->bnl_host + B;
    CK(cudaMemcpyAsync(nl, h->bnl_dev, (size_t)B * sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(stt, h->bstatus_dev, (size_t)B * sizeof(int), cudaMemcpyDeviceToHost, st));
    if (stats_host)
        CK(cudaMemcpyAsync(h->bstats_host, h->bstats_dev, (size_t)B * o.max_layers * sizeof(sp2_layer_stat_t),
                           cudaMemcpyDeviceToHost, st));
    if (bounds_out)
        CK(cudaMemcpyAsync(h->bbounds_host, h->bbounds_dev, (size_t)B * 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    CK(cudaGetLastError());
    if (bounds_out) memcpy(bounds_out, h->bbounds_host, (size_t)B * 2 * sizeof(double));
    if (stats_host)          // only the layers that ran (the caller's buffer beyond them is left untouched)
        for (int i = 0; i < B; ++i) {
            const int n = nl[i] < o.max_layers ? nl[i] : o.max_layers;
            if (n > 0) {
                memcpy(stats_host + (size_t)i * o.max_layers, h->bstats_host + (size_t)i * o.max_layers,
                       (size_t)n * sizeof(sp2_layer_stat_t));
                stats_to_double(stats_host + (size_t)i * o.max_layers, n);
            }
        }
    h->last_launches = 1;
    h->sparse_work[0] = h->sparse_work[1] = 0.0;             // the diagnostics of the single-matrix layer kernel do not
    if (h->ctrl_host) h->ctrl_host->round_sync_broken = 0;   // apply here: report "dense" / "not broken", not the last solve's
    int worst = SP2_OK;
    for (int i = 0; i < B; ++i) {
        if (n_layers) n_layers[i] = nl[i];
        if (status_out) status_out[i] = stt[i];
        if (stt[i] < 0) { if (worst >= 0 || stt[i] < worst) worst = stt[i]; }
        else if (stt[i] > worst && worst >= 0) worst = stt[i];
    }
    return (sp2_status_t)worst;
}

extern "C" sp2_status_t sp2_density_matrix_batched(sp2_handle_t h, const float* H_dev, int N, int B,
                                                   const double* N_occ, int nocc_is_scalar, const double* homo_lumo,
                                                   const sp2_opts_t* opts, float* D_dev, sp2_layer_stat_t* stats_host,
                                                   int* n_layers, int* status_out, void* stream) {
    if (!h || !H_dev || !D_dev || !N_occ || N < 1 || B < 1) return SP2_ERR_INVALID_ARG;
    if (N > 256) return SP2_ERR_UNSUPPORTED_N;
    if (B > h->batch_max) return SP2_ERR_WORKSPACE;
    sp2_status_t sd = check_device(h);
    if (sd != SP2_OK) return sd;
    sp2_opts_t o;
    if (opts) o = *opts; else sp2_default_opts(&o);
    if (o.max_layers < 1 || o.max_layers > h->max_layers) return SP2_ERR_INVALID_ARG;
    if (!o.auto_bounds) {
        if (!isfinite(o.eps_min) || !isfinite(o.eps_max)) return SP2_ERR_INVALID_ARG;
        if (!(o.eps_max > o.eps_min)) return SP2_ERR_BOUNDS_DEGENERATE;
    }
    // accelerated weights (section V.A): per-matrix estimates through homo_lumo[B][2]; opts->homo / lumo are not read
    if ((o.accelerated != 0) != (homo_lumo != nullptr)) return SP2_ERR_INVALID_ARG;
    if (homo_lumo)
        for (int i = 0; i < B; ++i) {
            const double ho = homo_lumo[2 * i], lu = homo_lumo[2 * i + 1];
            if (!isfinite(ho) || !isfinite(lu) || !(lu > ho)) return SP2_ERR_INVALID_ARG;
            if (!o.auto_bounds && !(o.eps_min <= ho && lu <= o.eps_max)) return SP2_ERR_INVALID_ARG;
        }
    for (int i = 0; i < (nocc_is_scalar ? 1 : B); ++i)
        if (!(N_occ[i] >= 0.0 && N_occ[i] <= (double)N)) return SP2_ERR_INVALID_ARG;
    return resident_solve(h, H_dev, N, B, N_occ, nocc_is_scalar, o, D_dev, stats_host, n_layers, status_out, nullptr,
                          (cudaStream_t)stream, MODE_STANDARD, homo_lumo);
}

// The generalized network (Eq. 17) on a batch: the same L layers (shared weights) applied to B inputs.
extern "C" sp2_status_t sp2_generalized_batched(sp2_handle_t h, const float* H_dev, int N, int B,
                                                const double* theta_host, int L, double eps_min, double eps_max,
                                                const sp2_opts_t* opts, float* X_L_dev, sp2_layer_stat_t* stats_host,
                                                int* status_out, void* stream) {
    if (!h || !H_dev || !X_L_dev || !theta_host || N < 1 || B < 1 || L < 1) return SP2_ERR_INVALID_ARG;
    if (N > 256) return SP2_ERR_UNSUPPORTED_N;
    if (B > h->batch_max) return SP2_ERR_WORKSPACE;
    if (L > h->max_layers) return SP2_ERR_INVALID_ARG;
    sp2_status_t sd = check_device(h);
    if (sd != SP2_OK) return sd;
    sp2_opts_t o;
    if (opts) o = *opts; else sp2_default_opts(&o);
    o.max_layers = L; o.tol = 0.0; o.eps_alt = 0.0;
    o.auto_bounds = !(eps_max > eps_min);
    o.eps_min = eps_min; o.eps_max = eps_max;
    if (!o.auto_bounds && (!isfinite(eps_min) || !isfinite(eps_max))) return SP2_ERR_INVALID_ARG;
    for (int n = 0; n < L; ++n) {
        for (int k = 0; k < 3; ++k) {
            if (!isfinite(theta_host[3 * n + k])) return SP2_ERR_INVALID_ARG;
            h->thetas_host[kThetaStride * n + k] = (float)theta_host[3 * n + k];
        }
        h->thetas_host[kThetaStride * n + 3] = 0.0f;
    }
    std::vector<int> nl((size_t)B);
    return resident_solve(h, H_dev, N, B, nullptr, 1, o, X_L_dev, stats_host, nl.data(), status_out, nullptr,
                          (cudaStream_t)stream, MODE_GENERALIZED, nullptr);
}

extern "C" sp2_status_t sp2_split_fp16(const float* X_dev, int N, int ldx, unsigned short* hi_dev,
                                       unsigned short* lo_dev, int ldo, int fp16_scale_log2, void* stream) {
    if (!X_dev || !hi_dev || !lo_dev || N < 1 || ldx < N || ldo < N) return SP2_ERR_INVALID_ARG;
    if (fp16_scale_log2 < 0 || fp16_scale_log2 > 14) return SP2_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CK(launch_split(X_dev, N, ldx, (__half*)hi_dev, (__half*)lo_dev, ldo, ldexpf(1.0f, fp16_scale_log2), sms,
                    (cudaStream_t)stream));
    return SP2_OK;
}

extern "C" sp2_status_t sp2_gershgorin(sp2_handle_t h, const float* H_dev, int N, int ldh, double bounds_host[2],
                                       void* stream) {
    if (!h || !H_dev || !bounds_host || N < 1 || ldh < N) return SP2_ERR_INVALID_ARG;
    if (N > h->N_max) return SP2_ERR_WORKSPACE;
    sp2_status_t sd = check_device(h);
    if (sd != SP2_OK) return sd;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaMemsetAsync(&h->ctrl->done_counter, 0, sizeof(unsigned int), st));
    CK(launch_gershgorin(H_dev, N, ldh, h->gpart, h->diag, h->ctrl, h->num_sms, st));
    CK(cudaMemcpyAsync(h->bounds_host, &h->ctrl->eps_min, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    bounds_host[0] = h->bounds_host[0];
    bounds_host[1] = h->bounds_host[1];
    return SP2_OK;
}

extern "C" int sp2_last_launch_count(sp2_handle_t h) { return h ? h->last_launches : 0; }
extern "C" void sp2_last_host_timing(sp2_handle_t h, double ms[3]) {
    if (!h || !ms) return;
    for (int i = 0; i < 3; ++i) ms[i] = (double)h->host_ms[i];
}
extern "C" void sp2_last_host_bytes(sp2_handle_t h, double out[2]) {
    if (!h || !out) return;
    out[0] = h->host_bytes[0]; out[1] = h->host_bytes[1];
}
extern "C" void sp2_last_sparse_work(sp2_handle_t h, double out[2]) {
    if (!h || !out) return;
    out[0] = h->sparse_work[0]; out[1] = h->sparse_work[1];
}
extern "C" int sp2_last_round_sync_broken(sp2_handle_t h) { return (h && h->ctrl_host) ? (int)h->ctrl_host->round_sync_broken : 0; }
