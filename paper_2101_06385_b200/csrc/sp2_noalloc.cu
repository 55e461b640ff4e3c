// sp2_gershgorin_static: the Gershgorin bounds (row a1 of DESIGN.md; Alg. 1's "spectral bound estimates") for
// callers that are not allowed to allocate device memory.
//
// Who that is.  The ordinary call, sp2_gershgorin, needs a handle, and sp2_create calls cudaMalloc.  Some hosts cannot
// afford that: a molecular-dynamics code (or a framework's caching allocator) that has already taken the whole of HBM
// into its own arena, so that a cudaMalloc coming from a library fails with "out of memory" although memory is free
// inside the arena; a time-step loop that cannot accept the device-wide synchronisation a cudaMalloc / cudaFree
// implies; a plug-in that is only handed pointers and a stream and has no say over the memory budget.  For them the
// scratch the two Gershgorin kernels need (per-tile row / column sums, the diagonal, per-block extrema) lives in a
// static __device__ array below: it is part of the library image, every GPU that loads libsp2b200.so holds these
// kStaticBytes (about 2.2 MB) until the process exits, and the entry point calls no cudaMalloc, cudaFree or any other
// allocating routine.  The price is the size limit SP2_GERSHGORIN_STATIC_MAX_N.
//
// The kernels are the ones sp2_gershgorin launches (k_gershgorin_rows / k_gershgorin_finalize in sp2_elementwise.cu),
// given addresses inside the static array instead of addresses inside a handle's workspace, so the bounds are the same
// bits.
#include <stdio.h>

#include <mutex>

#include "sp2_kernels.h"

using namespace sp2;

namespace {

constexpr int kStaticMaxN = 4096;                       // == SP2_GERSHGORIN_STATIC_MAX_N (checked below)
static_assert(kStaticMaxN == SP2_GERSHGORIN_STATIC_MAX_N, "header and source disagree on the size limit");
constexpr size_t round256(size_t b) { return (b + 255) / 256 * 256; }
// layout of the static scratch: [ Ctrl | diag: kStaticMaxN doubles | part: 2 * ceil(N / 64) * N floats ]
constexpr size_t kOffCtrl = 0;
constexpr size_t kOffDiag = round256(sizeof(Ctrl));
constexpr size_t kOffPart = kOffDiag + round256((size_t)kStaticMaxN * sizeof(double));
constexpr size_t kPartFloats = 2 * (size_t)((kStaticMaxN + 63) / 64) * (size_t)kStaticMaxN;
constexpr size_t kStaticBytes = kOffPart + round256(kPartFloats * sizeof(float));

// The scratch itself.  In host code this name is only a stand-in the runtime uses to look the symbol up; it is NOT a
// device address and must never be handed to a kernel.  The address each device holds it at comes from
// cudaGetSymbolAddress (device_scratch below).
static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

constexpr int kMaxDevices = 64;
struct PerDevice {
    unsigned char* base = nullptr;   // device address of g_static_scratch on this device
    int num_sms = 0;
};
PerDevice g_dev[kMaxDevices];
std::mutex g_dev_mutex;

thread_local char g_static_err[256] = "";

// Set-up, once per device, with that device current: ask the runtime where this device keeps the array.
cudaError_t device_scratch(int dev, PerDevice* out) {
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    PerDevice& d = g_dev[dev];
    if (d.base == nullptr) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        d.num_sms = sms;
        d.base = static_cast<unsigned char*>(p);
    }
    *out = d;
    return cudaSuccess;
}

sp2_status_t fail(sp2_status_t s, const char* fmt, long long a = 0, long long b = 0) {
    snprintf(g_static_err, sizeof(g_static_err), fmt, a, b);
    return s;
}

sp2_status_t cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_static_err, sizeof(g_static_err), "sp2_gershgorin_static: %s: %s", what, cudaGetErrorString(e));
    return SP2_ERR_CUDA;
}

}  // namespace

extern "C" int sp2_gershgorin_static_max_n(void) { return kStaticMaxN; }
extern "C" size_t sp2_gershgorin_static_bytes(void) { return kStaticBytes; }
extern "C" const char* sp2_gershgorin_static_last_error(void) { return g_static_err; }

extern "C" sp2_status_t sp2_gershgorin_static(const float* H_dev, int N, int ldh, double* bounds_dev, void* stream) {
    g_static_err[0] = 0;
    if (!H_dev || !bounds_dev) return fail(SP2_ERR_INVALID_ARG, "sp2_gershgorin_static: null pointer");
    if (N < 1 || ldh < N) return fail(SP2_ERR_INVALID_ARG, "sp2_gershgorin_static: need 1 <= N <= ldh (N = %lld, ldh = %lld)", N, ldh);
    if (N > kStaticMaxN)
        return fail(SP2_ERR_UNSUPPORTED_N,
                    "sp2_gershgorin_static: N = %lld exceeds the static scratch (N <= %lld); use sp2_gershgorin with a handle",
                    N, kStaticMaxN);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices) return fail(SP2_ERR_INVALID_ARG, "sp2_gershgorin_static: device %lld out of range", dev);
    PerDevice d;
    e = device_scratch(dev, &d);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(static scratch)");

    Ctrl* ctrl = reinterpret_cast<Ctrl*>(d.base + kOffCtrl);
    double* diag = reinterpret_cast<double*>(d.base + kOffDiag);
    float* part = reinterpret_cast<float*>(d.base + kOffPart);
    cudaStream_t st = (cudaStream_t)stream;
    // The array keeps whatever the previous call left.  Every part / diag slot the finalize kernel reads is rewritten by
    // the row kernel of THIS call; the one word that has to start at zero is the block counter.
    e = cudaMemsetAsync(&ctrl->done_counter, 0, sizeof(unsigned int), st);
    if (e == cudaSuccess) e = launch_gershgorin(H_dev, N, ldh, part, diag, ctrl, d.num_sms, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(bounds_dev, &ctrl->eps_min, 2 * sizeof(double), cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e, "enqueue");
    return SP2_OK;
}
