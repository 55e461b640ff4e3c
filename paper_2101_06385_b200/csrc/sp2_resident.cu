// placeholder, replaced below
#include "sp2_kernels.h"
namespace sp2 {
cudaError_t resident_kernel_setup() { return cudaSuccess; }
size_t resident_smem_bytes(int) { return 0; }
cudaError_t launch_resident(const ResidentParams&, int, cudaStream_t) { return cudaErrorNotSupported; }
}
