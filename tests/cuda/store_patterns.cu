// Store patterns of the layer epilogue (sp2_square_tiled.cu) in isolation: each warp owns 32 rows of a matrix with the
// N = 2048 operand pitch and writes 64 bytes of each row per iteration (the own-row FP16 piece of a 32 x 32 chunk), or the
// mirrored pieces row by row.  Prints "name GB_per_s" lines; built and run by tests/test_probe_hardware.py.  What it
// showed (B200, all 148 SMs): a lane that writes its own row in 16-byte stores gets 1.65 TB/s, in 32-byte st.global.v8
// 4.3 TB/s (a sector per lane either way); 64-byte row segments reach 4.5 - 4.7 TB/s however they are packaged, 128-byte
// ones 6.3 TB/s.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
__device__ __forceinline__ void st_v8(void* p, uint32_t a) {
    asm volatile("st.global.cs.v8.b32 [%0], {%1, %1, %1, %1, %1, %1, %1, %1};\n" ::"l"(p), "r"(a) : "memory");
}
__device__ __forceinline__ void st_v4(void* p, uint32_t a) {
    asm volatile("st.global.cs.v4.b32 [%0], {%1, %1, %1, %1};\n" ::"l"(p), "r"(a) : "memory");
}
// each warp owns 32 rows; per iteration it writes a 64-byte piece of each row (column block it)
template <int MODE>
__global__ void k(uint8_t* base, long long pitch, int iters) {
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    uint8_t* rows = base + (long long)warp * 32 * pitch;
    for (int it = 0; it < iters; ++it) {
        const long long col = (long long)it * 64;
        if (MODE == 0) {            // lane = row, 2 x 32 bytes
            st_v8(rows + lane * pitch + col, it); st_v8(rows + lane * pitch + col + 32, it);
        } else if (MODE == 1) {     // lane = row, 4 x 16 bytes
            for (int q = 0; q < 4; ++q) st_v4(rows + lane * pitch + col + 16 * q, it);
        } else if (MODE == 2) {     // 4 lanes per row (16 bytes each), 8 rows per instruction, 4 instructions
            for (int q = 0; q < 4; ++q) st_v4(rows + (long long)(8 * q + (lane >> 2)) * pitch + col + 16 * (lane & 3), it);
        } else if (MODE == 4) {     // mirrored FP16: one row per instruction, 2 bytes per lane (64 B), 32 rows
            for (int r = 0; r < 32; ++r) *reinterpret_cast<volatile unsigned short*>(rows + (long long)r * pitch + col + 2 * lane) = (unsigned short)it;
        } else if (MODE == 5) {     // mirrored FP32: one row per instruction, 4 bytes per lane (128 B), 16 rows = same bytes
            for (int r = 0; r < 16; ++r) *reinterpret_cast<volatile unsigned int*>(rows + (long long)r * pitch + 2 * col + 4 * lane) = it;
        } else if (MODE == 6) {     // two rows per instruction, 4 bytes per lane: lanes 0-15 row r, 16-31 row r + 1 (64 B each)
            for (int r = 0; r < 32; r += 2) *reinterpret_cast<volatile unsigned int*>(rows + (long long)(r + (lane >> 4)) * pitch + col + 4 * (lane & 15)) = it;
        } else {                    // 2 lanes per row (32 bytes each), 16 rows per instruction, 2 instructions
            for (int q = 0; q < 2; ++q) st_v8(rows + (long long)(16 * q + (lane >> 1)) * pitch + col + 32 * (lane & 1), it);
        }
    }
}
template <int MODE> float run(uint8_t* d, long long pitch, int iters) {
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    k<MODE><<<148, 256>>>(d, pitch, iters);
    cudaEventRecord(e0); k<MODE><<<148, 256>>>(d, pitch, iters); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); return ms;
}
int main() {
    const long long pitch = 4224;            // (2048 + 64) * 2 bytes: the N = 2048 operand pitch
    const int iters = 64;                    // 64 x 64 B = 4096 B of each row
    uint8_t* d; cudaMalloc(&d, (size_t)148 * 8 * 32 * pitch);
    const double bytes = 148.0 * 8 * 32 * 64 * iters;
    float t0 = run<0>(d, pitch, iters), t1 = run<1>(d, pitch, iters), t2 = run<2>(d, pitch, iters), t3 = run<3>(d, pitch, iters);
    float t4 = run<4>(d, pitch, iters), t5 = run<5>(d, pitch, iters), t6 = run<6>(d, pitch, iters);
    printf("mirrored_64B_per_instruction %.0f\nmirrored_128B_per_instruction %.0f\nmirrored_two_rows_of_64B_per_instruction %.0f\n", bytes / t4 / 1e6, bytes / t5 / 1e6, bytes / t6 / 1e6);
    printf("own_rows_16B_per_lane %.0f\nown_rows_32B_per_lane %.0f\nown_rows_4_lanes_per_row_16B %.0f\nown_rows_2_lanes_per_row_32B %.0f\n",
           bytes / t1 / 1e6, bytes / t0 / 1e6, bytes / t2 / 1e6, bytes / t3 / 1e6);
    return 0;
}
