// fn_peaks.cu -- roofline denominators measured in the same binary and run:
//   kind 0: shared memory, conflict-free 16-byte loads (512 contiguous bytes per warp instruction)
//   kind 1: shared memory, pseudo-random 32-bit word per lane (bank conflicts as they fall)
//   kind 2: L2-resident global memory, coalesced ld.global.nc 8-byte reads over a 32 MB buffer
// Returns requested bytes per second (bytes = lanes x bytes per load, the same currency in which
// the beam kernel's map traffic is counted).
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/flashnav.h"

namespace {

constexpr int kIters = 2048;
constexpr int kUnroll = 8;

__global__ void __launch_bounds__(1024, 2) smem_peak_kernel(int kind, unsigned* sink) {
    extern __shared__ uint32_t s_words[];
    const int nwords = 16384;                                    // 64 KB
    for (int i = threadIdx.x; i < nwords; i += blockDim.x) s_words[i] = i * 2654435761u;
    __syncthreads();
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(s_words);
    uint32_t acc = 0;
    if (kind == 0) {
        // conflict-free: lane i of a warp reads the 16 bytes at 16*i (+ a per-warp, per-step offset),
        // i.e. 512 contiguous bytes per warp instruction = 4 full 128-byte wavefronts
        const uint32_t lane16 = base + (threadIdx.x & 31) * 16u;
        for (int it = 0; it < kIters; ++it) {
            const uint32_t a0 = lane16 + (((threadIdx.x >> 5) + it) & 7) * 4096u;   // moves every iteration
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                uint32_t x, y, z, w;
                asm volatile("ld.volatile.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(x), "=r"(y), "=r"(z), "=r"(w)
                             : "r"(a0 + u * 512u));
                acc += x ^ y ^ z ^ w;
            }
        }
    } else {
        // one pseudo-random 32-bit word per lane per load (bank conflicts as they fall)
        uint32_t idx = threadIdx.x * 40503u + 12345u;
        for (int it = 0; it < kIters; ++it) {
#pragma unroll
            for (int u = 0; u < kUnroll; ++u) {
                uint32_t x;
                asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(x) : "r"(base + ((idx >> 8) & (nwords - 1)) * 4u));
                acc += x;
                idx = idx * 1664525u + 1013904223u;
            }
        }
    }
    if (acc == 0x12345678u) *sink = acc;
}

__global__ void __launch_bounds__(1024, 2) l2_peak_kernel(const uint2* buf, size_t n, int iters, unsigned* sink) {
    uint32_t acc = 0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
            uint2 v;
            asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(buf + i));
            acc += v.x ^ v.y;
            i += stride;
            if (i >= n) i -= n;
        }
    }
    if (acc == 0x12345678u) *sink = acc;
}

}  // namespace

extern "C" int fn_measure_peak(int kind, void* stream_v, double* out) {
    if (!out || kind < 0 || kind > 2) return FN_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream_v;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return FN_ERR_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    unsigned* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(unsigned)) != cudaSuccess) return FN_ERR_OOM;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    double best = 0.0;
    int rc = FN_OK;
    if (kind <= 1) {
        const size_t smem = 65536;
        cudaFuncSetAttribute(smem_peak_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        const int grid = sms * 2;
        for (int rep = 0; rep < 5; ++rep) {
            cudaEventRecord(e0, st);
            smem_peak_kernel<<<grid, 1024, smem, st>>>(kind, sink);
            cudaEventRecord(e1, st);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = FN_ERR_CUDA; break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            const double bytes = (double)grid * 1024.0 * kIters * kUnroll * (kind == 0 ? 16.0 : 4.0);
            if (rep > 0 && bytes / (ms * 1e-3) > best) best = bytes / (ms * 1e-3);
        }
    } else {
        const size_t n = (32u << 20) / sizeof(uint2);
        uint2* buf = nullptr;
        if (cudaMalloc(&buf, n * sizeof(uint2)) != cudaSuccess) { cudaFree(sink); return FN_ERR_OOM; }
        cudaMemsetAsync(buf, 1, n * sizeof(uint2), st);
        const int grid = sms * 2, iters = 64;
        for (int rep = 0; rep < 5; ++rep) {
            cudaEventRecord(e0, st);
            l2_peak_kernel<<<grid, 1024, 0, st>>>(buf, n, iters, sink);
            cudaEventRecord(e1, st);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = FN_ERR_CUDA; break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            const double bytes = (double)grid * 1024.0 * iters * kUnroll * 8.0;
            if (rep > 0 && bytes / (ms * 1e-3) > best) best = bytes / (ms * 1e-3);
        }
        cudaFree(buf);
    }
    if (cudaGetLastError() != cudaSuccess) rc = FN_ERR_CUDA;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    *out = best;
    return rc;
}
