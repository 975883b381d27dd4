// probe.cu -- roofline denominators measured on the device the library runs on.
//
// kind 0: dependent-free 32-bit integer adds (IADD3, ALU pipe)      kind 1: integer multiply-adds (IMAD, FMA pipe)
// kind 2: both interleaved                                          kind 3: LDS.32, conflict free
// kind 4: LDS.128, conflict free
// Each reports warp-level instructions per second over the whole chip (all SMs busy, enough warps to hide latency).
#include <cuda_runtime.h>

#include "kernels.h"

namespace spt {

constexpr int kProbeThreads = 512;
constexpr int kProbeIters = 4096;
constexpr int kIlp = 8;

__global__ void __launch_bounds__(kProbeThreads) probe_iadd(uint32_t* out, uint32_t seed) {
    uint32_t a[kIlp];
#pragma unroll
    for (int i = 0; i < kIlp; ++i) a[i] = threadIdx.x + i;
    uint32_t x = seed + threadIdx.x;
    for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
        for (int i = 0; i < kIlp; ++i) asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(x));
    }
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < kIlp; ++i) s ^= a[i];
    if (s == 0x12345678u) out[0] = s;
}

__global__ void __launch_bounds__(kProbeThreads) probe_imad(uint32_t* out, uint32_t seed) {
    uint32_t a[kIlp];
#pragma unroll
    for (int i = 0; i < kIlp; ++i) a[i] = threadIdx.x + i;
    uint32_t x = seed + threadIdx.x, y = seed | 3u;
    for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
        for (int i = 0; i < kIlp; ++i) asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a[i]) : "r"(x), "r"(y));
    }
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < kIlp; ++i) s ^= a[i];
    if (s == 0x12345678u) out[0] = s;
}

__global__ void __launch_bounds__(kProbeThreads) probe_mixed(uint32_t* out, uint32_t seed) {
    uint32_t a[kIlp], m[kIlp];
#pragma unroll
    for (int i = 0; i < kIlp; ++i) { a[i] = threadIdx.x + i; m[i] = threadIdx.x * 3 + i; }
    uint32_t x = seed + threadIdx.x, y = seed | 3u;
    for (int it = 0; it < kProbeIters / 2; ++it) {
#pragma unroll
        for (int i = 0; i < kIlp; ++i) {
            asm volatile("add.u32 %0, %0, %1;" : "+r"(a[i]) : "r"(x));
            asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(m[i]) : "r"(x), "r"(y));
        }
    }
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < kIlp; ++i) s ^= a[i] ^ m[i];
    if (s == 0x12345678u) out[0] = s;
}

template <int VEC>
__global__ void __launch_bounds__(kProbeThreads) probe_lds(uint32_t* out, uint32_t seed) {
    // 32 KB: the address moves every iteration so that no load can be merged with another
    __shared__ __align__(16) uint32_t buf[8192];
    for (int i = threadIdx.x; i < 8192; i += kProbeThreads) buf[i] = i ^ seed;
    __syncthreads();
    uint32_t acc = 0;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(buf);
    for (int it = 0; it < kProbeIters; ++it) {
        if (VEC == 1) {
            // lane-contiguous 128-byte rows (conflict free); 8 different rows per iteration
            const uint32_t a0 = sbase + ((threadIdx.x & 31) << 2) + (((threadIdx.x >> 5) + it) & 15) * 2048;
#pragma unroll
            for (int i = 0; i < kIlp; ++i) {
                uint32_t v;
                asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a0 + (uint32_t)(i * 128)) : "memory");
                acc ^= v;
            }
        } else {
            const uint32_t a0 = sbase + ((threadIdx.x & 31) << 4) + (((threadIdx.x >> 5) + it) & 7) * 4096;
#pragma unroll
            for (int i = 0; i < kIlp; ++i) {
                uint32_t v0, v1, v2, v3;
                asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v0), "=r"(v1), "=r"(v2), "=r"(v3)
                             : "r"(a0 + (uint32_t)((i & 3) * 512) + (uint32_t)((i >> 2) * 2048)) : "memory");
                acc ^= v0 ^ v1 ^ v2 ^ v3;
            }
        }
    }
    if (acc == 0x12345678u) out[0] = acc;
}

int run_probe(int kind, int reps, double* warp_instr_per_s, double* elapsed_ms) {
    if (reps < 1) reps = 1;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    uint32_t* d_out = nullptr;
    if (cudaMalloc(&d_out, 64) != cudaSuccess) return -1;
    cudaStream_t st;
    cudaEvent_t e0, e1;
    cudaStreamCreate(&st);
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = nsm * 4;  // 4 x 512 threads = 64 warps per SM (register use is tiny)
    auto launch = [&]() {
        switch (kind) {
            case 0: probe_iadd<<<blocks, kProbeThreads, 0, st>>>(d_out, 1u); break;
            case 1: probe_imad<<<blocks, kProbeThreads, 0, st>>>(d_out, 1u); break;
            case 2: probe_mixed<<<blocks, kProbeThreads, 0, st>>>(d_out, 1u); break;
            case 3: probe_lds<1><<<blocks, kProbeThreads, 0, st>>>(d_out, 1u); break;
            default: probe_lds<4><<<blocks, kProbeThreads, 0, st>>>(d_out, 1u); break;
        }
    };
    launch();  // warm-up
    cudaStreamSynchronize(st);
    cudaEventRecord(e0, st);
    for (int r = 0; r < reps; ++r) launch();
    cudaEventRecord(e1, st);
    cudaError_t err = cudaStreamSynchronize(st);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double per_thread = (double)kProbeIters * kIlp;  // counted instructions per thread per launch
    const double warps = (double)blocks * (kProbeThreads / 32);
    if (warp_instr_per_s) *warp_instr_per_s = per_thread * warps * reps / (ms * 1e-3);
    if (elapsed_ms) *elapsed_ms = ms;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaStreamDestroy(st);
    cudaFree(d_out);
    return err == cudaSuccess ? 0 : -1;
}

}  // namespace spt
