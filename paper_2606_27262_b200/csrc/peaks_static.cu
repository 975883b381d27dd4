// peaks_static.cu -- the peak filter (peaks.cu) for callers that must not allocate device memory.
//
// spt_peak_filter keeps its working memory (hash table of the candidates' S/N, two sets of live flags) in buffers it
// cudaMallocs and grows on demand.  Two kinds of caller cannot live with that:
//   * a real-time acquisition loop: cudaMalloc / cudaFree stall the whole device while they run, so one call that has to
//     grow a buffer makes every other stream of the process miss its deadline;
//   * a process whose device memory already belongs to somebody else's allocator (a framework's caching pool that has
//     taken the card, a fixed partition handed out at start-up): a library cudaMalloc there fails, or succeeds only by
//     taking memory the owner counted on.
// For them the same kernels run here on a fixed block of device memory that is part of the library image: the file-scope
// array below.  The price is a hard limit on the list length and 6.5 MiB held on every GPU that loads libspt.so, from
// the load of the module to the exit of the process, whether or not the call is ever made.
//
// The array's NAME is only meaningful to device code.  In host code it is a host-side handle, not a device address:
// handing it to a kernel would make the kernel fault (or, where the GPU can reach host memory, scribble over the wrong
// memory).  Host code therefore asks the runtime for the device address -- cudaGetSymbolAddress, once per device, with
// that device current -- and passes the address it got to the kernels.
#include <cuda_runtime.h>

#include <mutex>

#include "kernels.h"

namespace spt {

// layout of the block: hash keys | hash values | live flags A | live flags B
constexpr uint64_t kStaticSlots = 2ull * SPT_PEAKS_STATIC_MAX;         // two hash slots per record at the limit; a power of two
constexpr size_t kKeysOff = 0;
constexpr size_t kValsOff = kKeysOff + kStaticSlots * 8;
constexpr size_t kAliveOff0 = kValsOff + kStaticSlots * 4;
constexpr size_t kAliveOff1 = kAliveOff0 + SPT_PEAKS_STATIC_MAX;
constexpr size_t kStaticBytes = kAliveOff1 + SPT_PEAKS_STATIC_MAX;     // 6.5 MiB
static_assert((kStaticSlots & (kStaticSlots - 1)) == 0, "hash capacity must be a power of two");
static_assert(kValsOff % 256 == 0 && kAliveOff0 % 256 == 0 && kAliveOff1 % 256 == 0, "sub-buffers keep the alignment");

static __device__ __align__(256) unsigned char g_peaks_scratch[kStaticBytes];

// Every call shares the block and finds in it what the last call left: the keys of the slots this call will use are set
// to "empty" first.  (Values are only read where a key was found, and the live flags of all n records are written before
// they are read, so neither needs clearing.)  Device code may name the array directly, as here.
__global__ void peaks_static_clear_kernel(uint64_t nslots) {
    unsigned long long* keys = reinterpret_cast<unsigned long long*>(g_peaks_scratch + kKeysOff);
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nslots; i += (uint64_t)gridDim.x * blockDim.x)
        keys[i] = ~0ull;
}

// Device address of the block on the current device; asked of the runtime the first time a device is seen.
constexpr int kStaticMaxDev = 64;
static std::mutex g_static_mu;
static unsigned char* g_static_ptr[kStaticMaxDev] = {};

static cudaError_t static_scratch(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDev) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_peaks_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_static_ptr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_static_ptr[dev];
    return cudaSuccess;
}

// The hash-table peak filter of spt_peak_filter with every working buffer inside the static block.  `a` arrives with the
// list (cand, n <= SPT_PEAKS_STATIC_MAX) and the plan's tables filled in; d_peaks / d_count are the caller's.  Enqueues
// on st; no allocation, no synchronisation (after the first call on a device, which loads the module that holds the block).
cudaError_t peaks_static_filter(PeakArgs a, const int32_t* windows, int32_t nwindows, spt_candidate* d_peaks,
                                unsigned long long* d_count, long long capacity, cudaStream_t st, int64_t* nlaunch) {
    unsigned char* base = nullptr;
    cudaError_t e = static_scratch(&base);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(d_count, 0, 8, st);
    if (e != cudaSuccess || a.n <= 0) return e;
    uint64_t hcap = 1024;                                              // sized like spt_peak_filter's table
    while (hcap < 2 * (uint64_t)a.n) hcap <<= 1;
    if (hcap > kStaticSlots) return cudaErrorInvalidValue;             // the caller checks n first; not reached
    a.hkeys = reinterpret_cast<unsigned long long*>(base + kKeysOff);
    a.vals = reinterpret_cast<uint32_t*>(base + kValsOff);
    a.hmask = hcap - 1;
    uint8_t* alive[2] = {base + kAliveOff0, base + kAliveOff1};
    const unsigned nblk = (unsigned)((hcap + 1023) / 1024 < 1184 ? (hcap + 1023) / 1024 : 1184);
    peaks_static_clear_kernel<<<nblk, 256, 0, st>>>(hcap);
    launch_peaks_insert(a, st);
    const uint8_t* in = nullptr;
    for (int32_t i = 0; i < nwindows; ++i) {
        launch_peaks_stencil(a, windows[i], in, alive[i & 1], st);
        if (i + 1 < nwindows) launch_peaks_erase(a, in, alive[i & 1], false, st);
        in = alive[i & 1];
    }
    launch_peaks_compact(a, in, d_peaks, d_count, capacity, st);
    if (nlaunch) *nlaunch = 2 + 2 * nwindows;
    return cudaGetLastError();
}

}  // namespace spt
