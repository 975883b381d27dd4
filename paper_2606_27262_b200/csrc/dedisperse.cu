// dedisperse.cu -- a2 (time decimation) and a3 (brute-force incoherent dedispersion) for sm_100a.
//
//   y_k[c][j]  = sum_{m<k} x[c][k*j+m]                      (BASELINE.json north_star (3); reading B1)
//   out[d][t]  = sum_c y_k[c][t + delay[d][c]], t < nout[d]   (PAPER.md:80 shift-and-sum; PAPER.md:90 DM transform)
//
// Kernel design: DESIGN.md section 5.  No tensor cores: the path is integer shift-and-add, bound by the
// shared-memory load pipe and the integer ALUs, not a dense contraction.
#include <cuda_runtime.h>

#include <atomic>

#include "internal.h"
#include "kernels.h"

namespace spt {

// ---------------------------------------------------------------------------------------------------------------
// a2. Time decimation by k = 2^m.  One thread makes four consecutive outputs from 4k input bytes (k 32-bit words),
// each word reduced with DP4A against a byte mask.  HBM bound: reads nchan*nsamp bytes, writes 2*nchan*nsamp/k.  The bounds
// of the series (maxval[0] = largest, maxval[1] = smallest sample; the caller resets them) come out of the same pass.
// ---------------------------------------------------------------------------------------------------------------
__global__ void decimate_kernel(const uint8_t* __restrict__ x, int64_t in_row_stride, int64_t in_beam_stride,
                                uint16_t* __restrict__ y, int64_t out_row_stride, int64_t out_beam_stride,
                                int32_t nchan, int64_t nsamp_k, int32_t k, uint32_t* __restrict__ maxval) {
    const int64_t quads = (nsamp_k + 3) >> 2;  // groups of 4 outputs per row
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t vmax = 0u, vmin = 0xffffffffu;    // bounds of the outputs this thread makes (threads past the row: neutral)
    if (q < quads) {
        const int32_t c = blockIdx.y, b = blockIdx.z;
        const uint8_t* src = x + (int64_t)b * in_beam_stride + (int64_t)c * in_row_stride;
        uint16_t* dst = y + (int64_t)b * out_beam_stride + (int64_t)c * out_row_stride;
        const int64_t j0 = q << 2;
        uint32_t o[4] = {0u, 0u, 0u, 0u};
        if (j0 + 4 <= nsamp_k) {
            const uint32_t* w = reinterpret_cast<const uint32_t*>(src + j0 * k);  // 4-byte aligned: strides are multiples of 16
            if (k == 2) {
                const uint32_t w0 = __ldg(w), w1 = __ldg(w + 1);
                o[0] = __dp4a(w0, 0x00000101u, 0u); o[1] = __dp4a(w0, 0x01010000u, 0u);
                o[2] = __dp4a(w1, 0x00000101u, 0u); o[3] = __dp4a(w1, 0x01010000u, 0u);
            } else {
                const int wpo = k >> 2;  // words per output
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    for (int m = 0; m < wpo; ++m) o[i] = __dp4a(__ldg(w + i * wpo + m), 0x01010101u, o[i]);
            }
            uint2 pk;
            pk.x = o[0] | (o[1] << 16);
            pk.y = o[2] | (o[3] << 16);
            *reinterpret_cast<uint2*>(dst + j0) = pk;
            vmax = max(max(o[0], o[1]), max(o[2], o[3]));
            vmin = min(min(o[0], o[1]), min(o[2], o[3]));
        } else {  // ragged tail of the row
            for (int64_t j = j0; j < nsamp_k; ++j) {
                uint32_t s = 0;
                for (int m = 0; m < k; ++m) s += src[j * k + m];
                dst[j] = (uint16_t)s;
                vmax = max(vmax, s);
                vmin = min(vmin, s);
            }
        }
        // The row padding (rows are 16-element multiples) repeats the row's last sample.  No stored output reads it, but the
        // pass that makes the 8-bit copy runs over whole rows, and the lanes of discarded outputs next to a valid one must
        // stay inside the bounds the kernel was given.
        if (q == quads - 1) {
            const int64_t pad_end = min((nsamp_k + 15) & ~(int64_t)15, out_row_stride);
            const uint16_t last = dst[nsamp_k - 1];                    // written by this thread just above
            for (int64_t j = nsamp_k; j < pad_end; ++j) dst[j] = last;
        }
    }
    // Bounds of the series (largest and smallest sample, over the real samples only) as a by-product: they bound the 16-bit lanes
    // of the dedispersion and decide whether the series gets an 8-bit copy.  One warp reduction; the atomics are issued
    // only by warps that improve on what is already known, which after the first few blocks is next to none.
    if (maxval != nullptr) {
        vmax = __reduce_max_sync(0xffffffffu, vmax);
        vmin = __reduce_min_sync(0xffffffffu, vmin);
        if ((threadIdx.x & 31) == 0) {
            if (vmax > *reinterpret_cast<volatile uint32_t*>(maxval)) atomicMax(maxval, vmax);
            if (vmin < *reinterpret_cast<volatile uint32_t*>(maxval + 1)) atomicMin(maxval + 1, vmin);
        }
    }
}

// The same for a padded copy of a uint8 filterbank whose rows are not 16-byte multiples (one thread per row).
__global__ void fill_row_pad_u8_kernel(uint8_t* __restrict__ x, int64_t pitch, int64_t nsamp, int64_t nrows) {
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nrows) return;
    uint8_t* row = x + r * pitch;
    const uint8_t last = row[nsamp - 1];
    for (int64_t j = nsamp; j < pitch; ++j) row[j] = last;
}

// Largest and smallest sample of a uint8 filterbank -> maxval[0], maxval[1] (bounds for the ranges that read the raw input).
__global__ void max_u8_kernel(const uint4* __restrict__ x, int64_t n16, uint32_t* __restrict__ maxval) {
    uint32_t m = 0, lo = 0xffffffffu;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (int64_t)gridDim.x * blockDim.x) {
        const uint4 v = __ldg(x + i);
        m = __vmaxu4(__vmaxu4(v.x, v.y), __vmaxu4(__vmaxu4(v.z, v.w), m));
        lo = __vminu4(__vminu4(v.x, v.y), __vminu4(__vminu4(v.z, v.w), lo));
    }
    m = max(max(m & 0xffu, (m >> 8) & 0xffu), max((m >> 16) & 0xffu, m >> 24));
    lo = min(min(lo & 0xffu, (lo >> 8) & 0xffu), min((lo >> 16) & 0xffu, lo >> 24));
    m = __reduce_max_sync(0xffffffffu, m);
    lo = __reduce_min_sync(0xffffffffu, lo);
    if ((threadIdx.x & 31) == 0) {
        if (m > 0) atomicMax(maxval, m);
        atomicMin(maxval + 1, lo);
    }
}

// The same for a decimated (uint16) series (its row padding repeats real samples: decimate_kernel).
__global__ void max_u16_kernel(const uint4* __restrict__ x, int64_t n16, uint32_t* __restrict__ maxval) {
    uint32_t m = 0, lo = 0xffffffffu;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (int64_t)gridDim.x * blockDim.x) {
        const uint4 v = __ldg(x + i);
        m = __vmaxu2(__vmaxu2(v.x, v.y), __vmaxu2(__vmaxu2(v.z, v.w), m));
        lo = __vminu2(__vminu2(v.x, v.y), __vminu2(__vminu2(v.z, v.w), lo));
    }
    m = max(m & 0xffffu, m >> 16);
    lo = min(lo & 0xffffu, lo >> 16);
    m = __reduce_max_sync(0xffffffffu, m);
    lo = __reduce_min_sync(0xffffffffu, lo);
    if ((threadIdx.x & 31) == 0) {
        if (m > 0) atomicMax(maxval, m);
        atomicMin(maxval + 1, lo);
    }
}

// SM count of the current device (grid-stride kernels launch 8 blocks per SM); looked up once per device.
int sm_count() {
    constexpr int kMaxDev = 64;
    static std::atomic<int> cached[kMaxDev];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDev) return 148;
    int n = cached[dev].load(std::memory_order_relaxed);
    if (n > 0) return n;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) { cudaGetLastError(); n = 148; }
    cached[dev].store(n, std::memory_order_relaxed);
    return n;
}

void launch_max_u16(const uint16_t* x, int64_t nelem, uint32_t* maxval, cudaStream_t st) {
    const int64_t n16 = nelem / 8;            // rows are 16-element multiples
    if (n16 <= 0) return;
    max_u16_kernel<<<sm_count() * 8, 256, 0, st>>>(reinterpret_cast<const uint4*>(x), n16, maxval);
}

void launch_fill_row_pad_u8(uint8_t* x, int64_t pitch, int64_t nsamp, int64_t nrows, cudaStream_t st) {
    if (nrows <= 0 || nsamp <= 0 || pitch <= nsamp) return;
    fill_row_pad_u8_kernel<<<(unsigned)((nrows + 255) / 256), 256, 0, st>>>(x, pitch, nsamp, nrows);
}

void launch_max_u8(const uint8_t* x, int64_t nbytes, uint32_t* maxval, cudaStream_t st) {
    const int64_t n16 = nbytes / 16;          // rows are 16-byte multiples
    if (n16 <= 0) return;
    max_u8_kernel<<<sm_count() * 8, 256, 0, st>>>(reinterpret_cast<const uint4*>(x), n16, maxval);
}

// 8-bit copy of a decimated series: c = y - (smallest sample of the series), made only when the series spans less than 256
// (quantised noise does: its decimated sums sit within a few sigma of k times the mean).  info[0..3] = {largest value of
// the copy, 0 (its floor), flag: 1 = the copy is valid, bias = the smallest sample (added back per channel when the lanes
// are widened)}.  The dedispersion of the range is one dual launch (dedisp_dual_kernel): every block looks at the flag and
// takes the copy with the copy's tables, or the uint16 series with its own.
__global__ void compact_u16_kernel(const uint4* __restrict__ y, uint2* __restrict__ c, int64_t n8, const uint32_t* __restrict__ maxval,
                                   uint32_t* __restrict__ info) {
    const uint32_t vmax = __ldg(maxval), vmin = __ldg(maxval + 1);
    const bool ok = vmin <= vmax && vmax - vmin <= 255u;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        info[0] = ok ? vmax - vmin : 0u; info[1] = 0u; info[2] = ok ? 1u : 0u; info[3] = ok ? vmin : 0u;
    }
    if (!ok) return;
    const uint32_t m2 = vmin * 0x00010001u;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n8; i += (int64_t)gridDim.x * blockDim.x) {
        uint4 v = __ldg(y + i);                                   // eight samples
        v.x -= m2; v.y -= m2; v.z -= m2; v.w -= m2;               // no borrow between the halves: every sample >= vmin
        uint2 o;
        o.x = __byte_perm(v.x, v.y, 0x6420);
        o.y = __byte_perm(v.z, v.w, 0x6420);
        c[i] = o;
    }
}

void launch_compact_u16(const uint16_t* y, uint8_t* c, int64_t nelem, const uint32_t* maxval, uint32_t* info, cudaStream_t st) {
    const int64_t n8 = nelem / 8;             // rows are 16-element multiples
    if (n8 <= 0) return;
    compact_u16_kernel<<<sm_count() * 8, 256, 0, st>>>(reinterpret_cast<const uint4*>(y), reinterpret_cast<uint2*>(c), n8, maxval, info);
}

void launch_decimate(const uint8_t* x, int64_t in_row_stride, int64_t in_beam_stride, uint16_t* y,
                     int64_t out_row_stride, int64_t out_beam_stride, int32_t nchan, int32_t nbeam, int64_t nsamp_k,
                     int32_t k, uint32_t* maxval, cudaStream_t st) {
    const int64_t quads = (nsamp_k + 3) >> 2;
    if (quads <= 0) return;
    dim3 grid((unsigned)((quads + 255) / 256), (unsigned)nchan, (unsigned)nbeam);
    decimate_kernel<<<grid, 256, 0, st>>>(x, in_row_stride, in_beam_stride, y, out_row_stride, out_beam_stride, nchan,
                                          nsamp_k, k, maxval);
}

// ---------------------------------------------------------------------------------------------------------------
// a3, bring-up / cross-check kernel: one thread per output sample, straight from the definition, global memory only.
// ---------------------------------------------------------------------------------------------------------------
template <typename T>
__global__ void dedisp_naive_kernel(const T* __restrict__ y, int64_t row_stride, int64_t beam_stride,
                                    const int32_t* __restrict__ delay, const int32_t* __restrict__ nout,
                                    const int64_t* __restrict__ offset, int32_t nchan, int32_t* __restrict__ out,
                                    int64_t out_beam_stride) {
    const int32_t d = blockIdx.y, b = blockIdx.z;
    const int32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nout[d]) return;
    const T* src = y + (int64_t)b * beam_stride + t;
    const int32_t* dl = delay + (int64_t)d * nchan;
    int32_t acc = 0;
    for (int32_t c = 0; c < nchan; ++c) acc += (int32_t)src[(int64_t)c * row_stride + dl[c]];
    out[(int64_t)b * out_beam_stride + offset[d] + t] = acc;
}

template <typename T>
void launch_dedisp_naive(const T* y, int64_t row_stride, int64_t beam_stride, const int32_t* d_delay,
                         const int32_t* d_nout, const int64_t* d_offset, int32_t nchan, int32_t ndm, int32_t nbeam,
                         int32_t max_nout, int32_t* out, int64_t out_beam_stride, cudaStream_t st) {
    if (max_nout <= 0) return;
    dim3 grid((unsigned)((max_nout + 255) / 256), (unsigned)ndm, (unsigned)nbeam);
    dedisp_naive_kernel<T><<<grid, 256, 0, st>>>(y, row_stride, beam_stride, d_delay, d_nout, d_offset, nchan, out,
                                                 out_beam_stride);
}
template void launch_dedisp_naive<uint8_t>(const uint8_t*, int64_t, int64_t, const int32_t*, const int32_t*,
                                           const int64_t*, int32_t, int32_t, int32_t, int32_t, int32_t*, int64_t,
                                           cudaStream_t);
template void launch_dedisp_naive<uint16_t>(const uint16_t*, int64_t, int64_t, const int32_t*, const int32_t*,
                                            const int64_t*, int32_t, int32_t, int32_t, int32_t, int32_t*, int64_t,
                                            cudaStream_t);

// ---------------------------------------------------------------------------------------------------------------
// a3, the product kernel.  One block = DT trials x TT = 2*kH output samples of one beam; 8 warps, TPW = DT/8 trials
// per warp, two blocks per SM; lane l of a warp owns the packed words q = l + 32*j (j < kH/32) of each of its
// trials: the low 16 bits of word q accumulate output first+q, the high 16 bits output first+kH+q, where
// first = t0 - skew[trial] (every trial of the tile has its own window start, which narrows what the tile reads).
// Because both halves of a word move together, a read at ANY sample offset is one aligned 32-bit shared-memory load.
//
// Per stage (a run of channel groups that fits shared memory; tables built by plan.cpp):
//   T  TMA    : every warp issues its share of the cp.async.bulk copies of the stage's raw channel rows, warp 0 also the
//               table blob and the next stage's descriptors (global -> shared, completion on one mbarrier with one
//               arrive.expect_tx per warp); they land while the previous stage is gathered
//   B  presum : P_r[u] = sum_j y[c0+j][t0 + dmin + u + s_j + tau^r_j] | (same at +kH) << 16 for every variant r of
//               every group.  A lane makes 4 consecutive u from aligned 32-bit words of the raw rows: per channel the
//               five samples u..u+4 as packed words w0..w4, base += w_i, delta_i = w_{i+1} - w_i (the alternate shift
//               is one sample later), then walks the prefix chain: variant k = base + delta of the first k channels.
//   C  gather : acc[d][q] += P_{r(d)}[q + b(d)]       one LDS.32 + one add = 2*G algorithmic adds
//   F  flush  : a lane sums (sample - smallest sample of the launch); before it could exceed 65535 (every
//               floor(65535 / (largest - smallest sample)) channels, at worst every 257/decim) the 16-bit lanes are widened
//               into the int32 DM transform, the floor added back (first time a store, then RED).
// ---------------------------------------------------------------------------------------------------------------

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra WAIT_%=;\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// L2 policy of the DM-transform lines: a tile adds to its 64 x 512 outputs about once per 450 channels, eight or nine
// times in all; between two passes the lines should stay in L2 rather than go to HBM half summed and come back.
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void st_hint(int32_t* addr, int32_t v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.b32 [%0], %1, %2;" ::"l"(addr), "r"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void red_hint(int32_t* addr, int32_t v, uint64_t pol) {
    asm volatile("red.global.add.L2::cache_hint.s32 [%0], %1, %2;" ::"l"(addr), "r"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void lds64(uint32_t addr, uint32_t& a, uint32_t& b) {
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "r"(addr));
}
__device__ __forceinline__ void sts128(uint32_t addr, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}

__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}

// The five packed words w_i = y[u0+i] | y[u0+i+kH] << 16, i = 0..4, of one entry (a channel at one of its shifts).
// addr: shared-memory byte address of the aligned 32-bit word holding the lane's first sample; c1: the entry's second
// descriptor word (uint8: bits 0-4 = 8 * position of that sample inside the word, bits 8-23 = PRMT selector of sample 4;
// uint16: bits 0-1 = position inside the 8-byte unit the address points at).
template <typename T, int KH>
__device__ __forceinline__ void load_entry(uint32_t addr, uint32_t c1, uint32_t (&w)[5]) {
    constexpr int kH = KH;
    if (sizeof(T) == 1) {
        const uint32_t aL = lds32(addr), bL = lds32(addr + 4), aH = lds32(addr + kH), bH = lds32(addr + kH + 4);
        uint32_t Lw, Hw;   // samples 0..3 (the shift amount is taken modulo 32: the selector bits above do not matter)
        asm("shf.r.wrap.b32 %0, %1, %2, %3;" : "=r"(Lw) : "r"(aL), "r"(bL), "r"(c1));
        asm("shf.r.wrap.b32 %0, %1, %2, %3;" : "=r"(Hw) : "r"(aH), "r"(bH), "r"(c1));
        const uint32_t Le = Lw & 0x00FF00FFu, Lo = prmt(Lw, 0u, 0x4341u);
        const uint32_t He = Hw & 0x00FF00FFu, Ho = prmt(Hw, 0u, 0x4341u);
        w[0] = prmt(Le, He, 0x5410u);
        w[1] = prmt(Lo, Ho, 0x5410u);
        w[2] = prmt(Le, He, 0x7632u);
        w[3] = prmt(Lo, Ho, 0x7632u);
        w[4] = prmt(bL, bH, c1 >> 8) & 0x00FF00FFu;                    // sample 4 = byte a0 of the second word
    } else {
        // two 64-bit loads per half (a lane's samples start on an 8-byte boundary: conflict free), then the five samples
        // from position c1 = 0..3 of the eight
        uint32_t x0L, x1L, x2L, x3L, x0H, x1H, x2H, x3H;
        lds64(addr, x0L, x1L); lds64(addr + 8, x2L, x3L);
        lds64(addr + 2 * kH, x0H, x1H); lds64(addr + 2 * kH + 8, x2H, x3H);
        if (c1 & 2u) { x0L = x1L; x1L = x2L; x2L = x3L; x0H = x1H; x1H = x2H; x2H = x3H; }
        const bool odd = (c1 & 1u) != 0u;
        const uint32_t s_even = odd ? 0x7632u : 0x5410u, s_odd = odd ? 0x5410u : 0x7632u;
        w[0] = prmt(x0L, x0H, s_even);
        w[1] = prmt(odd ? x1L : x0L, odd ? x1H : x0H, s_odd);
        w[2] = prmt(x1L, x1H, s_even);
        w[3] = prmt(odd ? x2L : x1L, odd ? x2H : x1H, s_odd);
        w[4] = prmt(x2L, x2H, s_even);
    }
}

// B: one warp task = kChunkU variant words (4 per lane) of every variant of one group.  All control flow is warp
// uniform and the NE entries are straight-line code (unused entries repeat the first one; their deltas are never
// taken): a lane past the end of the variants works on the last four words and does not store.
template <typename T, int NE, int KH>
__device__ __forceinline__ void presum_task(const uint32_t* __restrict__ tb, uint32_t task, uint32_t var_addr,
                                            uint32_t raw_addr, int lane, uint32_t floor2, const uint4 gh) {
    const int vlen = (int)gh.y;
    const uint32_t meta = gh.z;
    const int ntog = (int)((meta >> 8) & 0xffu), ncorr = (int)((meta >> 16) & 0xffu);
    const uint4* cd = reinterpret_cast<const uint4*>(tb + (gh.w & 0xffffu));
    const uint4* vd = reinterpret_cast<const uint4*>(tb + (gh.w >> 16));
    int u0 = (int)(task >> 8) * kChunkU + lane * 4;
    const bool active = u0 < vlen;                // vlen is a multiple of 4
    u0 = active ? u0 : vlen - 4;
    const uint32_t rbase = raw_addr + (uint32_t)u0 * (uint32_t)sizeof(T);
    const uint32_t vbase = var_addr + (uint32_t)u0 * 4u;
    // every channel of the group enters the base sum once: take the launch's smallest sample off each (both lanes)
    const uint32_t bias = 0u - (gh.x >> 16) * floor2;
    uint32_t cur[4] = {bias, bias, bias, bias};
    uint32_t dl[NE][4];
#pragma unroll
    for (int q2 = 0; q2 < NE / 2; ++q2) {
        const uint4 c2 = cd[q2];                  // two entries per load
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int q = 2 * q2 + h;
            const uint32_t cx = h ? c2.z : c2.x, cy = h ? c2.w : c2.y;
            uint32_t w[5];
            load_entry<T, KH>(rbase + (cx & 0x3ffffu), cy, w);
#pragma unroll
            for (int i = 0; i < 4; ++i) dl[q][i] = w[i + 1] - w[i];
            if (cx & kEntryAddBase) {
#pragma unroll
                for (int i = 0; i < 4; ++i) cur[i] += w[i];
            }
        }
    }
    // prefix chain: after step k, cur = base sum + deltas of the first k entries
    uint4 v4 = vd[0];
#pragma unroll
    for (int k = 0; k <= NE; ++k) {
        if (k <= ntog) {
            if (k > 0) {
#pragma unroll
                for (int i = 0; i < 4; ++i) cur[i] += dl[k - 1][i];
            }
            if (k > 0 && (k & 3) == 0) v4 = vd[k >> 2];
            const uint32_t dst = (k & 3) == 0 ? v4.x : (k & 3) == 1 ? v4.y : (k & 3) == 2 ? v4.z : v4.w;
            if (dst != 0xffffffffu && active) sts128(vbase + dst * 4u, cur[0], cur[1], cur[2], cur[3]);
        }
    }
    // variants off the chain (few): all deltas, minus those the variant does not take
    for (int c = 0; c < ncorr; ++c) {
        const uint32_t* vc = reinterpret_cast<const uint32_t*>(vd) + (NE + 4) + 2 * c;   // chain_words(NE)
        const uint32_t dst = vc[0], mask = vc[1];
        uint32_t o[4] = {cur[0], cur[1], cur[2], cur[3]};
#pragma unroll
        for (int q = 0; q < NE; ++q)
            if (mask & (1u << q)) {
#pragma unroll
                for (int i = 0; i < 4; ++i) o[i] -= dl[q][i];
            }
        if (active) sts128(vbase + dst * 4u, o[0], o[1], o[2], o[3]);
    }
}

// NEMAX: the largest entry class the plan's tables hold (8, 12 or 16): the kernel carries only the pre-sum instances it
// needs, so that a plan of small groups does not pay for the registers of the large ones.
// KH: packed words per trial per tile (the tile is 2*KH outputs wide): 256, or 224 where the plan's cost model prefers it.
template <typename T, int DT, int NEMAX, int KH>
__device__ __forceinline__ void dedisp_tile_body(const TiledArgs& a) {
    constexpr int kH = KH, kTT = 2 * KH;
    constexpr int NW = kThreads / 32;
    constexpr int TPW = DT / NW;
    constexpr int NJ = kH / 32;
    static_assert(TPW >= 1 && TPW * NW == DT, "DT must be a multiple of the warp count");
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t bar = smem_u32(smem);
    // control area: mbarrier, then per trial of the tile {row pointer, nout} for the flush
    int32_t** const s_rowp = reinterpret_cast<int32_t**>(smem + 64);
    int2* const s_valid = reinterpret_cast<int2*>(smem + 64 + kMaxDT * 8);      // [lo, hi) valid outputs of the trial in this tile
    RowDesc* const s_rows = reinterpret_cast<RowDesc*>(smem + 64 + kMaxDT * 16);                          // [2][kMaxStageRows]
    StageIndex* const s_sidx = reinterpret_cast<StageIndex*>(smem + 64 + kMaxDT * 16 + 2 * kMaxStageRows * 16);  // [2]
    uint32_t* const s_var = reinterpret_cast<uint32_t*>(smem + kSmemCtrlBytes + 2 * kBlobBytes);
    uint8_t* const s_rawb = reinterpret_cast<uint8_t*>(s_var + a.vcap_words);
    const uint32_t var_addr = smem_u32(s_var), raw_addr = smem_u32(s_rawb);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (a.enable != nullptr && __ldg(a.enable) != a.enable_want) return;     // the other launch of this range does the work
    int bid = blockIdx.x;
    const int dmt = bid % a.ntile_dm; bid /= a.ntile_dm;
    const int ntt = a.tail > 0 ? a.tail_tiles : a.ntile_t;
    const int beam = bid / ntt;
    const TileDesc td = a.tiles[dmt];
    const int tt = a.tail > 0 ? td.tt_last - bid % ntt : (bid % ntt + ntt - td.tshift % ntt) % ntt;
    if (tt < 0) return;
    const int64_t t0 = (int64_t)tt * kTT;   // trial i of the tile computes the outputs t0 - skew[i] + [0, kTT)

    const T* in = reinterpret_cast<const T*>(a.in) + (int64_t)beam * a.beam_stride;

    // T: every warp issues its share of the bulk copies of stage s (a warp issues the copies of its lanes one after the
    // other, so eight short chains instead of one long one) and arrives on the stage barrier with the byte count of its
    // share: rows k = warp, warp + NW, ...; warp 0 also copies the table blob and the NEXT stage's index and row
    // descriptors, so that no global-memory latency sits between a stage's pre-sum and its gather.  Stage 0 reads its
    // descriptors from global memory, later stages from shared.
    auto issue_stage = [&](int s) {
        const StageIndex si = s == 0 ? a.sidx[td.stage0] : s_sidx[s & 1];
        const RowDesc* rows = s == 0 ? a.rows + si.row0 : s_rows + (s & 1) * kMaxStageRows;
        uint32_t bytes = 0;
        const uint32_t k = (uint32_t)warp + (uint32_t)NW * (uint32_t)lane;
        RowDesc r{0, 0, 0, 0};
        if (k < si.nrows) r = rows[k];
        __syncwarp();
        fence_proxy_async();  // generic-proxy reads of the buffers (previous stage) before async-proxy writes
        if (k < si.nrows) {
            // the window [pos, pos + nelem) of the channel's row, clipped to the row: the part before the row (skewed
            // output windows start before t = 0) and the part after it are not copied (all multiples of 16 elements)
            const int64_t pos = t0 + r.astart;
            const int64_t beg = pos < 0 ? 0 : pos;
            const int64_t end = min(pos + (int64_t)r.nelem, a.row_stride);
            const int64_t n = end > beg ? end - beg : 0;
            if (n > 0)
                bulk_g2s(smem_u32(s_rawb + r.soff) + (uint32_t)(beg - pos) * (uint32_t)sizeof(T),
                         in + (int64_t)r.chan * a.row_stride + beg, (uint32_t)n * (uint32_t)sizeof(T), bar);
            bytes = (uint32_t)n * (uint32_t)sizeof(T);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
        if (lane == 0) {
            if (warp == 0) {
                bulk_g2s(smem_u32(smem + kSmemCtrlBytes + (s & 1) * kBlobBytes), a.blob + si.blob_word0, si.blob_words * 4u, bar);
                bulk_g2s(smem_u32(s_sidx + ((s + 1) & 1)), a.sidx + td.stage0 + s + 1, 16u, bar);
                bulk_g2s(smem_u32(s_rows + ((s + 1) & 1) * kMaxStageRows), a.rows + si.row0 + si.nrows, kMaxStageRows * 16u, bar);
                bytes += si.blob_words * 4u + 16u + kMaxStageRows * 16u;
            }
            mbar_expect_tx(bar, bytes);   // one of the NW arrivals that let the phase end
        }
    };

    if (tid == 0) {
        mbar_init(bar, NW);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    int have = 0;
    if (tid < DT) {
        const int d = td.trial0 + (tid < td.ntrial ? tid : td.ntrial - 1);
        const int64_t first = t0 - a.skew[td.skew0 + tid];                 // output sample of accumulator index 0
        s_rowp[tid] = a.out + (int64_t)beam * a.out_beam_stride + a.offset[d] + first;
        // first valid output of the trial in this tile: the start of the row, or of the tail that is wanted
        const int64_t want = a.tail > 0 ? max((int64_t)0, (int64_t)a.nout[d] - a.tail) : 0;
        const int lo = (int)min((int64_t)kTT, max((int64_t)0, want - first));
        const int hi = tid < td.ntrial ? (int)min((int64_t)kTT, max((int64_t)lo, (int64_t)a.nout[d] - first)) : lo;
        s_valid[tid] = make_int2(lo, hi);
        have = hi > lo;
    }
    if (!__syncthreads_or(have)) return;    // no trial of the tile has an output here (ragged rows, skewed windows)
    if (t0 < (int64_t)a.skew_max + 32) {
        // Windows that start before the row are not copied.  What the raw region holds there feeds only outputs with t < 0,
        // which are discarded, but their 16-bit lanes must not carry into the valid high lanes: make the first contents
        // zero (later stages find there the bounded samples of an earlier stage).
        uint4* r4 = reinterpret_cast<uint4*>(s_rawb);
        const int n4 = (kSmemDataBytes - a.vcap_words * 4) / 16;
        for (int i = tid; i < n4; i += kThreads) r4[i] = make_uint4(0u, 0u, 0u, 0u);
        __syncthreads();
    }
    issue_stage(0);

    uint32_t acc[TPW][NJ];
#pragma unroll
    for (int q = 0; q < TPW; ++q)
#pragma unroll
        for (int j = 0; j < NJ; ++j) acc[q][j] = 0u;
    bool first_flush = true;
    // F: widen the 16-bit lanes into the int32 DM transform.  A lane may sum floor(65535 / largest sample) channels: the
    // bound comes from the data of this launch (255 * decimation in the worst case, which is what the stages are cut for)
    // What a lane sums is (sample - floor) with floor = the smallest sample of the launch, added back here: a lane may
    // then sum floor(65535 / (largest - smallest sample)) channels.  Tiles whose windows start before the rows (skew) keep
    // floor = 0: there the lanes of discarded outputs read zeros, which must not go negative next to a valid lane.
    const uint32_t vmax = __ldg(a.maxval), vmin = __ldg(a.maxval + 1);
    const uint32_t floor1 = (t0 < (int64_t)a.skew_max + 32 || vmin > vmax) ? 0u : vmin;
    const uint32_t floor2 = floor1 * 0x00010001u;
    const int lane_cap = (int)(65535u / max(1u, vmax - floor1));
    // what every channel summed owes when the lanes are widened: the floor taken off its samples here and, for the 8-bit
    // copy of a decimated series, the floor the copy was made with
    const uint32_t back1 = floor1 + ((a.enable != nullptr && a.enable_want == 1u) ? __ldg(a.enable + 1) : 0u);
    int since = 0;
    // A warp none of whose trials has an output in this tile (the last DM tile of a range holds fewer than DT trials; rows end
    // at different samples; a stream push wants only the tail) still does its share of the pre-sums but neither gathers nor
    // widens.  s_valid was published by the barrier above.
    bool warp_live = false;
#pragma unroll
    for (int q = 0; q < TPW; ++q) {
        const int2 ok = s_valid[warp * TPW + q];
        warp_live = warp_live || ok.y > ok.x;
    }
    auto flush_lanes = [&]() {
        if (!warp_live) return;
        const uint64_t pol_out = policy_evict_last();
        const uint32_t back = (uint32_t)since * back1;    // the floor of the channels summed since the last pass
#pragma unroll
        for (int q = 0; q < TPW; ++q) {
            const int dl = warp * TPW + q;
            int32_t* row = s_rowp[dl];
            const int2 ok = s_valid[dl];
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int i = lane + 32 * j;
                const int32_t lo = (int32_t)((acc[q][j] & 0xFFFFu) + back), hi = (int32_t)((acc[q][j] >> 16) + back);
                const bool ok_lo = i >= ok.x && i < ok.y, ok_hi = i + kH >= ok.x && i + kH < ok.y;
                if (first_flush) {
                    if (ok_lo) st_hint(row + i, lo, pol_out);
                    if (ok_hi) st_hint(row + i + kH, hi, pol_out);
                } else {
                    if (ok_lo) red_hint(row + i, lo, pol_out);  // fire-and-forget RED in L2
                    if (ok_hi) red_hint(row + i + kH, hi, pol_out);
                }
                acc[q][j] = 0u;
            }
        }
        first_flush = false;
    };

    for (int s = 0; s < td.nstage; ++s) {
        mbar_wait(bar, (uint32_t)(s & 1));
        const uint32_t* tb = reinterpret_cast<const uint32_t*>(smem + kSmemCtrlBytes + (s & 1) * kBlobBytes);
        const int ngrp = (int)tb[0];
        const int nch_stage = (int)(tb[1] >> 8);      // channels this stage adds to every lane
        const int ntask = (int)tb[2];
        const uint16_t* toff = reinterpret_cast<const uint16_t*>(tb + tb[3]);

        // ---- B: pre-sum every variant of every group ---------------------------------------------------------
        for (int tk = warp; tk < ntask; tk += NW) {
            const uint32_t task = tb[kBlobHdrWords + 4 * ngrp + tk];
            const uint4 gh = *reinterpret_cast<const uint4*>(tb + kBlobHdrWords + 4 * (task & 0xffu));   // 128-bit broadcast load
            const uint32_t nent = gh.z & 0xffu;       // warp uniform: the smallest straight-line instance that holds the group
            if (NEMAX == 8 || nent <= 8u) presum_task<T, 8, KH>(tb, task, var_addr, raw_addr, lane, floor2, gh);
            else if (NEMAX == 12 || nent <= 12u) presum_task<T, 12, KH>(tb, task, var_addr, raw_addr, lane, floor2, gh);
            else presum_task<T, 16, KH>(tb, task, var_addr, raw_addr, lane, floor2, gh);
        }
        __syncthreads();  // variants complete; raw rows and the other blob buffer are free
        if (s + 1 < td.nstage) issue_stage(s + 1);

        if (since + nch_stage > lane_cap) { flush_lanes(); since = 0; }
        // ---- C: gather-accumulate ------------------------------------------------------------------------------
        if (warp_live) {
            const uint32_t lane_addr = var_addr + (uint32_t)lane * 4u;
            const uint16_t* to = toff + warp * TPW;
            auto offsets = [&](const uint16_t* t, uint32_t (&off)[TPW]) {
                if (TPW == 8) {
                    const uint4 o4 = *reinterpret_cast<const uint4*>(t);
                    off[0] = o4.x & 0xffffu; off[1] = o4.x >> 16; off[2] = o4.y & 0xffffu; off[3] = o4.y >> 16;
                    off[4 % TPW] = o4.z & 0xffffu; off[5 % TPW] = o4.z >> 16; off[6 % TPW] = o4.w & 0xffffu; off[7 % TPW] = o4.w >> 16;
                } else {
#pragma unroll
                    for (int q = 0; q < TPW; ++q) off[q] = t[q];
                }
            };
            int g = 0;
            for (; g + 2 <= ngrp; g += 2, to += 2 * DT) {   // two groups per pass: one 3-input add per pair of loads
                uint32_t off0[TPW], off1[TPW];
                offsets(to, off0);
                offsets(to + DT, off1);
#pragma unroll
                for (int q = 0; q < TPW; ++q) {
                    const uint32_t s0 = lane_addr + off0[q] * 4u, s1 = lane_addr + off1[q] * 4u;
#pragma unroll
                    for (int j = 0; j < NJ; ++j) acc[q][j] += lds32(s0 + 128u * j) + lds32(s1 + 128u * j);
                }
            }
            if (g < ngrp) {
                uint32_t off0[TPW];
                offsets(to, off0);
#pragma unroll
                for (int q = 0; q < TPW; ++q) {
                    const uint32_t s0 = lane_addr + off0[q] * 4u;
#pragma unroll
                    for (int j = 0; j < NJ; ++j) acc[q][j] += lds32(s0 + 128u * j);
                }
            }
        }
        since += nch_stage;
        __syncthreads();  // everyone is done with this stage's variants
    }
    flush_lanes();
}

template <typename T, int DT, int NEMAX, int KH>
__global__ void __launch_bounds__(kThreads, 2) dedisp_tiled_kernel(const TiledArgs a) {
    dedisp_tile_body<T, DT, NEMAX, KH>(a);
}

// A decimated range in ONE launch: the 8-bit copy of its series with the copy's tables when the copy was made (a8.enable
// points at {flag, bias}, written on the device just before), the uint16 series with its own tables otherwise.  The two
// table sets tile the range identically (same DM tiles, same skews, same grid), so a block does the same tile either way.
template <int DT, int NEMAX, int KH>
__global__ void __launch_bounds__(kThreads, 2) dedisp_dual_kernel(const TiledArgs a8, const TiledArgs a16) {
    if (__ldg(a8.enable) == 1u) dedisp_tile_body<uint8_t, DT, NEMAX, KH>(a8);
    else dedisp_tile_body<uint16_t, DT, NEMAX, KH>(a16);
}

// the opt-in to 113 KB of dynamic shared memory is a per-device attribute of the function: one flag per device and instance
template <typename K>
static int opt_in_smem(K kern, std::atomic<bool>* attr_set) {
    constexpr int kMaxDev = 64;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (dev < 0 || dev >= kMaxDev || !attr_set[dev].load(std::memory_order_acquire)) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes) != cudaSuccess) return -1;
        if (dev >= 0 && dev < kMaxDev) attr_set[dev].store(true, std::memory_order_release);
    }
    return 0;
}

static int64_t blocks_of(const TiledArgs& a) {
    return (int64_t)a.ntile_dm * (a.tail > 0 ? a.tail_tiles : a.ntile_t) * a.nbeam;
}

template <typename T, int DT, int NEMAX, int KH>
static int launch_tiled_inst(const TiledArgs& a, cudaStream_t st) {
    static std::atomic<bool> attr_set[64];
    auto kern = dedisp_tiled_kernel<T, DT, NEMAX, KH>;
    if (opt_in_smem(kern, attr_set) != 0) return -1;
    const int64_t nblocks = blocks_of(a);
    if (nblocks <= 0) return 0;
    if (nblocks > 0x7fffffffLL) return -1;
    kern<<<(unsigned)nblocks, kThreads, kSmemBytes, st>>>(a);
    return 0;
}

template <int DT, int NEMAX, int KH>
static int launch_dual_inst(const TiledArgs& a8, const TiledArgs& a16, cudaStream_t st) {
    static std::atomic<bool> attr_set[64];
    auto kern = dedisp_dual_kernel<DT, NEMAX, KH>;
    if (opt_in_smem(kern, attr_set) != 0) return -1;
    const int64_t nblocks = blocks_of(a16);
    if (nblocks != blocks_of(a8)) return -1;
    if (nblocks <= 0) return 0;
    if (nblocks > 0x7fffffffLL) return -1;
    kern<<<(unsigned)nblocks, kThreads, kSmemBytes, st>>>(a8, a16);
    return 0;
}

// Instances: 64-trial tiles at both tile widths, 32-trial tiles (option dm_tile, tests) at the wide one only.
#define SPT_DISPATCH(CALL)                                                                   \
    if (DT == 64 && kh == 256 && max_ent == 8) return CALL(64, 8, 256);                       \
    if (DT == 64 && kh == 256 && max_ent == 12) return CALL(64, 12, 256);                     \
    if (DT == 64 && kh == 256 && max_ent == 16) return CALL(64, 16, 256);                     \
    if (DT == 64 && kh == 224 && max_ent == 8) return CALL(64, 8, 224);                       \
    if (DT == 64 && kh == 224 && max_ent == 12) return CALL(64, 12, 224);                     \
    if (DT == 64 && kh == 224 && max_ent == 16) return CALL(64, 16, 224);                     \
    if (DT == 32 && kh == 256 && max_ent == 8) return CALL(32, 8, 256);                       \
    if (DT == 32 && kh == 256 && max_ent == 12) return CALL(32, 12, 256);                     \
    if (DT == 32 && kh == 256 && max_ent == 16) return CALL(32, 16, 256);                     \
    return -1;

int launch_dedisp_dual(int DT, int max_ent, int kh, const TiledArgs& a8, const TiledArgs& a16, cudaStream_t st) {
#define SPT_CALL_DUAL(D, N, K) launch_dual_inst<D, N, K>(a8, a16, st)
    SPT_DISPATCH(SPT_CALL_DUAL)
#undef SPT_CALL_DUAL
}

int launch_dedisp_tiled(bool is_u16, int DT, int max_ent, int kh, const TiledArgs& a, cudaStream_t st) {
#define SPT_CALL_TILED(D, N, K) (is_u16 ? launch_tiled_inst<uint16_t, D, N, K>(a, st) : launch_tiled_inst<uint8_t, D, N, K>(a, st))
    SPT_DISPATCH(SPT_CALL_TILED)
#undef SPT_CALL_TILED
}
#undef SPT_DISPATCH

}  // namespace spt
