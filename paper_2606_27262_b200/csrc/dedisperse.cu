// dedisperse.cu -- a2 (time decimation) and a3 (brute-force incoherent dedispersion) for sm_100a.
//
//   y_k[c][j]  = sum_{m<k} x[c][k*j+m]                      (BASELINE.json north_star (3); reading B1)
//   out[d][t]  = sum_c y_k[c][t + delay[d][c]], t < nout[d]   (PAPER.md:80 shift-and-sum; PAPER.md:90 DM transform)
//
// Kernel design: DESIGN.md section 5.  No tensor cores: the path is integer shift-and-add, bound by the
// shared-memory load pipe and the integer ALUs, not a dense contraction.
#include <cuda_runtime.h>

#include "internal.h"
#include "kernels.h"

namespace spt {

// ---------------------------------------------------------------------------------------------------------------
// a2. Time decimation by k = 2^m.  One thread makes four consecutive outputs from 4k input bytes (k 32-bit words),
// each word reduced with DP4A against a byte mask.  HBM bound: reads nchan*nsamp bytes, writes 2*nchan*nsamp/k.
// ---------------------------------------------------------------------------------------------------------------
__global__ void decimate_kernel(const uint8_t* __restrict__ x, int64_t in_row_stride, int64_t in_beam_stride,
                                uint16_t* __restrict__ y, int64_t out_row_stride, int64_t out_beam_stride,
                                int32_t nchan, int64_t nsamp_k, int32_t k) {
    const int64_t quads = (nsamp_k + 3) >> 2;  // groups of 4 outputs per row
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= quads) return;
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
    } else {  // ragged tail of the row
        for (int64_t j = j0; j < nsamp_k; ++j) {
            uint32_t s = 0;
            for (int m = 0; m < k; ++m) s += src[j * k + m];
            dst[j] = (uint16_t)s;
        }
    }
}

void launch_decimate(const uint8_t* x, int64_t in_row_stride, int64_t in_beam_stride, uint16_t* y,
                     int64_t out_row_stride, int64_t out_beam_stride, int32_t nchan, int32_t nbeam, int64_t nsamp_k,
                     int32_t k, cudaStream_t st) {
    const int64_t quads = (nsamp_k + 3) >> 2;
    if (quads <= 0) return;
    dim3 grid((unsigned)((quads + 255) / 256), (unsigned)nchan, (unsigned)nbeam);
    decimate_kernel<<<grid, 256, 0, st>>>(x, in_row_stride, in_beam_stride, y, out_row_stride, out_beam_stride, nchan,
                                          nsamp_k, k);
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
// a3, the product kernel.  One block = DT trials x TT = 2*kH output samples of one beam; 16 warps, TPW = DT/16
// trials per warp; lane l of a warp owns the packed words q = l + 32*j (j < 16) of each of its trials: the low
// 16 bits of word q accumulate output t0+q, the high 16 bits output t0+kH+q.  Because both halves of a word
// move together, a read at ANY sample offset is one aligned 32-bit shared-memory load (no byte realignment).
//
// Per stage (a run of channel groups that fits shared memory; tables built by plan.cpp):
//   T  TMA    : one elected warp issues cp.async.bulk copies of the stage's table blob and raw channel rows
//               (global -> shared, completion on an mbarrier); they land while the previous stage is gathered
//   B  presum : P_r[u] = sum_j y[c0+j][t0 + dmin + u + rho^r_j] | (same at +kH) << 16 for every variant r of every
//               group, in one sweep over the group's (channel, shift) pairs: base pairs go to all variants, delta
//               pairs replace the base for the variants in their mask (predicated adds)
//   C  gather : acc[d][q] += P_{r(d)}[q + b(d)]       one LDS.32 + one add = 2*G algorithmic adds
//   F  flush  : every <= 257/decim channels the 16-bit lanes are widened into the int32 DM transform (L2 RMW).
// ---------------------------------------------------------------------------------------------------------------
struct TiledArgs {
    const void* in;            // series of beam 0
    int64_t row_stride;        // elements (multiple of 16)
    int64_t beam_stride;       // elements
    int32_t* out;
    int64_t out_beam_stride;
    const TileDesc* tiles;
    const StageIndex* sidx;
    const RowDesc* rows;
    const uint32_t* blob;
    const int32_t* nout;       // range local
    const int64_t* offset;     // range local
    int32_t vcap_words, ntile_dm, ntile_t, nbeam;
};

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
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <typename T, int DT>
__global__ void __launch_bounds__(kThreads, 1) dedisp_tiled_kernel(const TiledArgs a) {
    constexpr int NW = kThreads / 32;
    constexpr int TPW = DT / NW;
    static_assert(TPW >= 1 && TPW * NW == DT, "DT must be a multiple of the warp count");
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t bar = smem_u32(smem);
    uint32_t* const s_var = reinterpret_cast<uint32_t*>(smem + kSmemCtrlBytes + 2 * kBlobBytes);
    uint8_t* const s_rawb = reinterpret_cast<uint8_t*>(s_var + a.vcap_words);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    int bid = blockIdx.x;
    const int dmt = bid % a.ntile_dm; bid /= a.ntile_dm;
    const int tt = bid % a.ntile_t;
    const int beam = bid / a.ntile_t;
    const TileDesc td = a.tiles[dmt];
    const int64_t t0 = (int64_t)tt * kTT;
    if (t0 >= a.nout[td.trial0]) return;  // nout is non-increasing in the trial index (delays grow with DM)

    const T* in = reinterpret_cast<const T*>(a.in) + (int64_t)beam * a.beam_stride;

    // T: the elected warp arms the stage barrier with the byte count and issues the bulk copies
    auto issue_stage = [&](int s) {
        const StageIndex si = a.sidx[td.stage0 + s];
        uint32_t bytes = 0;
        for (uint32_t k = lane; k < si.nrows; k += 32) {
            const RowDesc r = a.rows[si.row0 + k];
            const int64_t room = a.row_stride - (t0 + r.astart);
            const int64_t n = room < (int64_t)r.nelem ? (room > 0 ? room : 0) : (int64_t)r.nelem;
            bytes += (uint32_t)n * (uint32_t)sizeof(T);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
        if (lane == 0) {
            fence_proxy_async();  // generic-proxy reads of the buffers (previous stage) before async-proxy writes
            mbar_expect_tx(bar, bytes + si.blob_words * 4u);
            bulk_g2s(smem_u32(smem + kSmemCtrlBytes + (s & 1) * kBlobBytes), a.blob + si.blob_word0, si.blob_words * 4u, bar);
        }
        __syncwarp();
        for (uint32_t k = lane; k < si.nrows; k += 32) {
            const RowDesc r = a.rows[si.row0 + k];
            const int64_t pos = t0 + r.astart;
            const int64_t room = a.row_stride - pos;
            const int64_t n = room < (int64_t)r.nelem ? (room > 0 ? room : 0) : (int64_t)r.nelem;
            if (n > 0)
                bulk_g2s(smem_u32(s_rawb + r.soff), in + (int64_t)r.chan * a.row_stride + pos,
                         (uint32_t)n * (uint32_t)sizeof(T), bar);
        }
    };

    if (tid == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    __syncthreads();
    if (warp == 0) issue_stage(0);

    uint32_t acc[TPW][16];
#pragma unroll
    for (int q = 0; q < TPW; ++q)
#pragma unroll
        for (int j = 0; j < 16; ++j) acc[q][j] = 0u;
    bool first_flush = true;

    for (int s = 0; s < td.nstage; ++s) {
        mbar_wait(bar, (uint32_t)(s & 1));
        const uint32_t* tb = reinterpret_cast<const uint32_t*>(smem + kSmemCtrlBytes + (s & 1) * kBlobBytes);
        const int ngrp = (int)tb[0];
        const bool flush = tb[1] != 0u;
        const uint32_t* pairs = tb + kBlobHdrWords + 4 * ngrp;
        const uint16_t* toff = reinterpret_cast<const uint16_t*>(pairs + tb[2]);

        // ---- B: pre-sum every variant of every group ---------------------------------------------------------
        {
            int task = 0;
            for (int g = 0; g < ngrp; ++g) {
                const uint32_t* gh = tb + kBlobHdrWords + 4 * g;
                const int vlen = (int)gh[1];
                const int nchunk = (vlen + 63) >> 6;
                for (int ch = 0; ch < nchunk; ++ch, ++task) {
                    if ((task & (NW - 1)) != warp) continue;
                    const int vbase = (int)gh[0], nvar = (int)gh[3];
                    const uint32_t pair0 = gh[2] & 0xffffu, npairs = gh[2] >> 16;
                    const int u0 = (ch << 6) + lane, u1 = u0 + 32;   // rows carry kRowSlack elements past vlen
                    uint32_t av0[kMaxVar], av1[kMaxVar];
#pragma unroll
                    for (int r = 0; r < kMaxVar; ++r) { av0[r] = 0u; av1[r] = 0u; }
                    uint32_t base0 = 0u, base1 = 0u, wb0 = 0u, wb1 = 0u;
                    for (uint32_t q = 0; q < npairs; ++q) {
                        const uint32_t d = pairs[pair0 + q];
                        const T* row = reinterpret_cast<const T*>(s_rawb + (d & 0x1ffffu));
                        const uint32_t w0 = __byte_perm((uint32_t)row[u0], (uint32_t)row[u0 + kH], 0x5410);
                        const uint32_t w1 = __byte_perm((uint32_t)row[u1], (uint32_t)row[u1 + kH], 0x5410);
                        if (d & kPairBaseBit) {
                            wb0 = w0; wb1 = w1; base0 += w0; base1 += w1;
                        } else {
                            const uint32_t m = d >> 20, d0 = w0 - wb0, d1 = w1 - wb1;
#pragma unroll
                            for (int r = 0; r < kMaxVar; ++r)
                                if (m & (1u << r)) { av0[r] += d0; av1[r] += d1; }
                        }
                    }
                    uint32_t* P = s_var + vbase;
#pragma unroll
                    for (int r = 0; r < kMaxVar; ++r)
                        if (r < nvar) {
                            if (u0 < vlen) P[r * vlen + u0] = base0 + av0[r];
                            if (u1 < vlen) P[r * vlen + u1] = base1 + av1[r];
                        }
                }
            }
        }
        __syncthreads();  // variants complete; raw rows and the other blob buffer are free
        if (warp == 0 && s + 1 < td.nstage) issue_stage(s + 1);

        // ---- C: gather-accumulate ------------------------------------------------------------------------------
        for (int g = 0; g < ngrp; ++g) {
            const uint16_t* to = toff + g * DT + warp * TPW;
#pragma unroll
            for (int q = 0; q < TPW; ++q) {
                const uint32_t* src = s_var + to[q] + lane;
#pragma unroll
                for (int j = 0; j < 16; ++j) acc[q][j] += src[32 * j];
            }
        }
        // ---- F: widen the 16-bit lanes into the int32 DM transform -------------------------------------------
        if (flush) {
#pragma unroll
            for (int q = 0; q < TPW; ++q) {
                const int dl = warp * TPW + q;
                if (dl < td.ntrial) {
                    const int d = td.trial0 + dl;
                    const int64_t n = a.nout[d];
                    int32_t* row = a.out + (int64_t)beam * a.out_beam_stride + a.offset[d] + t0;
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const int i = lane + 32 * j;
                        const int32_t lo = (int32_t)(acc[q][j] & 0xFFFFu), hi = (int32_t)(acc[q][j] >> 16);
                        if (t0 + i < n) row[i] = first_flush ? lo : row[i] + lo;
                        if (t0 + i + kH < n) row[i + kH] = first_flush ? hi : row[i + kH] + hi;
                    }
                }
#pragma unroll
                for (int j = 0; j < 16; ++j) acc[q][j] = 0u;
            }
            first_flush = false;
        }
        __syncthreads();  // everyone is done with this stage's variants
    }
}

template <typename T, int DT>
static int launch_tiled_inst(const TiledArgs& a, cudaStream_t st) {
    static bool attr_set = false;
    auto kern = dedisp_tiled_kernel<T, DT>;
    if (!attr_set) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes) != cudaSuccess) return -1;
        attr_set = true;
    }
    const int64_t nblocks = (int64_t)a.ntile_dm * a.ntile_t * a.nbeam;
    if (nblocks <= 0) return 0;
    if (nblocks > 0x7fffffffLL) return -1;
    kern<<<(unsigned)nblocks, kThreads, kSmemBytes, st>>>(a);
    return 0;
}

int launch_dedisp_tiled(bool is_u16, int DT, const void* in, int64_t row_stride, int64_t beam_stride, int32_t* out,
                        int64_t out_beam_stride, const TileDesc* tiles, const StageIndex* sidx, const RowDesc* rows,
                        const uint32_t* blob, int32_t vcap_words, const int32_t* nout, const int64_t* offset,
                        int32_t ntile_dm, int32_t ntile_t, int32_t nbeam, cudaStream_t st) {
    TiledArgs a{in, row_stride, beam_stride, out, out_beam_stride, tiles, sidx, rows, blob, nout, offset,
                vcap_words, ntile_dm, ntile_t, nbeam};
    if (DT == 64) return is_u16 ? launch_tiled_inst<uint16_t, 64>(a, st) : launch_tiled_inst<uint8_t, 64>(a, st);
    if (DT == 32) return is_u16 ? launch_tiled_inst<uint16_t, 32>(a, st) : launch_tiled_inst<uint8_t, 32>(a, st);
    return -1;
}

}  // namespace spt
