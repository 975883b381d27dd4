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
// Per stage (a run of channel groups that fits shared memory), see plan.cpp for the tables:
//   A  expand : E_j[e]  = y[c0+j][t0+wlo+e] | y[c0+j][t0+wlo+e+kH] << 16          (global -> shared)
//   B  presum : P_r[u]  = sum_j E_j[u + shift_r[j]]   for every variant r of every group  (shared -> shared)
//   C  gather : acc[d][q] += P_{r(d)}[q + b(d)]       one LDS.32 + one IADD = 2*G algorithmic adds, packed
//   F  flush  : every <= 257/decim channels the 16-bit lanes are widened into the int32 DM transform (L2 RMW).
// ---------------------------------------------------------------------------------------------------------------
struct TiledArgs {
    const void* in;            // series of beam 0
    int64_t row_stride;        // elements
    int64_t beam_stride;       // elements
    int32_t* out;
    int64_t out_beam_stride;
    const TileDesc* tiles;
    const StageDesc* stages;
    const GroupDesc* groups;
    const int16_t* var_shift;
    const uint16_t* trial_off;
    const int32_t* nout;       // range local
    const int64_t* offset;     // range local
    int32_t ntile_dm, ntile_t, nbeam;
};

__device__ __forceinline__ uint32_t ld_word_or_zero(const uint32_t* p, bool ok) { return ok ? __ldg(p) : 0u; }

template <typename T, int DT, int G>
__global__ void __launch_bounds__(kThreads, 1) dedisp_tiled_kernel(const TiledArgs a) {
    constexpr int TPW = DT / (kThreads / 32);
    static_assert(TPW >= 1, "DT must be a multiple of the warp count");
    extern __shared__ __align__(16) uint32_t smem[];
    uint16_t* s_tab = reinterpret_cast<uint16_t*>(smem);                    // [ngrp][DT]
    GroupDesc* s_grp = reinterpret_cast<GroupDesc*>(smem + kTabWords);      // [ngrp]
    uint32_t* s_data = smem + kTabWords + kDescWords;                       // variants, then expansion rows

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    int bid = blockIdx.x;
    const int dmt = bid % a.ntile_dm; bid /= a.ntile_dm;
    const int tt = bid % a.ntile_t;
    const int beam = bid / a.ntile_t;
    const TileDesc td = a.tiles[dmt];
    const int64_t t0 = (int64_t)tt * kTT;
    if (t0 >= a.nout[td.trial0]) return;  // nout is non-increasing in the trial index (delays grow with DM)

    const T* in = reinterpret_cast<const T*>(a.in) + (int64_t)beam * a.beam_stride;
    uint32_t acc[TPW][16];
#pragma unroll
    for (int q = 0; q < TPW; ++q)
#pragma unroll
        for (int j = 0; j < 16; ++j) acc[q][j] = 0u;
    bool first_flush = true;

    for (int s = 0; s < td.nstage; ++s) {
        const StageDesc sd = a.stages[td.stage0 + s];
        uint32_t* s_var = s_data;
        uint32_t* s_exp = s_data + ((sd.vwords + 3) & ~3);
        __syncthreads();  // everyone is done with the previous stage's tables and variants
        // stage tables -> shared
        {
            const uint32_t* gsrc = reinterpret_cast<const uint32_t*>(a.groups + sd.grp0);
            uint32_t* gdst = reinterpret_cast<uint32_t*>(s_grp);
            for (int i = tid; i < sd.ngrp * (int)(sizeof(GroupDesc) / 4); i += kThreads) gdst[i] = __ldg(gsrc + i);
            const uint16_t* tsrc = a.trial_off + (int64_t)sd.grp0 * DT;
            for (int i = tid; i < sd.ngrp * DT; i += kThreads) s_tab[i] = __ldg(tsrc + i);
        }
        // ---- A: expand raw samples into half-interleaved 16-bit words --------------------------------------
        {
            int idx = 0;
            for (int g = 0; g < sd.ngrp; ++g) {
              const GroupDesc gd = a.groups[sd.grp0 + g];
              for (int j = 0; j < gd.nch; ++j, ++idx) {
                if ((idx & (kThreads / 32 - 1)) != warp) continue;
                const T* row = in + (int64_t)(gd.chan0 + j) * a.row_stride;
                const int64_t p0 = t0 + gd.wlo;  // multiple of 4
                uint32_t* E = s_exp + gd.ebase + j * gd.elen;
                for (int e4 = lane; e4 < (gd.elen >> 2); e4 += 32) {
                    const int64_t plo = p0 + 4 * e4, phi = plo + kH;
                    uint4 w;
                    if (sizeof(T) == 1) {
                        const uint32_t lo = ld_word_or_zero(reinterpret_cast<const uint32_t*>(row + plo), plo < a.row_stride);
                        const uint32_t hi = ld_word_or_zero(reinterpret_cast<const uint32_t*>(row + phi), phi < a.row_stride);
                        const uint32_t lo_e = lo & 0x00FF00FFu, lo_o = __byte_perm(lo, 0u, 0x4341);
                        const uint32_t hi_e = hi & 0x00FF00FFu, hi_o = __byte_perm(hi, 0u, 0x4341);
                        w.x = __byte_perm(lo_e, hi_e, 0x5410);
                        w.y = __byte_perm(lo_o, hi_o, 0x5410);
                        w.z = __byte_perm(lo_e, hi_e, 0x7632);
                        w.w = __byte_perm(lo_o, hi_o, 0x7632);
                    } else {
                        uint2 lo = make_uint2(0u, 0u), hi = make_uint2(0u, 0u);
                        if (plo < a.row_stride) lo = __ldg(reinterpret_cast<const uint2*>(row + plo));
                        if (phi < a.row_stride) hi = __ldg(reinterpret_cast<const uint2*>(row + phi));
                        w.x = __byte_perm(lo.x, hi.x, 0x5410);
                        w.y = __byte_perm(lo.x, hi.x, 0x7632);
                        w.z = __byte_perm(lo.y, hi.y, 0x5410);
                        w.w = __byte_perm(lo.y, hi.y, 0x7632);
                    }
                    *reinterpret_cast<uint4*>(E + 4 * e4) = w;
                }
              }
            }
        }
        __syncthreads();
        // ---- B: pre-sum every variant of every group -------------------------------------------------------
        {
            int idx = 0;
            for (int g = 0; g < sd.ngrp; ++g) {
                const GroupDesc gd = s_grp[g];
                for (int r = 0; r < gd.nvar; ++r, ++idx) {
                    if ((idx & (kThreads / 32 - 1)) != warp) continue;
                    const int16_t* sh = a.var_shift + (int64_t)(gd.var0 + r) * kMaxG;
                    const uint32_t* E0 = s_exp + gd.ebase;
                    uint32_t* P = s_var + gd.vbase + r * gd.vlen;
                    if (gd.nch == G) {
                        const uint32_t* E[G];
#pragma unroll
                        for (int j = 0; j < G; ++j) E[j] = E0 + j * gd.elen + (int)sh[j];
                        for (int u = lane; u < gd.vlen; u += 32) {
                            uint32_t sum = E[0][u];
#pragma unroll
                            for (int j = 1; j < G; ++j) sum += E[j][u];
                            P[u] = sum;
                        }
                    } else {  // a group the plan had to shrink (few channels, many relative-delay vectors)
                        for (int u = lane; u < gd.vlen; u += 32) {
                            uint32_t sum = 0;
                            for (int j = 0; j < gd.nch; ++j) sum += E0[j * gd.elen + (int)sh[j] + u];
                            P[u] = sum;
                        }
                    }
                }
            }
        }
        __syncthreads();
        // ---- C: gather-accumulate ------------------------------------------------------------------------------
        for (int g = 0; g < sd.ngrp; ++g) {
            const uint16_t* to = s_tab + g * DT + warp * TPW;
#pragma unroll
            for (int q = 0; q < TPW; ++q) {
                const uint32_t* src = s_data + to[q] + lane;
#pragma unroll
                for (int j = 0; j < 16; ++j) acc[q][j] += src[32 * j];
            }
        }
        // ---- F: widen the 16-bit lanes into the int32 DM transform -------------------------------------------
        if (sd.flush) {
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
    }
}

template <typename T, int DT, int G>
static int launch_tiled_inst(const TiledArgs& a, cudaStream_t st) {
    static bool attr_set = false;
    auto kern = dedisp_tiled_kernel<T, DT, G>;
    const int smem_bytes = kSmemWords * 4;
    if (!attr_set) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes) != cudaSuccess) return -1;
        attr_set = true;
    }
    const int64_t nblocks = (int64_t)a.ntile_dm * a.ntile_t * a.nbeam;
    if (nblocks <= 0) return 0;
    if (nblocks > 0x7fffffffLL) return -1;
    kern<<<(unsigned)nblocks, kThreads, smem_bytes, st>>>(a);
    return 0;
}

int launch_dedisp_tiled(bool is_u16, int DT, int G, const void* in, int64_t row_stride, int64_t beam_stride,
                        int32_t* out, int64_t out_beam_stride, const TileDesc* tiles, const StageDesc* stages,
                        const GroupDesc* groups, const int16_t* var_shift, const uint16_t* trial_off,
                        const int32_t* nout, const int64_t* offset, int32_t ntile_dm, int32_t ntile_t, int32_t nbeam,
                        cudaStream_t st) {
    TiledArgs a{in, row_stride, beam_stride, out, out_beam_stride, tiles, stages, groups, var_shift, trial_off,
                nout, offset, ntile_dm, ntile_t, nbeam};
#define SPT_CASE(DT_, G_)                                                              \
    if (DT == DT_ && G == G_)                                                          \
        return is_u16 ? launch_tiled_inst<uint16_t, DT_, G_>(a, st) : launch_tiled_inst<uint8_t, DT_, G_>(a, st);
    SPT_CASE(64, 1) SPT_CASE(64, 2) SPT_CASE(64, 4) SPT_CASE(64, 8)
    SPT_CASE(32, 1) SPT_CASE(32, 2) SPT_CASE(32, 4) SPT_CASE(32, 8)
#undef SPT_CASE
    return -1;
}

}  // namespace spt
