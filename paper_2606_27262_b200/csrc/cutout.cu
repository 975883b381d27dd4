// cutout.cu -- candidate cut-outs (Eq. 4; reading H): the two features the classifier is fed,
// the dedispersed dynamic spectrum at the candidate's DM and a DM transform over a narrow range around it, as exact integers.
//   dds[f][j] = sum_{c in band f} sum_{m<tbin} x[c][ts + j*tbin + m + delay(dm0, c)]
//   dmt[i][j] = sum_c            sum_{m<tbin} x[c][ts + j*tbin + m + delay(DM_i, c)],   DM_i = (dm0 - ddm) + i*step
// Samples outside the data count as 0.
//
// cutout_tiled_kernel: many candidates per launch (10-100 per beam per block; "custom, optimised
// GPU kernels").  One block = one candidate x 32 consecutive trial DMs x 256 time bins x a chunk of 256 channels.  The same
// idea as the search's dedispersion at small scale: a channel's window [ts + j0*tbin + delay(first trial), ... + delay(last
// trial)) is staged in shared memory ONCE and serves all 32 trials x 256 bins (a trial is a shift of the read position), so
// an output costs one shared-memory load and one add per channel (two loads when bins are wider than a sample: the window is
// staged as prefix sums and a bin is a difference).  Delays are made in the block with the plan's formula in double without
// contraction -- the integers equal the host's -- so there is no delay table in device memory.  Channel chunks meet in the
// outputs with integer RED.ADD (exact in any order).  The dynamic spectrum is one more "trial group" holding the single
// pseudo-trial dm0, whose sums are flushed per band.
#include <cuda_runtime.h>

#include <atomic>

#include "kernels.h"

namespace spt {

constexpr int kCutThreads = 256;
constexpr int kCutTrials = 32;     // trial DMs per block (4 per warp)
constexpr int kCutBins = 256;      // time bins per block (8 per lane)
constexpr int kCutChunk = 256;     // channels per block
constexpr int kCutSubMax = 16;     // channels staged at a time, at most

__device__ __forceinline__ int32_t cut_delay(double fch1, double foff, double tsamp, double dm, int c) {
    const double f = fch1 + (double)c * foff;
    const double inv_top = 1.0 / (fch1 * fch1);
    const double seconds = kDispersionConstantS * dm * (1.0 / (f * f) - inv_top);    // same expression and order as build_plan
    return (int32_t)floor(seconds / tsamp + 0.5);
}

__device__ __forceinline__ int cut_pad(int e) { return e + (e >> 5); }   // strided reads of the prefix sums stay conflict free

template <bool BINNED>
__global__ void __launch_bounds__(kCutThreads) cutout_tiled_kernel(const __grid_constant__ CutoutArgs a) {
    extern __shared__ __align__(16) uint32_t sm[];
    const int nsub = a.nsub;
    int32_t* const s_delay = reinterpret_cast<int32_t*>(sm);            // [kCutTrials][nsub]
    uint32_t* const s_w = sm + kCutTrials * nsub;                      // [nsub][wstride]: samples, or padded prefix sums
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const CutoutCand cd = a.cand[blockIdx.z];
    const int ngrp = (a.ndm + kCutTrials - 1) / kCutTrials;
    const int g = blockIdx.x % (ngrp + 1), jt = blockIdx.x / (ngrp + 1);
    const bool spectrum = g == ngrp;                                   // the extra group: the dynamic spectrum at dm0
    const int ntr = spectrum ? 1 : min(kCutTrials, a.ndm - g * kCutTrials);
    const int j0 = jt * kCutBins;
    const int nj = min(kCutBins, a.nt - j0);
    const int c_begin = blockIdx.y * kCutChunk, c_end = min(a.nchan, c_begin + kCutChunk);
    const int tbin = cd.tbin;
    const double step = a.ndm > 1 ? (2.0 * cd.ddm) / (double)(a.ndm - 1) : 0.0;
    const uint8_t* const beam = a.x + (int64_t)cd.beam * a.beam_stride;
    const int per = a.nchan / a.nf;
    int32_t* const dds = a.dds + (int64_t)cd.out * a.nf * a.nt;
    int32_t* const dmt = a.dmt + (int64_t)cd.out * a.ndm * a.nt;

    int32_t acc[4][8];
#pragma unroll
    for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int m = 0; m < 8; ++m) acc[q][m] = 0;

    for (int cs = c_begin; cs < c_end; cs += nsub) {
        const int ncs = min(nsub, c_end - cs);
        __syncthreads();                                               // the previous sub-chunk's readers are done
        // 1. delays of the group's trials at these channels (unused trial slots repeat the last trial)
        for (int idx = tid; idx < kCutTrials * ncs; idx += kCutThreads) {
            const int tl = idx / ncs, cc = idx - tl * ncs;
            const int i = g * kCutTrials + min(tl, ntr - 1);
            const double dm = spectrum ? cd.dm0 : (cd.dm0 - cd.ddm) + (double)i * step;
            s_delay[tl * nsub + cc] = cut_delay(a.fch1, a.foff, a.tsamp, dm, cs + cc);
        }
        __syncthreads();
        // 2. stage the windows: one warp per channel.  Delays grow with the trial DM, so the window runs from the first
        //    trial's delay to the last one's.
        for (int cc = warp; cc < ncs; cc += kCutThreads / 32) {
            const int first = s_delay[cc], last = s_delay[(ntr - 1) * nsub + cc];
            const int W = min(nj * tbin + (last - first), a.wcap);     // the host sized wcap for it; min() is a seat belt
            const int64_t base = cd.ts + (int64_t)j0 * tbin + first;
            const uint8_t* row = beam + (int64_t)(cs + cc) * a.nsamp;
            uint32_t* dst = s_w + cc * a.wstride;
            if (!BINNED) {
                for (int e = lane; e < W; e += 32) {
                    const int64_t s = base + e;
                    dst[e] = (s >= 0 && s < a.nsamp) ? (uint32_t)__ldg(row + s) : 0u;
                }
            } else {                                                   // dst[pad(e)] = sum of the first e samples of the window
                uint32_t run = 0;
                if (lane == 0) dst[0] = 0u;
                for (int e0 = 0; e0 < W; e0 += 128) {
                    uint32_t v[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const int e = e0 + 4 * lane + k;
                        const int64_t s = base + e;
                        v[k] = (e < W && s >= 0 && s < a.nsamp) ? (uint32_t)__ldg(row + s) : 0u;
                    }
                    const uint32_t p0 = v[0], p1 = p0 + v[1], p2 = p1 + v[2], p3 = p2 + v[3];
                    uint32_t incl = p3;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
                        if (lane >= o) incl += y;
                    }
                    const uint32_t b0 = run + incl - p3;
                    const int e = e0 + 4 * lane;
                    if (e < W) dst[cut_pad(e + 1)] = b0 + p0;
                    if (e + 1 < W) dst[cut_pad(e + 2)] = b0 + p1;
                    if (e + 2 < W) dst[cut_pad(e + 3)] = b0 + p2;
                    if (e + 3 < W) dst[cut_pad(e + 4)] = b0 + p3;
                    run += __shfl_sync(0xffffffffu, incl, 31);
                }
            }
        }
        __syncthreads();
        // 3. every output of the block takes its sample (its bin) of every staged channel
        for (int cc = 0; cc < ncs; ++cc) {
            const uint32_t* src = s_w + cc * a.wstride;
            const int first = s_delay[cc];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int tl = warp * 4 + q;
                if (tl >= ntr) break;                                   // warp uniform
                const int off = s_delay[tl * nsub + cc] - first;
                if (!BINNED) {
#pragma unroll
                    for (int m = 0; m < 8; ++m) acc[q][m] += (int32_t)src[off + lane + 32 * m];
                } else {
#pragma unroll
                    for (int m = 0; m < 8; ++m) {
                        const int e = min((lane + 32 * m) * tbin + off, a.wcap - tbin);   // bins past nj are dropped below
                        acc[q][m] += (int32_t)(src[cut_pad(e + tbin)] - src[cut_pad(e)]);
                    }
                }
            }
            if (spectrum && warp == 0) {                               // the band of this channel ends here: flush
                const int c = cs + cc;
                if ((c + 1) % per == 0 || c + 1 == c_end) {
                    const int f = c / per;
#pragma unroll
                    for (int m = 0; m < 8; ++m) {
                        const int j = lane + 32 * m;
                        if (j < nj) atomicAdd(dds + (int64_t)f * a.nt + j0 + j, acc[0][m]);
                        acc[0][m] = 0;
                    }
                }
            }
        }
    }
    if (!spectrum) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int tl = warp * 4 + q;
            if (tl >= ntr) break;
            int32_t* out = dmt + (int64_t)(g * kCutTrials + tl) * a.nt + j0;
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int j = lane + 32 * m;
                if (j < nj) atomicAdd(out + j, acc[q][m]);               // RED.ADD: the channel chunks meet here
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// The definition, one thread per output (kept for windows too long for shared memory: time bins of hundreds of samples).
// ---------------------------------------------------------------------------------------------------------------------
__global__ void cutout_naive_kernel(const __grid_constant__ CutoutArgs a) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int r = blockIdx.y;                                            // rows 0..ndm-1: DM transform; then nf spectrum bands
    if (j >= a.nt) return;
    const CutoutCand cd = a.cand[blockIdx.z];
    const bool band = r >= a.ndm;
    const int per = a.nchan / a.nf;
    const int c0 = band ? (r - a.ndm) * per : 0, c1 = band ? c0 + per : a.nchan;
    const double step = a.ndm > 1 ? (2.0 * cd.ddm) / (double)(a.ndm - 1) : 0.0;
    const double dm = band ? cd.dm0 : (cd.dm0 - cd.ddm) + (double)r * step;
    const uint8_t* beam = a.x + (int64_t)cd.beam * a.beam_stride;
    const int64_t base = cd.ts + (int64_t)j * cd.tbin;
    int32_t acc = 0;
    for (int c = c0; c < c1; ++c) {
        const uint8_t* row = beam + (int64_t)c * a.nsamp;
        const int64_t s0 = base + cut_delay(a.fch1, a.foff, a.tsamp, dm, c);
        for (int m = 0; m < cd.tbin; ++m) {
            const int64_t s = s0 + m;
            if (s >= 0 && s < a.nsamp) acc += (int32_t)row[s];
        }
    }
    if (band) a.dds[((int64_t)cd.out * a.nf + (r - a.ndm)) * a.nt + j] = acc;
    else a.dmt[((int64_t)cd.out * a.ndm + r) * a.nt + j] = acc;
}

// Host copy of the device's delay expression (plan.cpp's, compiled without contraction): sizes the windows.
static int32_t host_delay(double fch1, double foff, double tsamp, double dm, int c) {
    const double f = fch1 + (double)c * foff;
    const double inv_top = 1.0 / (fch1 * fch1);
    const double seconds = kDispersionConstantS * dm * (1.0 / (f * f) - inv_top);
    return (int32_t)std::floor(seconds / tsamp + 0.5);
}

// The outputs of the candidates in `a` must be zero when the launch starts (the tiled kernel adds into them).
int launch_cutout_batch(CutoutArgs& a, cudaStream_t st) {
    if (a.ncand < 1 || a.ncand > kCutoutMaxCand) return -1;
    // the widest window any block stages: a group's 32 trials at the lowest channel, plus 256 bins
    int64_t wmax = 0;
    int tbin_max = 1;
    const double step_den = a.ndm > 1 ? (double)(a.ndm - 1) : 1.0;
    for (int k = 0; k < a.ncand; ++k) {
        const CutoutCand& c = a.cand[k];
        const double step = a.ndm > 1 ? (2.0 * c.ddm) / step_den : 0.0;
        int64_t spread = 0;
        for (int g0 = 0; g0 < a.ndm; g0 += kCutTrials) {
            const int g1 = std::min(a.ndm - 1, g0 + kCutTrials - 1);
            const int64_t lo = host_delay(a.fch1, a.foff, a.tsamp, (c.dm0 - c.ddm) + (double)g0 * step, a.nchan - 1);
            const int64_t hi = host_delay(a.fch1, a.foff, a.tsamp, (c.dm0 - c.ddm) + (double)g1 * step, a.nchan - 1);
            spread = std::max(spread, hi - lo);
        }
        wmax = std::max<int64_t>(wmax, (int64_t)kCutBins * c.tbin + spread + c.tbin);
        tbin_max = std::max(tbin_max, c.tbin);
    }
    bool binned = false, unbinned = false;
    for (int k = 0; k < a.ncand; ++k) (a.cand[k].tbin > 1 ? binned : unbinned) = true;
    constexpr int64_t kSmemBudget = 96 * 1024;
    const int64_t wstride = wmax + wmax / 32 + 4;
    const int64_t nsub = std::min<int64_t>(kCutSubMax, (kSmemBudget - 1024) / ((wstride + kCutTrials) * 4));
    if (binned && unbinned) return -2;          // the caller launches the two kinds separately
    if (nsub < 1) {                             // windows too long for shared memory: the definition
        dim3 grid((unsigned)((a.nt + 127) / 128), (unsigned)(a.ndm + a.nf), (unsigned)a.ncand);
        cutout_naive_kernel<<<grid, 128, 0, st>>>(a);
        return cudaGetLastError() == cudaSuccess ? 0 : -1;
    }
    a.wcap = (int32_t)wmax;
    a.wstride = (int32_t)wstride;
    a.nsub = (int32_t)nsub;
    const size_t smem = (size_t)(kCutTrials * nsub + nsub * wstride) * 4;
    auto kern = binned ? cutout_tiled_kernel<true> : cutout_tiled_kernel<false>;
    if (smem > 48 * 1024) {
        constexpr int kMaxDev = 64;
        static std::atomic<bool> attr_set[2][kMaxDev];
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return -1;
        if (dev < 0 || dev >= kMaxDev || !attr_set[binned][dev].load(std::memory_order_acquire)) {
            if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBudget) != cudaSuccess) return -1;
            if (dev >= 0 && dev < kMaxDev) attr_set[binned][dev].store(true, std::memory_order_release);
        }
    }
    const int ngrp = (a.ndm + kCutTrials - 1) / kCutTrials + 1;
    const int njt = (a.nt + kCutBins - 1) / kCutBins;
    dim3 grid((unsigned)(ngrp * njt), (unsigned)((a.nchan + kCutChunk - 1) / kCutChunk), (unsigned)a.ncand);
    kern<<<grid, kCutThreads, smem, st>>>(a);
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace spt
