// sps.cu -- a4: boxcar single-pulse search over the DM transform (readings C1-C5, D1).
//
// One block per (beam, trial) row of N = nout samples:
//   pass 1  Sx = sum x (int64), Sxx = sum x^2 (uint64): exact, order independent -> mu, sigma in double
//   pass 2  segments of kSeg samples: block-wide inclusive prefix sum C (uint32, modulo 2^32) in shared memory,
//           S_w[t] = C[t+w] - C[t];  snr_w[t] = (N*S_w[t] - w*Sx) / (N*sigma*sqrt(w))  (numerator exact int64);
//           best width per t scanned in increasing w with strict '>' ; best >= threshold -> warp-aggregated
//           atomic append of {beam, trial, t, width, snr}.
// HBM bound by design (one compulsory read of the DM transform; the second pass of a row re-reads it from L2).
#include <cuda_runtime.h>

#include "kernels.h"

namespace spt {

constexpr int kSpsThreads = 512;
constexpr int kEpt = 8;                        // samples per thread per segment
constexpr int kSeg = kSpsThreads * kEpt;       // 4096 samples per segment (outputs + halo of the widest boxcar)

__device__ __forceinline__ int padi(int i) { return i + (i >> 5); }  // bank-conflict-free stride-8 access

__device__ __forceinline__ long long shfl_down_ll(long long v, int d) {
    int lo = (int)(v & 0xffffffffll), hi = (int)(v >> 32);
    lo = __shfl_down_sync(0xffffffffu, lo, d);
    hi = __shfl_down_sync(0xffffffffu, hi, d);
    return ((long long)hi << 32) | (unsigned int)lo;
}

__global__ void __launch_bounds__(kSpsThreads) sps_kernel(const SpsArgs a) {
    __shared__ uint32_t s_c[kSeg + 1 + (kSeg + 1) / 32 + 1];
    __shared__ long long s_red[2][kSpsThreads / 32];
    __shared__ uint32_t s_wtot[kSpsThreads / 32];
    __shared__ double s_scale[kMaxWidths];
    __shared__ long long s_wsum[kMaxWidths];
    __shared__ int s_live;

    const int d = blockIdx.x, b = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = a.nout[d];
    if (n <= 0) {
        if (tid == 0) { a.sum[(int64_t)b * a.ntrials + d] = 0; a.sumsq[(int64_t)b * a.ntrials + d] = 0ull; }
        return;
    }
    const int32_t* x = a.dmt + (int64_t)b * a.beam_stride + a.offset[d];  // 128-byte aligned row

    // ---- pass 1: exact integer statistics (reading C1) --------------------------------------------------------
    long long sx = 0;
    unsigned long long sxx = 0;
    {
        const int n4 = n >> 2;
        const int4* x4 = reinterpret_cast<const int4*>(x);
        for (int i = tid; i < n4; i += kSpsThreads) {
            const int4 v = x4[i];
            sx += (long long)v.x + v.y + v.z + v.w;
            sxx += (unsigned long long)(unsigned)v.x * (unsigned)v.x + (unsigned long long)(unsigned)v.y * (unsigned)v.y +
                   (unsigned long long)(unsigned)v.z * (unsigned)v.z + (unsigned long long)(unsigned)v.w * (unsigned)v.w;
        }
        for (int i = (n4 << 2) + tid; i < n; i += kSpsThreads) {
            const int v = x[i];
            sx += v;
            sxx += (unsigned long long)(unsigned)v * (unsigned)v;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            sx += shfl_down_ll(sx, o);
            sxx += (unsigned long long)shfl_down_ll((long long)sxx, o);
        }
        if (lane == 0) { s_red[0][warp] = sx; s_red[1][warp] = (long long)sxx; }
        __syncthreads();
        if (tid == 0) {
            long long S = 0; unsigned long long Q = 0;
            for (int w = 0; w < kSpsThreads / 32; ++w) { S += s_red[0][w]; Q += (unsigned long long)s_red[1][w]; }
            a.sum[(int64_t)b * a.ntrials + d] = S;
            a.sumsq[(int64_t)b * a.ntrials + d] = Q;
            // sigma^2 = (N*Sxx - Sx^2)/N^2 from 128-bit integers (N*Sxx reaches ~1e23)
            const unsigned long long N = (unsigned long long)n, US = (unsigned long long)S;
            const unsigned long long alo = N * Q, ahi = __umul64hi(N, Q);
            const unsigned long long blo = US * US, bhi = __umul64hi(US, US);
            unsigned long long dlo = alo - blo, dhi = ahi - bhi - (alo < blo ? 1ull : 0ull);
            if (ahi < bhi || (ahi == bhi && alo < blo)) { dlo = 0; dhi = 0; }  // cannot happen (Cauchy-Schwarz)
            const double num = (double)dhi * 18446744073709551616.0 + (double)dlo;
            const double sigma = sqrt(num / ((double)n * (double)n));
            const int live = (sigma > 0.0 && n >= 2) ? 1 : 0;
            s_live = live;
            for (int k = 0; k < a.nw; ++k) {
                const double w = (double)a.widths[k];
                s_scale[k] = live ? 1.0 / (((double)n * sigma) * sqrt(w)) : 0.0;
                s_wsum[k] = (long long)a.widths[k] * S;
            }
        }
        __syncthreads();
    }
    if (!s_live) return;  // sigma == 0 or N < 2: S/N == 0 everywhere, no candidates (reading C1)

    // ---- pass 2: boxcars, best width, threshold ------------------------------------------------------------------
    const int w0 = a.widths[0], wmax = a.widths[a.nw - 1];
    const int nbest = n - w0 + 1;              // best[t] is defined for t in [0, N - wmin]  (reading C5)
    if (nbest <= 0) return;
    const int halo = min(wmax, n);             // widths > N never apply
    const int adv = (kSeg - halo) & ~31;       // outputs per segment (launch_sps guarantees wmax <= kSeg - 32)
    const long long N64 = n;

    for (int tb = 0; tb < nbest; tb += adv) {
        // load kEpt consecutive samples per thread (coalesced via shared memory), zero beyond N
        __syncthreads();
        for (int i = tid; i < kSeg; i += kSpsThreads) {
            const int t = tb + i;
            s_c[padi(i + 1)] = t < n ? (uint32_t)x[t] : 0u;
        }
        __syncthreads();
        uint32_t v[kEpt];
        uint32_t run = 0;
#pragma unroll
        for (int i = 0; i < kEpt; ++i) { run += s_c[padi(tid * kEpt + i + 1)]; v[i] = run; }
        uint32_t incl = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += y;
        }
        if (lane == 31) s_wtot[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t wt = lane < kSpsThreads / 32 ? s_wtot[lane] : 0u;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_up_sync(0xffffffffu, wt, o);
                if (lane >= o) wt += y;
            }
            if (lane < kSpsThreads / 32) s_wtot[lane] = wt;  // inclusive over warps
        }
        __syncthreads();
        const uint32_t base = (incl - run) + (warp > 0 ? s_wtot[warp - 1] : 0u);
#pragma unroll
        for (int i = 0; i < kEpt; ++i) s_c[padi(tid * kEpt + i + 1)] = base + v[i];
        if (tid == 0) s_c[0] = 0u;
        __syncthreads();

        const int nthis = min(adv, nbest - tb);
        for (int i0 = 0; i0 < nthis; i0 += kSpsThreads) {
            const int i = i0 + tid;
            const int t = tb + i;
            bool hit = false;
            double best = 0.0;
            int bw = w0;
            if (i < nthis) {
                const uint32_t c0 = s_c[padi(i)];
                bool first = true;
                for (int k = 0; k < a.nw; ++k) {
                    const int w = a.widths[k];
                    if (t + w > n) break;
                    const uint32_t S = s_c[padi(i + w)] - c0;                       // exact: S < 2^32 (plan check)
                    const long long num = N64 * (long long)S - s_wsum[k];           // exact int64
                    const double snr = (double)num * s_scale[k];
                    if (first || snr > best) { best = snr; bw = w; first = false; }
                }
                hit = best >= a.threshold;
            }
            const unsigned m = __ballot_sync(0xffffffffu, hit);
            if (m) {
                unsigned long long slot0 = 0;
                if (lane == 0) slot0 = atomicAdd(a.count, (unsigned long long)__popc(m));
                slot0 = __shfl_sync(0xffffffffu, slot0, 0);
                if (hit) {
                    const long long slot = (long long)(slot0 + __popc(m & ((1u << lane) - 1u)));
                    if (slot < a.capacity) {
                        spt_candidate c;
                        c.beam = b; c.trial = d; c.t = t; c.width = bw; c.snr = (float)best;
                        a.cand[slot] = c;
                    }
                }
            }
        }
    }
}

void launch_sps(const SpsArgs& a, int32_t nbeam, cudaStream_t st) {
    if (a.ntrials <= 0 || nbeam <= 0) return;
    dim3 grid((unsigned)a.ntrials, (unsigned)nbeam);
    sps_kernel<<<grid, kSpsThreads, 0, st>>>(a);
}

}  // namespace spt
