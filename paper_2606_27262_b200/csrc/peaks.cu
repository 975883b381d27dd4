// peaks.cu -- peak filtering of the candidate plane (reading E): "Peaks are filtered out by
// sliding a window across the candidates in the DM-time plane.  From each window, the peak with the highest S/N is
// picked, and all others are rejected.  Two different stencils are used: a 3x3 window, and an 11x11 window."
//
// The candidate list of the last search is sparse in the (trial, t) plane, so the plane is a lookup table, not an
// image: plane[beam][offset[trial] + t] = 1 + index of the candidate in the list (0 = none), laid out like the DM
// transform.  One thread per candidate walks its window (same beam, same DM range, inside each row's valid length)
// and dies if a live neighbour is stronger: larger S/N, or equal S/N and smaller (trial, t).  Stencils run one after
// the other on the survivors; the survivors are appended (warp aggregated) to the peak list, and the plane entries are
// cleared again so that the table stays all-zero between calls.
#include <cuda_runtime.h>

#include "kernels.h"

namespace spt {

__global__ void peaks_scatter_kernel(const PeakArgs a, uint32_t value_or_clear) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n) return;
    const spt_candidate c = a.cand[i];
    a.plane[(int64_t)c.beam * a.beam_stride + a.offset[c.trial] + c.t] = value_or_clear ? (uint32_t)(i + 1) : 0u;
}

__global__ void peaks_stencil_kernel(const PeakArgs a, int32_t h, const uint8_t* __restrict__ alive_in,
                                     uint8_t* __restrict__ alive_out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n) return;
    if (alive_in && !alive_in[i]) { alive_out[i] = 0; return; }
    const spt_candidate c = a.cand[i];
    const int32_t d_lo = max(c.trial - h, a.range_lo[c.trial]), d_hi = min(c.trial + h, a.range_hi[c.trial]);
    const uint32_t* pl = a.plane + (int64_t)c.beam * a.beam_stride;
    bool beaten = false;
    for (int32_t dd = d_lo; dd <= d_hi && !beaten; ++dd) {
        const int32_t t_lo = max(c.t - h, 0), t_hi = min(c.t + h, a.nout[dd] - 1);
        const uint32_t* row = pl + a.offset[dd];
        for (int32_t tt = t_lo; tt <= t_hi; ++tt) {
            const uint32_t j1 = row[tt];
            if (j1 == 0u || (int64_t)(j1 - 1u) == i) continue;
            const int64_t j = (int64_t)(j1 - 1u);
            if (alive_in && !alive_in[j]) continue;
            const float sj = a.cand[j].snr;             // (trial, t) of j are (dd, tt)
            if (sj > c.snr || (sj == c.snr && (dd < c.trial || (dd == c.trial && tt < c.t)))) { beaten = true; break; }
        }
    }
    alive_out[i] = beaten ? 0 : 1;
}

__global__ void peaks_compact_kernel(const PeakArgs a, const uint8_t* __restrict__ alive, spt_candidate* __restrict__ out,
                                     unsigned long long* __restrict__ out_count, long long out_capacity) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool keep = i < a.n && alive[i];
    const unsigned m = __ballot_sync(0xffffffffu, keep);
    if (!m) return;
    const int lane = threadIdx.x & 31;
    unsigned long long slot0 = 0;
    if (lane == 0) slot0 = atomicAdd(out_count, (unsigned long long)__popc(m));
    slot0 = __shfl_sync(0xffffffffu, slot0, 0);
    if (keep) {
        const long long slot = (long long)(slot0 + __popc(m & ((1u << lane) - 1u)));
        if (slot < out_capacity) out[slot] = a.cand[i];
    }
}

static unsigned blocks_for(int64_t n) { return (unsigned)((n + 255) / 256); }

void launch_peaks_scatter(const PeakArgs& a, bool set, cudaStream_t st) {
    if (a.n > 0) peaks_scatter_kernel<<<blocks_for(a.n), 256, 0, st>>>(a, set ? 1u : 0u);
}
void launch_peaks_stencil(const PeakArgs& a, int32_t window, const uint8_t* alive_in, uint8_t* alive_out, cudaStream_t st) {
    if (a.n > 0) peaks_stencil_kernel<<<blocks_for(a.n), 256, 0, st>>>(a, (window - 1) / 2, alive_in, alive_out);
}
void launch_peaks_compact(const PeakArgs& a, const uint8_t* alive, spt_candidate* out, unsigned long long* out_count,
                          long long out_capacity, cudaStream_t st) {
    if (a.n > 0) peaks_compact_kernel<<<blocks_for(a.n), 256, 0, st>>>(a, alive, out, out_count, out_capacity);
}

}  // namespace spt
