// peaks.cu -- peak filtering of the candidate plane (reading E): "Peaks are filtered out by
// sliding a window across the candidates in the DM-time plane.  From each window, the peak with the highest S/N is
// picked, and all others are rejected.  Two different stencils are used: a 3x3 window, and an 11x11 window."
//
// One thread per candidate walks its window (same beam, same DM range, inside each row's valid length) and dies if a live
// neighbour is stronger: larger S/N, or equal S/N and smaller (trial, t).  What it needs of a neighbour is the S/N at a
// (beam, trial, t) cell; the lookup structure holds exactly that, the float bits of the live candidates' S/N:
//   sparse lists (the paper's regime, 1e3-1e6 candidates per beam): an open-addressing hash table keyed by the cell number,
//     two slots per candidate -- memory follows the list, not the DM transform;
//   dense lists (unmitigated RFI: a third of all cells above threshold): a dense plane laid out like the DM transform, for
//     a slice of beams at a time, so that its size is bounded whatever max_beams is.
// The stencils run one after the other: after each, the cells of the candidates it removed are marked empty, so the next
// one sees survivors only.  Survivors are appended (warp aggregated) to the peak list.
#include <cuda_runtime.h>

#include "kernels.h"

namespace spt {

constexpr uint32_t kNoCand = 0xffffffffu;                 // a NaN pattern: no S/N has it
constexpr unsigned long long kEmptyKey = ~0ull;

__device__ __forceinline__ uint64_t peaks_hash(uint64_t k) {   // splitmix64 finaliser
    k ^= k >> 30; k *= 0xbf58476d1ce4e5b9ull;
    k ^= k >> 27; k *= 0x94d049bb133111ebull;
    k ^= k >> 31;
    return k;
}

__device__ __forceinline__ bool in_slice(const PeakArgs& a, int32_t beam) {
    return a.hkeys != nullptr || (beam >= a.beam0 && beam < a.beam0 + a.nbeam_slice);
}

// slot of the cell in the lookup structure: dense -> index in the plane; hash -> slot holding the key (or the first empty
// slot of its probe sequence when the key is absent)
__device__ __forceinline__ uint64_t find_slot(const PeakArgs& a, int32_t beam, int64_t cell, bool* present) {
    if (a.hkeys == nullptr) {
        *present = true;
        return (uint64_t)((int64_t)(beam - a.beam0) * a.beam_stride + cell);
    }
    const unsigned long long key = (unsigned long long)((int64_t)beam * a.beam_stride + cell);
    uint64_t h = peaks_hash(key) & a.hmask;
    for (;;) {
        const unsigned long long k = a.hkeys[h];
        if (k == key) { *present = true; return h; }
        if (k == kEmptyKey) { *present = false; return h; }
        h = (h + 1) & a.hmask;
    }
}

// put the candidates of the slice into the lookup structure (value = float bits of their S/N)
__global__ void peaks_insert_kernel(const PeakArgs a) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n) return;
    const spt_candidate c = a.cand[i];
    if (!in_slice(a, c.beam)) return;
    const int64_t cell = a.offset[c.trial] + c.t;
    if (a.hkeys == nullptr) {
        a.vals[(int64_t)(c.beam - a.beam0) * a.beam_stride + cell] = __float_as_uint(c.snr);
        return;
    }
    const unsigned long long key = (unsigned long long)((int64_t)c.beam * a.beam_stride + cell);
    uint64_t h = peaks_hash(key) & a.hmask;
    for (;;) {                                                     // keys are unique: (beam, trial, t) occurs once in the list
        const unsigned long long old = atomicCAS(a.hkeys + h, kEmptyKey, key);
        if (old == kEmptyKey) { a.vals[h] = __float_as_uint(c.snr); return; }
        h = (h + 1) & a.hmask;
    }
}

__global__ void peaks_stencil_kernel(const PeakArgs a, int32_t h, const uint8_t* __restrict__ alive_in,
                                     uint8_t* __restrict__ alive_out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n) return;
    const spt_candidate c = a.cand[i];
    if (!in_slice(a, c.beam)) return;
    if (alive_in && !alive_in[i]) { alive_out[i] = 0; return; }
    const int32_t d_lo = max(c.trial - h, a.range_lo[c.trial]), d_hi = min(c.trial + h, a.range_hi[c.trial]);
    bool beaten = false;
    for (int32_t dd = d_lo; dd <= d_hi && !beaten; ++dd) {
        const int32_t t_lo = max(c.t - h, 0), t_hi = min(c.t + h, a.nout[dd] - 1);
        const int64_t row = a.offset[dd];
        for (int32_t tt = t_lo; tt <= t_hi; ++tt) {
            if (dd == c.trial && tt == c.t) continue;
            bool present;
            const uint64_t slot = find_slot(a, c.beam, row + tt, &present);
            if (!present) continue;
            const uint32_t v = a.vals[slot];
            if (v == kNoCand) continue;                                // no candidate there, or one a previous stencil removed
            const float sj = __uint_as_float(v);
            if (sj > c.snr || (sj == c.snr && (dd < c.trial || (dd == c.trial && tt < c.t)))) { beaten = true; break; }
        }
    }
    alive_out[i] = beaten ? 0 : 1;
}

// after a stencil: the cells of the candidates it removed (mode 0), or of every candidate of the slice (mode 1: the dense
// plane is left all-empty for the next call), become empty
__global__ void peaks_erase_kernel(const PeakArgs a, const uint8_t* __restrict__ alive_before, const uint8_t* __restrict__ alive_after,
                                   int mode) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n) return;
    const spt_candidate c = a.cand[i];
    if (!in_slice(a, c.beam)) return;
    if (mode == 0 && !((alive_before == nullptr || alive_before[i]) && !alive_after[i])) return;
    bool present;
    const uint64_t slot = find_slot(a, c.beam, a.offset[c.trial] + c.t, &present);
    if (present) a.vals[slot] = kNoCand;
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

void launch_peaks_insert(const PeakArgs& a, cudaStream_t st) {
    if (a.n > 0) peaks_insert_kernel<<<blocks_for(a.n), 256, 0, st>>>(a);
}
void launch_peaks_stencil(const PeakArgs& a, int32_t window, const uint8_t* alive_in, uint8_t* alive_out, cudaStream_t st) {
    if (a.n > 0) peaks_stencil_kernel<<<blocks_for(a.n), 256, 0, st>>>(a, (window - 1) / 2, alive_in, alive_out);
}
void launch_peaks_erase(const PeakArgs& a, const uint8_t* alive_before, const uint8_t* alive_after, bool all, cudaStream_t st) {
    if (a.n > 0) peaks_erase_kernel<<<blocks_for(a.n), 256, 0, st>>>(a, alive_before, alive_after, all ? 1 : 0);
}
void launch_peaks_compact(const PeakArgs& a, const uint8_t* alive, spt_candidate* out, unsigned long long* out_count,
                          long long out_capacity, cudaStream_t st) {
    if (a.n > 0) peaks_compact_kernel<<<blocks_for(a.n), 256, 0, st>>>(a, alive, out, out_count, out_capacity);
}

}  // namespace spt
