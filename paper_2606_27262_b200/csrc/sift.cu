// sift.cu -- candidate optimisation after the search (reading G): per beam DBSCAN in the
// (arrival time, DM) plane, the strongest member of every cluster, cuts on S/N, DM and width, anti-coincidence over beams.
// The lists at this stage are small (after peak filtering 10^2 - 10^4 per beam), so every step is a brute-force pass of one
// thread per candidate over the candidates of its beam: exact, order independent, a few launches.
#include <cuda_runtime.h>

#include "kernels.h"

namespace spt {

__device__ __forceinline__ bool sift_near(const SiftArgs& a, int64_t i, int64_t j) {
    const double dx = a.x[i] - a.x[j], dy = a.y[i] - a.y[j];
    return dx * dx + dy * dy <= a.eps2;                         // no contraction (--fmad=false): same doubles as the oracle
}

// core[i]: at least min_pts candidates of the beam (itself included) within eps
__global__ void sift_core_kernel(const SiftArgs a) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n) return;
    int cnt = 0;
    for (int64_t j = a.seg_lo[i]; j < a.seg_hi[i]; ++j) cnt += sift_near(a, i, j) ? 1 : 0;
    a.core[i] = cnt >= a.min_pts ? 1 : 0;
    a.parent[i] = (int32_t)i;
}

__device__ __forceinline__ int32_t sift_find(int32_t* parent, int32_t v) {
    while (true) {
        const int32_t p = parent[v];
        if (p == v) return v;
        const int32_t g = parent[p];
        if (g != p) parent[v] = g;                                // path halving; races only shorten paths
        v = p;
    }
}

// core candidates within eps of each other are one cluster: lock-free union-find, the smaller index becomes the root
__global__ void sift_union_kernel(const SiftArgs a) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n || !a.core[i]) return;
    for (int64_t j = a.seg_lo[i]; j < i; ++j) {
        if (!a.core[j] || !sift_near(a, i, j)) continue;
        int32_t u = (int32_t)i, v = (int32_t)j;
        while (true) {
            u = sift_find(a.parent, u);
            v = sift_find(a.parent, v);
            if (u == v) break;
            if (u < v) { const int32_t s = u; u = v; v = s; }    // u > v: hang u under v
            if (atomicCAS(&a.parent[u], u, v) == u) break;
        }
    }
}

__device__ __forceinline__ unsigned long long sift_key(float snr, int64_t i) {
    unsigned int b = __float_as_uint(snr);
    b = (b & 0x80000000u) ? ~b : (b | 0x80000000u);              // order-preserving map of floats to unsigned
    return ((unsigned long long)b << 32) | (unsigned long long)(0xffffffffu - (unsigned int)i);   // ties: smaller index
}

// member[i]: root of the cluster (core: its own; border: that of its strongest core neighbour; noise: -1); every member
// bids for its cluster's representative with (S/N, smaller index first)
__global__ void sift_member_kernel(const SiftArgs a) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n) return;
    int32_t m = -1;
    if (a.core[i]) m = sift_find(a.parent, (int32_t)i);
    else {
        unsigned long long best = 0ull;
        int64_t bj = -1;
        for (int64_t j = a.seg_lo[i]; j < a.seg_hi[i]; ++j)
            if (a.core[j] && sift_near(a, i, j)) {
                const unsigned long long k = sift_key(a.snr[j], j);
                if (bj < 0 || k > best) { best = k; bj = j; }
            }
        if (bj >= 0) m = sift_find(a.parent, (int32_t)bj);
    }
    a.member[i] = m;
    if (m >= 0) atomicMax(&a.rep[m], sift_key(a.snr[i], i));
}

// stage masks: representative of its cluster; then the cuts
__global__ void sift_select_kernel(const SiftArgs a) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n) return;
    const int32_t m = a.member[i];
    const bool k1 = m >= 0 && a.rep[m] == sift_key(a.snr[i], i);
    const bool k2 = k1 && (double)a.snr[i] >= a.snr_min && a.dm[i] >= a.dm_min && a.wsec[i] <= a.width_max_s;
    a.keep[i] = (k1 ? 1 : 0) | (k2 ? 2 : 0);
}

// anti-coincidence: survivors of more than fraction * nbeam distinct beams within the window of this one -> RFI
__global__ void sift_coinc_kernel(const SiftArgs a) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n || !(a.keep[i] & 2)) return;
    bool k3 = true;
    if (a.coinc_window_s > 0.0) {
        unsigned long long seen[kSiftMaxBeams / 64];
        for (int w = 0; w < kSiftMaxBeams / 64; ++w) seen[w] = 0ull;
        for (int64_t j = 0; j < a.n; ++j)
            if ((a.keep[j] & 2) && fabs(a.arrival[j] - a.arrival[i]) <= a.coinc_window_s)
                seen[a.beam[j] >> 6] |= 1ull << (a.beam[j] & 63);
        int nb = 0;
        for (int w = 0; w < kSiftMaxBeams / 64; ++w) nb += __popcll(seen[w]);
        k3 = !((double)nb > a.coinc_beam_fraction * (double)a.nbeam);
    }
    if (k3) a.keep[i] |= 4;
}

void launch_sift(const SiftArgs& a, cudaStream_t st) {
    if (a.n <= 0) return;
    const unsigned nb = (unsigned)((a.n + 127) / 128);
    sift_core_kernel<<<nb, 128, 0, st>>>(a);
    sift_union_kernel<<<nb, 128, 0, st>>>(a);
    sift_member_kernel<<<nb, 128, 0, st>>>(a);
    sift_select_kernel<<<nb, 128, 0, st>>>(a);
    sift_coinc_kernel<<<nb, 128, 0, st>>>(a);
}

}  // namespace spt
