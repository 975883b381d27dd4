// cutout.cu -- candidate cut-outs (Eq. 4; reading H): the two features the classifier is fed,
// the dedispersed dynamic spectrum at the candidate's DM and a DM transform over a narrow range around it, as exact integers.
//   dds[f][j] = sum_{c in band f} sum_{m<tbin} x[c][ts + j*tbin + m + delay(dm0, c)]
//   dmt[i][j] = sum_c            sum_{m<tbin} x[c][ts + j*tbin + m + delay(DM_i, c)],   DM_i = (dm0 - ddm) + i*step
// Samples outside the data count as 0.  A cut-out is small (256 x 256 outputs over 4096 channels): a delay table made on
// the device with the plan's formula, then one thread per output walking the channels.
#include <cuda_runtime.h>

#include "kernels.h"

namespace spt {

// row i < ndm: DM_i; row ndm: dm0 (for the dynamic spectrum).  Same expression, same order as build_plan (no contraction).
__global__ void cutout_delay_kernel(int32_t* __restrict__ delay, int32_t nchan, int32_t ndm, double fch1, double foff,
                                    double tsamp, double dm0, double ddm, double step) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = blockIdx.y;
    if (c >= nchan) return;
    const double dm = i < ndm ? (dm0 - ddm) + (double)i * step : dm0;
    const double f = fch1 + (double)c * foff;
    const double inv_top = 1.0 / (fch1 * fch1);
    const double seconds = kDispersionConstantS * dm * (1.0 / (f * f) - inv_top);
    delay[(size_t)i * nchan + c] = (int32_t)floor(seconds / tsamp + 0.5);
}

// grid (time blocks, rows): rows 0..ndm-1 are DM-transform rows over all channels, rows ndm..ndm+nf-1 spectrum bands
__global__ void cutout_sum_kernel(const uint8_t* __restrict__ x, int32_t nchan, int64_t nsamp, const int32_t* __restrict__ delay,
                                  int32_t ndm, int32_t nf, int64_t ts, int32_t tbin, int32_t nt, int32_t* __restrict__ dds,
                                  int32_t* __restrict__ dmt) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int r = blockIdx.y;
    if (j >= nt) return;
    const bool band = r >= ndm;
    const int per = nchan / nf;
    const int c0 = band ? (r - ndm) * per : 0, c1 = band ? c0 + per : nchan;
    const int32_t* dl = delay + (size_t)(band ? ndm : r) * nchan;
    const int64_t base = ts + (int64_t)j * tbin;
    int32_t acc = 0;
    for (int c = c0; c < c1; ++c) {
        const uint8_t* row = x + (size_t)c * nsamp;
        const int64_t s0 = base + dl[c];
        for (int m = 0; m < tbin; ++m) {
            const int64_t s = s0 + m;
            if (s >= 0 && s < nsamp) acc += (int32_t)row[s];
        }
    }
    if (band) dds[(size_t)(r - ndm) * nt + j] = acc;
    else dmt[(size_t)r * nt + j] = acc;
}

int launch_cutout(const uint8_t* x, int32_t nchan, int64_t nsamp, double fch1, double foff, double tsamp, double dm0,
                  double ddm, int32_t ndm, int64_t ts, int32_t tbin, int32_t nt, int32_t nf, int32_t* dds, int32_t* dmt,
                  cudaStream_t st) {
    int32_t* delay = nullptr;
    if (cudaMallocAsync((void**)&delay, sizeof(int32_t) * (size_t)(ndm + 1) * nchan, st) != cudaSuccess) return -1;
    const double step = ndm > 1 ? (2.0 * ddm) / (double)(ndm - 1) : 0.0;
    cutout_delay_kernel<<<dim3((unsigned)((nchan + 127) / 128), (unsigned)(ndm + 1)), 128, 0, st>>>(delay, nchan, ndm, fch1, foff,
                                                                                                 tsamp, dm0, ddm, step);
    cutout_sum_kernel<<<dim3((unsigned)((nt + 127) / 128), (unsigned)(ndm + nf)), 128, 0, st>>>(x, nchan, nsamp, delay, ndm, nf, ts,
                                                                                              tbin, nt, dds, dmt);
    cudaFreeAsync(delay, st);
    return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace spt
