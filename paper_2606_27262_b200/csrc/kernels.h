// kernels.h -- launchers of the CUDA kernels (dedisperse.cu, sps.cu, probe.cu).  Not part of the ABI.
#pragma once

#include <cuda_runtime.h>

#include "internal.h"

namespace spt {

void launch_decimate(const uint8_t* x, int64_t in_row_stride, int64_t in_beam_stride, uint16_t* y,
                     int64_t out_row_stride, int64_t out_beam_stride, int32_t nchan, int32_t nbeam, int64_t nsamp_k,
                     int32_t k, cudaStream_t st);
void launch_max_u16(const uint16_t* x, int64_t nelem, uint32_t* maxval, cudaStream_t st);
void launch_max_u8(const uint8_t* x, int64_t nbytes, uint32_t* maxval, cudaStream_t st);

template <typename T>
void launch_dedisp_naive(const T* y, int64_t row_stride, int64_t beam_stride, const int32_t* d_delay,
                         const int32_t* d_nout, const int64_t* d_offset, int32_t nchan, int32_t ndm, int32_t nbeam,
                         int32_t max_nout, int32_t* out, int64_t out_beam_stride, cudaStream_t st);

int launch_dedisp_tiled(bool is_u16, int DT, const void* in, int64_t row_stride, int64_t beam_stride, int32_t* out,
                        int64_t out_beam_stride, const TileDesc* tiles, const StageIndex* sidx, const RowDesc* rows,
                        const uint32_t* blob, const uint32_t* maxval, const int32_t* skew, int32_t skew_max, int32_t vcap_words,
                        const int32_t* nout, const int64_t* offset,
                        int32_t ntile_dm, int32_t ntile_t, int32_t nbeam, cudaStream_t st);

struct SpsArgs {
    const int32_t* dmt;
    int64_t beam_stride;            // int32 elements per beam
    const int32_t* nout;            // [ntrials] global trial index
    const int64_t* offset;          // [ntrials]
    int32_t ntrials;
    int32_t nw;
    int32_t widths[kMaxWidths];
    double threshold;
    int64_t* sum;                   // [nbeam][ntrials]
    unsigned long long* sumsq;      // [nbeam][ntrials]
    spt_candidate* cand;
    unsigned long long* count;      // exact number found (may exceed capacity)
    long long capacity;
    const int32_t* win_len;         // [ntrials] or NULL: search only the last win_len[d] samples of row d ...
    const int32_t* win_starts;      // [ntrials] or NULL: ... and report only the first win_starts[d] start positions
};
void launch_sps(const SpsArgs& a, int32_t nbeam, cudaStream_t st);

struct PeakArgs {
    const spt_candidate* cand;      // the list of the last search
    int64_t n;                      // records in it
    uint32_t* plane;                // [nbeam][beam_stride] lookup table, all zero between calls
    int64_t beam_stride;
    const int32_t* nout;            // [ntrials]
    const int64_t* offset;          // [ntrials]
    const int32_t* range_lo;        // [ntrials] first / last trial of the trial's DM range
    const int32_t* range_hi;
};
void launch_peaks_scatter(const PeakArgs& a, bool set, cudaStream_t st);
void launch_peaks_stencil(const PeakArgs& a, int32_t window, const uint8_t* alive_in, uint8_t* alive_out, cudaStream_t st);
void launch_peaks_compact(const PeakArgs& a, const uint8_t* alive, spt_candidate* out, unsigned long long* out_count,
                          long long out_capacity, cudaStream_t st);

void launch_corner_turn(const uint8_t* in, int32_t nbeam, int64_t nsamp, int32_t nchan, int32_t flip, uint8_t* out,
                        int64_t out_row_stride, int64_t out_beam_stride, int64_t out_t0, cudaStream_t st);
void launch_keep_history(const uint8_t* src, uint8_t* dst, int64_t row_bytes, int64_t shift_bytes, int64_t keep_bytes,
                         int64_t nrows, cudaStream_t st);

int run_probe(int kind, int reps, double* warp_instr_per_s, double* elapsed_ms);

}  // namespace spt
