// kernels.h -- launchers of the CUDA kernels (dedisperse.cu, sps.cu, probe.cu).  Not part of the ABI.
#pragma once

#include <cuda_runtime.h>

#include "internal.h"

namespace spt {

int sm_count();   // SMs of the current device (dedisperse.cu)

void launch_decimate(const uint8_t* x, int64_t in_row_stride, int64_t in_beam_stride, uint16_t* y,
                     int64_t out_row_stride, int64_t out_beam_stride, int32_t nchan, int32_t nbeam, int64_t nsamp_k,
                     int32_t k, uint32_t* maxval /* {largest, smallest} sample of the series, updated; may be NULL */, cudaStream_t st);
void launch_fill_row_pad_u8(uint8_t* x, int64_t pitch, int64_t nsamp, int64_t nrows, cudaStream_t st);
void launch_max_u16(const uint16_t* x, int64_t nelem, uint32_t* maxval, cudaStream_t st);
void launch_max_u8(const uint8_t* x, int64_t nbytes, uint32_t* maxval, cudaStream_t st);

template <typename T>
void launch_dedisp_naive(const T* y, int64_t row_stride, int64_t beam_stride, const int32_t* d_delay,
                         const int32_t* d_nout, const int64_t* d_offset, int32_t nchan, int32_t ndm, int32_t nbeam,
                         int32_t max_nout, int32_t* out, int64_t out_beam_stride, cudaStream_t st);

// One launch of the tiled dedispersion kernel (dedisperse.cu) over one series and one set of kernel tables.
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
    const uint32_t* maxval;    // {largest, smallest} input sample of this launch (device): bound the 16-bit lanes
    const int32_t* skew;       // [ntile_dm][DT] output skew of every trial of a DM tile
    int32_t skew_max;
    const int32_t* nout;       // range local
    const int64_t* offset;     // range local
    int32_t vcap_words, ntile_dm, ntile_t, nbeam;
    int32_t tail;              // > 0: only the last `tail` outputs of every row are computed (a pushed stream segment) ...
    int32_t tail_tiles;        // ... by this many time tiles per DM tile, counted back from the tile's last one
    const uint32_t* enable;    // NULL, or {flag, bias} (device): the launch runs only when flag == enable_want (a decimated
    uint32_t enable_want;      // range is enqueued on its 8-bit copy and on the uint16 series; the copy may not exist) and
                               // every channel summed owes `bias` (the floor the 8-bit copy was made with) when want == 1
};
int launch_dedisp_tiled(bool is_u16, int DT, int max_ent, int kh, const TiledArgs& a, cudaStream_t st);
// a decimated range in one launch: a8 = the 8-bit copy of the series (a8.enable -> {valid flag, bias}, a8.enable_want = 1), a16
// = the uint16 series (a16.enable = NULL); the block takes whichever the flag says
int launch_dedisp_dual(int DT, int max_ent, int kh, const TiledArgs& a8, const TiledArgs& a16, cudaStream_t st);
void launch_compact_u16(const uint16_t* y, uint8_t* c, int64_t nelem, const uint32_t* maxval, uint32_t* info, cudaStream_t st);

struct SpsArgs {
    const int32_t* dmt;
    int64_t beam_stride;            // int32 elements per beam
    const int32_t* nout;            // [ntrials] global trial index
    const int64_t* offset;          // [ntrials]
    int32_t ntrials;
    int32_t trial0, nlaunch;        // the launch searches the trials [trial0, trial0 + nlaunch)
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
    uint32_t* vals;                 // float bits of the live candidates' S/N (0xffffffff: none): dense plane cells or hash slots
    unsigned long long* hkeys;      // hash table keys (cell number over all beams), NULL: dense plane
    uint64_t hmask;                 // hash capacity - 1
    int64_t beam_stride;            // cells per beam (= DM-transform elements per beam)
    int32_t beam0, nbeam_slice;     // dense plane: the beams it covers in this pass
    const int32_t* nout;            // [ntrials]
    const int64_t* offset;          // [ntrials]
    const int32_t* range_lo;        // [ntrials] first / last trial of the trial's DM range
    const int32_t* range_hi;
};
void launch_peaks_insert(const PeakArgs& a, cudaStream_t st);
void launch_peaks_stencil(const PeakArgs& a, int32_t window, const uint8_t* alive_in, uint8_t* alive_out, cudaStream_t st);
void launch_peaks_erase(const PeakArgs& a, const uint8_t* alive_before, const uint8_t* alive_after, bool all, cudaStream_t st);
void launch_peaks_compact(const PeakArgs& a, const uint8_t* alive, spt_candidate* out, unsigned long long* out_count,
                          long long out_capacity, cudaStream_t st);

// peaks_static.cu: the hash-table filter with its working memory in a fixed block inside the library image (no allocation)
cudaError_t peaks_static_filter(PeakArgs a, const int32_t* windows, int32_t nwindows, spt_candidate* d_peaks,
                                unsigned long long* d_count, long long capacity, cudaStream_t st, int64_t* nlaunch);

void launch_corner_turn(const uint8_t* in, int32_t nbeam, int64_t nsamp, int32_t nchan, int32_t flip, int32_t spliced,
                        uint8_t* out, int64_t out_row_stride, int64_t out_beam_stride, int64_t out_t0, cudaStream_t st);
void launch_keep_history(const uint8_t* src, uint8_t* dst, int64_t row_bytes, int64_t shift_bytes, int64_t keep_bytes,
                         int64_t nrows, cudaStream_t st);

constexpr int kSiftMaxBeams = 1024;
struct SiftArgs {                   // all arrays DEVICE, n entries sorted by (beam, trial, t)
    int64_t n;
    int32_t nbeam, min_pts;
    double eps2, snr_min, dm_min, width_max_s, coinc_window_s, coinc_beam_fraction;
    const double* x;                // arrival time / time unit
    const double* y;                // DM / DM unit
    const double* dm;
    const double* wsec;             // width in seconds
    const double* arrival;          // seconds
    const float* snr;
    const int32_t* beam;
    const int64_t* seg_lo;          // [n] first / one-past-last candidate of the same beam
    const int64_t* seg_hi;
    int32_t* core;
    int32_t* parent;
    int32_t* member;
    unsigned long long* rep;        // [n] zeroed: best (S/N, index) key of the cluster rooted here
    int32_t* keep;                  // bit 0 after clustering, bit 1 after the cuts, bit 2 after anti-coincidence
};
void launch_sift(const SiftArgs& a, cudaStream_t st);

constexpr int kCutoutMaxCand = 96;   // candidates per launch: they travel in the kernel's parameter block (< 4 KB)
struct CutoutCand {
    double dm0, ddm;
    long long ts;
    int32_t tbin, beam;
    int32_t out, pad_;               // index of the candidate's outputs in dds / dmt
};
struct CutoutArgs {
    const uint8_t* x;                // [nbeam][nchan][nsamp]
    long long nsamp, beam_stride;
    double fch1, foff, tsamp;
    int32_t nchan, ndm, nt, nf, ncand;
    int32_t wcap, wstride, nsub;     // set by the launcher: window capacity (elements), row stride (words), channels staged at a time
    int32_t* dds;                    // [..][nf][nt]
    int32_t* dmt;                    // [..][ndm][nt]
    CutoutCand cand[kCutoutMaxCand];
};
int launch_cutout_batch(CutoutArgs& a, cudaStream_t st);

int run_probe(int kind, int reps, double* warp_instr_per_s, double* elapsed_ms);

}  // namespace spt
