/*
 * spt.h -- C ABI of libspt: the data-parallel hot path of the SPOTLIGHT real-time FRB search
 * (arxiv/paper_2606_27262) for NVIDIA B200 (sm_100a).
 *
 *   host-side delay plan  ->  time decimation  ->  brute-force incoherent dedispersion (DM transform)
 *   ->  boxcar single-pulse search  ->  candidate readback
 *
 * What each call computes is fixed by the paper (PAPER.md line numbers below) and, where the paper is
 * silent, by the readings listed in DESIGN.md section 2 (same letters as SURVEY.md section 8(c)).
 *
 * Conventions
 *   - plain pointers and sizes only; every pointer argument says HOST or DEVICE.
 *   - every call returns SPT_OK (0) or a negative spt_status; nothing throws, aborts or prints.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - spt_dedisperse / spt_single_pulse_search / spt_search only ENQUEUE work on that stream (internal side streams are
 *     forked from it and joined back into it before the call returns, so stream order holds for the caller);
 *     spt_candidates_*, spt_trial_stats and the *_host calls synchronise it.  One plan is used by one thread at a time.
 *   - the caller owns the filterbank and DM-transform device buffers; the library owns everything
 *     reachable from the plan (tables, decimated series, statistics, candidate list) until spt_plan_destroy.
 *   - there is no CPU fallback: a call that needs the GPU fails with SPT_ERR_CUDA when none is usable.
 */
#ifndef SPT_H_
#define SPT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    SPT_OK = 0,
    SPT_ERR_INVALID = -1,     /* null pointer, non-positive size, widths not strictly increasing, nbeam > max_beams ... */
    SPT_ERR_UNSUPPORTED = -2, /* foff >= 0 (band must be highest frequency first), decimation not a
                                 power of two or > 64, sums that would not fit the integer types (see spt_plan_create) */
    SPT_ERR_NOMEM = -3,       /* host or device allocation failed */
    SPT_ERR_CUDA = -4,        /* CUDA runtime error or no usable device; text via spt_last_error() */
    SPT_ERR_SHAPE = -5,       /* caller buffer too small / index out of range */
    SPT_ERR_STATE = -6        /* call order: e.g. search before any dedisperse, stats before a search */
} spt_status;

typedef struct spt_plan spt_plan; /* opaque, library owned */

/* One DM sub-range of the dedispersion plan ("the DM range is divided into sub-ranges, each
 * with its own DM step"): trials DM_i = dm_lo + i*dm_step, i in [0, ndm), searched on the input decimated in
 * time by `decim` (1 = full resolution; BASELINE.json north_star (3): "a time-decimation kernel for the
 * high-DM ranges").  Global trial index = concatenation of the ranges in the order given. */
typedef struct {
    double dm_lo;   /* pc cm^-3 */
    double dm_step; /* pc cm^-3, > 0 */
    int32_t ndm;    /* >= 1 */
    int32_t decim;  /* 1, 2, 4, ..., 64 */
} spt_dm_range;

/* One single-pulse candidate (boxcar matched filter, "all candidates above a threshold ... are
 * taken to the next stage").  t and width are in samples OF THE TRIAL'S OWN (decimated) rate. */
typedef struct {
    int32_t beam;
    int32_t trial; /* global trial index */
    int32_t t;     /* start sample of the boxcar */
    int32_t width; /* boxcar width that maximises S/N at t */
    float snr;
} spt_candidate;

/* -------------------------------------------------------------------------------------------------------
 * spt_plan_create -- a1 of SURVEY.md section 8(a): trial list, delay table, output geometry.  Host only: needs
 * no GPU (device buffers are created on first use).
 *
 *   f_c   = fch1_mhz + c*foff_mhz, c in [0, nchan); channel 0 is the highest frequency and the reference
 *           ("highest frequency in the observation band"); foff_mhz < 0 is required.
 *   delay[d][c] = floor( 4.148808e3 * DM_d * (f_c^-2 - f_0^-2) / (tsamp_s * decim) + 0.5 )      int32
 *           (Eq. 1-2; constant and "rounded to integer samples" per BASELINE.json north_star (2);
 *           evaluated in IEEE double, no FMA contraction)
 *   nout[d]     = max(0, floor(nsamp/decim) - delay[d][nchan-1])   valid output samples of trial d
 *   offset[d]   = start of row d inside one beam's DM transform, in int32 elements; rows are padded to a multiple
 *                 of 32 elements so that every row starts 128-byte aligned (padding is never written or read).
 *
 * widths: boxcar widths in samples of each trial's own rate, strictly increasing, >= 1 ("multiple
 * trial widths").  max_beams bounds nbeam of later calls.  cand_capacity = records the device candidate list
 * can hold (overflow is reported, not an error).
 * Unsupported (SPT_ERR_UNSUPPORTED): foff >= 0; decim not a power of two <= 64; nchan*255*decim >= 2^31 (int32
 * DM transform); widths[last]*nchan*255*decim >= 2^32 (boxcar sums are formed modulo 2^32);
 * floor(nsamp/decim)*(nchan*255*decim)^2 >= 2^64 for any range (the exact sum of squares of a row is kept in 64 bits).
 * ----------------------------------------------------------------------------------------------------- */
int spt_plan_create(double fch1_mhz, double foff_mhz, int32_t nchan, double tsamp_s, int64_t nsamp,
                    const spt_dm_range* ranges /*HOST*/, int32_t nranges,
                    const int32_t* widths /*HOST*/, int32_t nwidths,
                    int32_t max_beams, int64_t cand_capacity, spt_plan** out /*HOST*/);
int spt_plan_destroy(spt_plan* plan);

/* Sizing: number of trials over all ranges; int32 elements of ONE beam's DM transform (sum of padded rows). */
int spt_plan_info(const spt_plan* plan, int32_t* ntrials, int64_t* dmt_elems_per_beam);
/* Per-trial metadata (any out pointer may be NULL). */
int spt_plan_trial(const spt_plan* plan, int32_t trial, double* dm, int32_t* range, int32_t* decim,
                   int32_t* nout, int64_t* offset);
/* The delay-table row of one trial, host_out[nchan] (HOST) -- for the bit-exact delay-table parity. */
int spt_plan_delays(const spt_plan* plan, int32_t trial, int32_t* host_out);

/* Kernel-selection knobs, for A/B measurements and tests; must be set before the first spt_dedisperse.
 *   "dedisp_kernel": 0 = tiled shared-memory kernel (default, the product), 1 = one-thread-per-output kernel
 *                    reading global memory (bring-up / cross-check kernel, same results; it always computes whole rows,
 *                    also for spt_segment_push with whole_rows = 0)
 *   "group":         largest pre-summed channel group of the tiled kernel in channels: 1, 2, 4, 8, 12 or 16 (default: 8, or 16
 *                    where the cost model picks groups of 12 entries)
 *   "dm_tile":       trials per block tile (32 or 64; default 64)
 *   "skew":          1 (default) = every trial of a DM tile computes an output window shifted by its own delay at a
 *                    reference channel, which narrows the windows the tile reads; 0 = one window start per tile
 *   "profile":       1 = bracket every kernel launch with CUDA events on the caller's stream (see
 *                    spt_plan_kernel_times); may be switched at any time.  NOTE: it also changes the schedule -- with
 *                    profile = 1 the DM ranges run one after the other on the caller's stream (so that each launch can
 *                    be timed alone) instead of side by side on the library's side streams; results are identical, the
 *                    step is about 3 % slower.  Leave it 0 for production and for end-to-end timing.
 *   "max_entries":   largest pre-summed group of the tiled kernel in entries (a channel at one of its shifts): 8, 12 or 16;
 *                    default: chosen per DM range by the cost model
 *   "tile_words":    width of the tiled kernel's time tile in packed words (the tile is twice as many outputs): 224 or 256
 *                    (224 only with dm_tile = 64); default 0: chosen per DM range by the cost model together with the
 *                    entry cap
 *   "compact":       1 (default) = a decimated range is dedispersed from an 8-bit copy of its series (sample - smallest
 *                    sample) whenever the series spans fewer than 256 values -- decided on the device per call; 0 = always
 *                    from the uint16 series; same results
 *   "peaks_lookup":  how spt_peak_filter finds a neighbour's S/N: 0 (default) = by the density of the list, 1 = hash table
 *                    (memory follows the list), 2 = dense plane laid out like the DM transform (at most 4 GiB: a slice of
 *                    beams at a time), 3 = dense plane of one beam at a time; same results; may be switched at any time
 * Unknown names / values -> SPT_ERR_INVALID. */
int spt_plan_set_option(spt_plan* plan, const char* name, int64_t value);

/* Host-side view of the tables the tiled kernel runs on, for tests and reports; builds them
 * if needed, needs no GPU.  Per range: DM tiles, stages, channel groups and pre-summed variants over all tiles, time
 * tiles, and the largest shared-memory footprint (32-bit words) of a stage.  Any out pointer may be NULL.  The call also
 * bounds-checks every shared-memory address the kernel will form from the tables (variant stores, gather reads, the pre-sum's
 * raw loads incl. the words its aligned loads reach past a sample) and returns SPT_ERR_STATE if one leaves its region. */
int spt_plan_tiling_info(spt_plan* plan, int32_t range, int64_t* ntiles_dm, int64_t* nstages, int64_t* ngroups,
                         int64_t* nvariants, int64_t* ntiles_t, int64_t* max_stage_words);
/* Work of the kernel's pre-sum phase over all DM tiles of a range (one time tile each): warp tasks, entries processed by
 * them (the straight-line class size of each task's group), variants stored, and rounds of eight tasks -- what the entry
 * cap is chosen by, for reports.  Any out pointer may be NULL. */
int spt_plan_tiling_cost(spt_plan* plan, int32_t range, int64_t* ntasks, int64_t* task_entries, int64_t* task_variants,
                         int64_t* presum_rounds);
/* The kernel instance the plan chose for a range (by its cost model, or as the options fixed it): packed words per trial
 * per time tile (224 or 256), entry cap of a pre-summed group (8, 12 or 16), largest group in channels, and whether the
 * range has a second table set for the 8-bit copy of its decimated series.  For reports.  Any out pointer may be NULL. */
int spt_plan_tiling_choice(spt_plan* plan, int32_t range, int32_t* tile_words, int32_t* max_entries, int32_t* group,
                           int32_t* has_compact);
/* The delay row of one trial as the tiled kernel will apply it, reconstructed from those tables alone:
 * host_out[nchan] (HOST).  Must equal spt_plan_delays for every trial (checked by the CPU tests). */
int spt_plan_tiling_delays(spt_plan* plan, int32_t trial, int32_t* host_out);

/* -------------------------------------------------------------------------------------------------------
 * spt_dedisperse -- a2 + a3: time decimation of the ranges with decim > 1, then the DM transform
 *   y_k[b][c][j]  = sum_{m<k} x[b][c][k*j+m]                  uint16, j < floor(nsamp/k)   (decimation: a sum)
 *   out[b][d][t]  = sum_c y_k[b][c][t + delay[d][c]]          int32,  t in [0, nout[d])
 * ("shifting each channel ... by the appropriate time delay" and summing; the output is
 * the DM transform, one row per trial.)
 *   d_fb : DEVICE, uint8 [nbeam][nchan][nsamp], time contiguous, channel 0 = fch1 (highest frequency).
 *   d_dmt: DEVICE, int32, at least nbeam*dmt_elems_per_beam elements, 128-byte aligned; beam b's row d starts at
 *          b*dmt_elems_per_beam + offset[d].  Every element t < nout[d] of every row is written.
 * Enqueues on cuda_stream and returns.
 * SPT_ERR_UNSUPPORTED (from the first call, when the kernel tables are built): a tile of 64 consecutive trials whose
 * delays at one channel spread over more samples than the shared-memory tile holds (DM steps of several pc cm^-3 over a
 * wide, low band).  Options "dm_tile" = 32 halves the spread; "dedisp_kernel" = 1 takes any plan (slowly).
 * ----------------------------------------------------------------------------------------------------- */
int spt_dedisperse(spt_plan* plan, const uint8_t* d_fb, int32_t nbeam, int32_t* d_dmt, void* cuda_stream);

/* DEVICE pointer to the decimated series made by the last spt_dedisperse for range `range` (decim > 1):
 * uint16 [nbeam][nchan][nsamp_k].  Library owned; valid until the next spt_dedisperse / destroy.
 * For a range with decim == 1 returns *d_ptr = NULL and nsamp_k = nsamp. */
int spt_decimated(const spt_plan* plan, int32_t range, const uint16_t** d_ptr, int64_t* nsamp_k);
/* Row stride (elements) of that series: rows are padded to a multiple of 16 elements; beam stride = nchan*row_stride. */
int spt_decimated_stride(const spt_plan* plan, int32_t range, int64_t* row_stride);
/* Copy of one beam of that series without the row padding: host_out (HOST) uint16 [nchan][nsamp_k].  Synchronises. */
int spt_decimated_read(spt_plan* plan, int32_t range, int32_t beam, uint16_t* host_out);
/* Which form of that series the last spt_dedisperse read (read-only; for tests and reports).  A decimated series whose
 * samples span fewer than 256 values -- quantised noise does -- is dedispersed from an 8-bit copy (sample minus the smallest
 * sample of the series), decided on the device per call.  in_use = 1: the copy was made and read; floor_value = the smallest
 * sample, span = largest minus smallest.  in_use = 0: the uint16 series was read (or the range has no copy: decim == 1,
 * option "compact" = 0).  The results are the same either way.  Synchronises. */
int spt_decimated_compact(spt_plan* plan, int32_t range, int32_t* in_use, uint32_t* floor_value, uint32_t* span);

/* -------------------------------------------------------------------------------------------------------
 * spt_single_pulse_search -- a4 (readings C1-C5, D1 of DESIGN.md): per (beam, trial) with N = nout > 0
 *   Sx = sum x, Sxx = sum x^2 (exact integers);  mu = Sx/N;  sigma = sqrt((N*Sxx - Sx^2)/N^2)
 *   S_w[t]   = sum_{j<w} x[t+j]                              t in [0, N-w]
 *   snr_w[t] = (N*S_w[t] - w*Sx) / (N*sigma*sqrt(w))         (= (S_w - w*mu)/(sigma*sqrt(w)))
 *   best[t]  = max over widths w <= N-t, scanned in increasing w with strict '>' ; t in [0, N-widths[0]]
 *   a candidate {beam, trial, t, argmax width, best} is appended for every t with best[t] >= threshold.
 * sigma == 0 or N < 2: no candidates.  The list and the statistics of the previous search are discarded.
 * Order of the list is arbitrary.  Enqueues on cuda_stream and returns.
 * ----------------------------------------------------------------------------------------------------- */
int spt_single_pulse_search(spt_plan* plan, const int32_t* d_dmt /*DEVICE*/, int32_t nbeam, float threshold,
                            void* cuda_stream);

/* -------------------------------------------------------------------------------------------------------
 * spt_search -- a2 + a3 + a4 in one call: exactly spt_dedisperse(plan, d_fb, nbeam, d_dmt, stream) followed by
 * spt_single_pulse_search(plan, d_dmt, nbeam, threshold, stream) -- same arguments, same results (DM transform,
 * decimated series, statistics, candidate list up to its order) -- but enqueued so that a DM range is searched as soon
 * as its own rows of the DM transform are complete, while later ranges are still being dedispersed.  Work on
 * cuda_stream after this call sees everything finished.  The host-buffer calls (spt_search_host, spt_stream_push) use
 * the same schedule.
 * ----------------------------------------------------------------------------------------------------- */
int spt_search(spt_plan* plan, const uint8_t* d_fb /*DEVICE*/, int32_t nbeam, int32_t* d_dmt /*DEVICE*/, float threshold,
               void* cuda_stream);

/* Exact statistics of one (beam, trial) from the last search (synchronises).  n = nout. */
int spt_trial_stats(spt_plan* plan, int32_t beam, int32_t trial, int64_t* n, int64_t* sum, uint64_t* sumsq);
/* All of them at once: host arrays [nbeam*ntrials] (beam major), any may be NULL. */
int spt_trial_stats_all(spt_plan* plan, int32_t nbeam, int64_t* sum /*HOST*/, uint64_t* sumsq /*HOST*/);

/* a5 Candidate readback (both synchronise the stream of the last search).
 * total = exact number of candidates found (may exceed capacity); overflowed = 1 when records were dropped. */
int spt_candidates_count(spt_plan* plan, int64_t* total, int32_t* overflowed);
/* Copies min(total, capacity, cap) records to host_out (HOST); nwritten gets that number. */
int spt_candidates_read(spt_plan* plan, spt_candidate* host_out, int64_t cap, int64_t* nwritten);

/* -------------------------------------------------------------------------------------------------------
 * spt_peak_filter -- the stage after the search ("Peaks are filtered out by sliding a window across the
 * candidates in the DM-time plane.  From each window, the peak with the highest S/N is picked, and all others are
 * rejected.  Two different stencils are used: a 3x3 window, and an 11x11 window"; reading E).
 * Works on the candidate list of the last search (or of the batch popped last).  The plane of one beam and one DM
 * range has axes (trial, t); the window of odd size windows[i] is centred on each candidate in turn; a candidate is
 * kept iff no other live candidate of the same beam and range inside its window is stronger (larger snr field, or
 * equal snr and smaller (trial, t)).  The windows are applied one after the other on the survivors; {3, 11} is the
 * paper's pair.  windows: HOST, odd, 1..255, at most 8.  The candidate list itself is left untouched.
 * SPT_ERR_SHAPE if the list overflowed its capacity (an incomplete list cannot be filtered).  Waits for the search,
 * then enqueues on cuda_stream and returns.
 * spt_peaks_count / spt_peaks_read synchronise and return the survivors (order arbitrary).
 * ----------------------------------------------------------------------------------------------------- */
int spt_peak_filter(spt_plan* plan, const int32_t* windows /*HOST*/, int32_t nwindows, void* cuda_stream);
int spt_peaks_count(spt_plan* plan, int64_t* total);
int spt_peaks_read(spt_plan* plan, spt_candidate* host_out /*HOST*/, int64_t cap, int64_t* nwritten);

/* -------------------------------------------------------------------------------------------------------
 * spt_peak_filter_static -- the same filter (same rule, same tie-break) for callers that must not allocate
 * device memory: a real-time loop, where a cudaMalloc or cudaFree inside the library would stall every stream of the
 * device while it runs, and a process whose device memory is already owned by another allocator (a framework's pool
 * that took the whole card, a fixed partition), where a library allocation fails or eats into someone else's budget.
 * spt_peak_filter grows its hash table and flag arrays with cudaMalloc; this call never calls cudaMalloc, cudaFree or
 * any routine that allocates.  Its working memory is a fixed 6.5 MiB block inside the library image, which every GPU
 * that loads libspt.so holds until the process exits -- hence the limit:
 *     n <= SPT_PEAKS_STATIC_MAX records; a longer list gets SPT_ERR_UNSUPPORTED (text via spt_last_error) and nothing
 *     is enqueued.
 * The caller passes input and output:
 *   d_cand   DEVICE, n records of a search made with THIS plan (beam >= 0, trial and t inside the plan's rows; the
 *            (beam, trial, t) of a record occurs once), e.g. copied from spt_candidates_read; not modified
 *   windows  HOST, as for spt_peak_filter
 *   d_peaks  DEVICE, room for n records: the survivors, order arbitrary
 *   d_count  DEVICE, one 64-bit word: set to the number of survivors
 * Enqueues on cuda_stream and returns; read d_count / d_peaks after synchronising that stream.  The plan's own peak
 * list (spt_peaks_count / spt_peaks_read) and candidate list are not touched.
 * SPT_ERR_STATE if the plan has not dedispersed or searched yet (that is where its device tables are made).
 * First call on a device: it looks up the block's device address (cudaGetSymbolAddress, which also makes the runtime
 *   load the library's device code if nothing did before); make that first call during set-up, before any stream
 *   capture.  Later calls on that device only launch kernels.
 * One block per device, shared by every call, plan and thread: it still holds the previous call's contents (the call
 *   clears what it needs first), and two calls that overlap on the GPU -- different streams, or different threads --
 *   race on it and give wrong survivors.  Order them (one stream, or events) yourself.
 * ----------------------------------------------------------------------------------------------------- */
#define SPT_PEAKS_STATIC_MAX 262144
int spt_peak_filter_static(spt_plan* plan, const spt_candidate* d_cand /*DEVICE*/, int64_t n, const int32_t* windows /*HOST*/,
                           int32_t nwindows, spt_candidate* d_peaks /*DEVICE*/, uint64_t* d_count /*DEVICE*/, void* cuda_stream);

/* -------------------------------------------------------------------------------------------------------
 * spt_search_host -- the whole path from HOST memory: H2D copy of h_fb (uint8 [nbeam][nchan][nsamp]; pinned
 * memory makes the copy asynchronous), spt_dedisperse + spt_single_pulse_search into a library-owned DM
 * transform, then the candidate count back to the host.  Synchronous.  Candidates are then read with
 * spt_candidates_read.  h_dmt (HOST, may be NULL): when given, receives the nbeam*dmt_elems_per_beam int32 DM transform.
 * ----------------------------------------------------------------------------------------------------- */
int spt_search_host(spt_plan* plan, const uint8_t* h_fb, int32_t nbeam, float threshold, int32_t* h_dmt,
                    int64_t* ncand, int32_t* overflowed);

/* -------------------------------------------------------------------------------------------------------
 * Streaming form of spt_search_host: a two-deep pipeline in which the H2D copy of one batch runs on the copy engine
 * while the kernels of the previous batch run (the search consumes a continuous stream of blocks).
 *   spt_stream_push: enqueue {H2D of h_fb, decimation, dedispersion, search, count readback} and return at once.
 *       h_fb (HOST, pinned for a truly asynchronous copy) must stay valid and unchanged until the matching pop.
 *       At most two batches may be in flight: a third push returns SPT_ERR_STATE.
 *   spt_stream_pop: wait for the OLDEST batch in flight; ncand / overflowed as in spt_search_host.  Until the next push
 *       (which reuses this batch's buffers), spt_candidates_read / spt_candidates_count / spt_trial_stats* refer to this
 *       batch, while the other batch keeps running (the two batches in flight have their own lists and statistics; the DM
 *       transform buffer is shared and not kept).  SPT_ERR_STATE if nothing is in flight.
 * Results are identical to spt_search_host on the same input.
 * ----------------------------------------------------------------------------------------------------- */
int spt_stream_push(spt_plan* plan, const uint8_t* h_fb /*HOST*/, int32_t nbeam, float threshold);
int spt_stream_pop(spt_plan* plan, int64_t* ncand, int32_t* overflowed);

/* -------------------------------------------------------------------------------------------------------
 * The step before the hot path for a continuous stream (blocks arrive time-major, the band is flipped to
 * highest frequency first; every segment is read with an overlap so that each DM trial has its full
 * sweep; reading F).
 *
 * spt_corner_turn: d_out[b][c'][t] = d_in(b, t, c), c' = flip ? nchan-1-c : c.   d_in DEVICE uint8, time-major:
 *   spliced = 0: [nbeam][nsamp][nchan] (one block per beam); spliced = 1: [nsamp][nbeam][nchan] (the beams of a host
 *   time-spliced sample by sample, as the telescope's rings hold them).  d_out DEVICE uint8
 *   [nbeam][nchan][nsamp] (what spt_dedisperse takes).  Needs no plan.  Enqueues.
 *
 * spt_segment_push: overlap-save.  The plan's nsamp is the length of a library-owned working buffer per channel row =
 *   history + new samples.  A push drops the oldest nnew samples of every row, appends the corner-turned new block
 *   (d_new DEVICE uint8, time-major, [nbeam][nnew][nchan] or, spliced = 1, [nnew][nbeam][nchan]; flip as above) and
 *   dedisperses the buffer into d_dmt in the layout of spt_dedisperse.  The buffer starts as zeros.  With
 *   nsamp - nnew >= min_history every trial d gains nnew/decim new outputs per push: the LAST nnew/decim of its nout[d]
 *   samples; the ones before them repeat outputs of earlier pushes.
 *     whole_rows = 1: every row is computed in full, exactly as spt_dedisperse would;
 *     whole_rows = 0: only what is new is computed -- the last nnew/decim + wmax - 1 outputs of every row (wmax = the
 *       widest boxcar; those wmax - 1 repeat the end of the previous push's row: they are the lead-in of the window
 *       spt_segment_search reads) -- and every other element of d_dmt is left as it was.  Per push that is
 *       nchan * sum_d (nnew/decim_d + wmax - 1) additions instead of nchan * sum_d nout[d].
 *   nnew must be a multiple of `granule` (16, or the largest decimation factor if larger) so that the shift keeps the
 *   decimation phase and the row alignment.  SPT_ERR_SHAPE when the history is shorter than min_history.  Enqueues on
 *   cuda_stream (the history copy runs on a side stream beside the corner turn and is joined before the dedispersion).
 * spt_segment_info: min_history = the longest sweep of the plan in raw samples, rounded up to the granule;
 *   min_history_search = the same plus (widest boxcar - 1) samples of the coarsest rate (what spt_segment_search needs).
 *
 * spt_segment_search: the single-pulse search of one pushed segment (readings C1-C5, D1 applied to a window).  For every
 *   trial d (decimation k, row length n = nout[d]) the window is the last L = nnew/k + wmax - 1 samples of the row; the
 *   statistics (N = L, Sx, Sxx) and S/N are those of the window; reported are the start positions in its first nnew/k
 *   samples -- exactly those for which every boxcar width fits in the data seen so far and that no earlier segment has
 *   reported -- so that consecutive segments report every start position of the stream exactly once.  Candidate t is
 *   the index inside the row (add the row's stream offset for an absolute time).  d_dmt: what spt_segment_push wrote.
 *   Needs nsamp - nnew >= min_history_search (else SPT_ERR_SHAPE).  Read-out calls as after spt_single_pulse_search.
 * ----------------------------------------------------------------------------------------------------- */
int spt_corner_turn(const uint8_t* d_in /*DEVICE*/, int32_t nbeam, int64_t nsamp, int32_t nchan, int32_t flip, int32_t spliced,
                    uint8_t* d_out /*DEVICE*/, void* cuda_stream);
int spt_segment_info(const spt_plan* plan, int64_t* min_history, int64_t* min_history_search, int64_t* granule);
int spt_segment_search(spt_plan* plan, const int32_t* d_dmt /*DEVICE*/, int32_t nbeam, int64_t nnew, float threshold,
                       void* cuda_stream);
int spt_segment_push(spt_plan* plan, const uint8_t* d_new /*DEVICE*/, int32_t nbeam, int64_t nnew, int32_t flip, int32_t spliced,
                     int32_t whole_rows, int32_t* d_dmt /*DEVICE*/, void* cuda_stream);

/* -------------------------------------------------------------------------------------------------------
 * spt_sift -- candidate optimisation after the search (reading G), on a HOST list (typically
 * what spt_peaks_read returned for all beams of a batch):
 *   1 per beam, DBSCAN (Ester et al. 1996) in the plane (arrival time / time_unit_s, DM / dm_unit) with radius eps and
 *     min_pts points (the point itself included) for a core point (eps = 0.5, 5 points); a border point
 *     joins the cluster of its strongest core neighbour; out of each cluster the member with the highest snr (then the
 *     smaller (trial, t)) is kept, candidates in no cluster are rejected;
 *   2 cuts: rejected when snr < snr_min, DM < dm_min or width*decim*tsamp > width_max_s (10, 10, 0.1 s);
 *   3 anti-coincidence (off when coinc_window_s <= 0): rejected when survivors of more than
 *     coinc_beam_fraction * nbeam distinct beams (its own included) arrive within coinc_window_s of it.
 * Arrival time = t*decim*tsamp at the top of the band.  h_out (HOST, cap records) receives the survivors, order
 * arbitrary; stage_counts (HOST, 3 entries, may be NULL) the number left after each stage.  Synchronous; the plan only
 * supplies the trial table.  nbeam <= 1024.
 * ----------------------------------------------------------------------------------------------------- */
typedef struct {
    double eps;                 /* neighbourhood radius in plane units (paper: 0.5) */
    double time_unit_s;         /* seconds per plane unit of the time axis */
    double dm_unit;             /* pc cm^-3 per plane unit of the DM axis */
    int32_t min_pts;            /* paper: 5 */
    float snr_min;              /* paper: 10 */
    double dm_min;              /* paper: 10 pc cm^-3 */
    double width_max_s;         /* paper: 0.1 s */
    double coinc_window_s;      /* <= 0: no anti-coincidence stage */
    double coinc_beam_fraction; /* "a majority of the beams": 0.5 */
} spt_sift_params;
int spt_sift(spt_plan* plan, const spt_candidate* h_in /*HOST*/, int64_t n, int32_t nbeam, const spt_sift_params* params,
             spt_candidate* h_out /*HOST*/, int64_t cap, int64_t* nwritten, int64_t* stage_counts /*HOST[3]*/);

/* -------------------------------------------------------------------------------------------------------
 * spt_cutout -- the two classifier features of one candidate ("the dedispersed dynamic spectrum, and the DM
 * transform.  The former is created at the candidate's detected DM, while the latter is created at a narrow DM range
 * centred around that DM"; reading H), as exact integers:
 *   d_dds[f][j] = sum_{c in band f} sum_{m<tbin} x[c][ts + j*tbin + m + delay(dm0, c)]       int32 [nf][nt]
 *   d_dmt[i][j] = sum_c            sum_{m<tbin} x[c][ts + j*tbin + m + delay(DM_i, c)]        int32 [ndm][nt]
 *   DM_i = (dm0 - ddm) + i*(2*ddm)/(ndm-1); delay() as in spt_plan_create at full time resolution; band f = channels
 *   [f*nchan/nf, (f+1)*nchan/nf) (nf must divide nchan); samples outside [0, nsamp) count as 0 (ts may be negative).
 * d_fb: DEVICE uint8 [nchan][nsamp] of ONE beam.  Needs no plan.  Enqueues on cuda_stream.
 * spt_delta_dm: Eq. 4: sqrt(pi)/1382 * width_s * (1/snr_ratio) * nu_mhz^3 / bw_mhz -- the half-width of
 *   the DM range at which the S/N has dropped to snr_ratio (candies' default 0.1) of its peak.
 * ----------------------------------------------------------------------------------------------------- */
int spt_cutout(const uint8_t* d_fb /*DEVICE*/, int32_t nchan, int64_t nsamp, double fch1_mhz, double foff_mhz, double tsamp_s,
               double dm0, double ddm, int32_t ndm, int64_t ts, int32_t tbin, int32_t nt, int32_t nf,
               int32_t* d_dds /*DEVICE*/, int32_t* d_dmt /*DEVICE*/, void* cuda_stream);
/* spt_cutout_batch -- the same two features for MANY candidates in one launch (10 to 100 candidates per beam
 * per block reach this stage; "custom, optimised GPU kernels").  d_fb: DEVICE uint8 [nbeam][nchan][nsamp];
 * h_cands: HOST array of ncand records {dm0, ddm, ts, tbin, beam}; ndm, nt, nf are common to the batch (the classifier's
 * input shape).  Outputs, DEVICE int32: d_dds [ncand][nf][nt], d_dmt [ncand][ndm][nt], candidate k at index k.  Same
 * definitions, argument checks and error codes as spt_cutout (which is a batch of one).  The records are copied into the
 * launch: h_cands may be reused as soon as the call returns.  Enqueues on cuda_stream; allocates nothing. */
typedef struct {
    double dm0;     /* the candidate's DM, pc cm^-3 */
    double ddm;     /* half-width of the DM range of the narrow DM transform (Eq. 4: spt_delta_dm) */
    int64_t ts;     /* first raw sample of the window at the top of the band (may be negative) */
    int32_t tbin;   /* raw samples per time bin, >= 1 */
    int32_t beam;   /* which beam of d_fb */
} spt_cutout_params;
int spt_cutout_batch(const uint8_t* d_fb /*DEVICE*/, int32_t nbeam, int32_t nchan, int64_t nsamp, double fch1_mhz, double foff_mhz,
                     double tsamp_s, const spt_cutout_params* h_cands /*HOST*/, int32_t ncand, int32_t ndm, int32_t nt, int32_t nf,
                     int32_t* d_dds /*DEVICE*/, int32_t* d_dmt /*DEVICE*/, void* cuda_stream);
double spt_delta_dm(double width_s, double snr_ratio, double nu_mhz, double bw_mhz);

/* With option "profile" = 1: device time (ms) of each kernel launched by the LAST spt_dedisperse and the LAST
 * spt_single_pulse_search, in launch order; kinds: 1 = decimate, 2 = dedisperse, 3 = single-pulse search; `range` is the
 * DM range the launch served (-1 for the search).  Synchronises.  Arrays (HOST) hold `cap` entries; n = entries written. */
int spt_plan_kernel_times(spt_plan* plan, int32_t cap, int32_t* kind, int32_t* range, double* ms, int32_t* n);

/* Number of kernel launches the library has enqueued through this plan since creation (bench bookkeeping). */
int spt_plan_launches(const spt_plan* plan, int64_t* launches);

/* Roofline probes: time `reps` launches of a register-only 32-bit integer-add loop
 * (kind 0: IADD3 chain on the ALU pipe, kind 1: IMAD chain on the FMA pipe, kind 2: both interleaved) or of a
 * conflict-free shared-memory load loop (kind 3: LDS.32, kind 4: LDS.128) on the current device and report warp
 * instructions per second.  Synchronous; uses its own stream. */
int spt_probe(int32_t kind, int32_t reps, double* warp_instr_per_s, double* elapsed_ms);

const char* spt_strerror(int code);
/* Text of the last CUDA error seen by this thread's calls ("" if none). */
const char* spt_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SPT_H_ */
