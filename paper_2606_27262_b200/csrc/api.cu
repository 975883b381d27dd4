// api.cu -- the C ABI of libspt (include/spt.h): argument checking, device state, launch sequencing.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>

#include "internal.h"
#include "kernels.h"

namespace spt {

static thread_local std::string g_last_error;

static int cuda_fail(cudaError_t e, const char* what) {
    g_last_error = std::string(what) + ": " + cudaGetErrorString(e);
    cudaGetLastError();  // clear the sticky-less error state
    return e == cudaErrorMemoryAllocation ? SPT_ERR_NOMEM : SPT_ERR_CUDA;
}
#define SPT_CUDA(call)                                             \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call);        \
    } while (0)

struct RangeDev {
    int32_t* delay = nullptr;       // only for the naive kernel
    TileDesc* tiles = nullptr;
    StageIndex* sidx = nullptr;
    RowDesc* rows = nullptr;
    uint32_t* blob = nullptr;
    int32_t* skew = nullptr;
    uint16_t* series = nullptr;     // decimated input [max_beams][nchan][stride_k] (decim > 1)
    // decim > 1: the 8-bit copy of the series (sample - smallest sample, made per call when the series spans < 256), its
    // kernel tables, and {largest value, 0, valid flag, smallest sample} written by the kernel that makes it
    uint8_t* series8 = nullptr;
    uint32_t* cinfo = nullptr;
    TileDesc* c_tiles = nullptr;
    StageIndex* c_sidx = nullptr;
    RowDesc* c_rows = nullptr;
    uint32_t* c_blob = nullptr;
    int32_t* c_skew = nullptr;
};

struct DeviceState {
    std::vector<RangeDev> r;
    int32_t* nout = nullptr;        // [ntrials]
    int64_t* offset = nullptr;      // [ntrials]
    uint32_t* maxval = nullptr;     // [nranges][2] largest and smallest sample of the series each range read last
    int32_t* range_lo = nullptr;    // [ntrials] first / last trial of the trial's DM range (peak filter)
    int32_t* range_hi = nullptr;
    // continuous stream (lazily allocated): two working buffers [max_beams][nchan][nsamp], the current one holds the last
    // nsamp samples of every channel row
    uint8_t* work[2] = {nullptr, nullptr};
    int work_cur = 0;
    cudaStream_t hist_stream = nullptr;  // the history copy of a push runs beside the corner turn of the new block
    cudaEvent_t hist_fork = nullptr, hist_join = nullptr;
    int32_t* win_len = nullptr;     // [ntrials] search window of a segment and the start positions it reports,
    int32_t* win_starts = nullptr;  // for the segment length win_nnew
    int64_t win_nnew = -1;
    // peak filter (lazily allocated): S/N lookup -- a hash table for sparse lists, a dense plane over a slice of beams for
    // dense ones --, live flags, peak list
    uint32_t* plane = nullptr;
    int32_t plane_beams = 0;        // beams the plane covers
    unsigned long long* hkeys = nullptr;
    uint32_t* hvals = nullptr;
    uint64_t hcap = 0;
    uint8_t* alive[2] = {nullptr, nullptr};
    int64_t alive_cap = 0;
    spt_candidate* peaks = nullptr;
    int64_t peaks_cap = 0;
    unsigned long long* peaks_count = nullptr;
    bool peaks_valid = false;
    // results of a search: statistics [max_beams][ntrials], candidate list, exact count.  Set 0 serves the plain calls;
    // the streaming calls (spt_stream_push/pop) alternate between set 0 and a lazily allocated set 1.
    struct SearchBufs {
        int64_t* sum = nullptr;
        unsigned long long* sumsq = nullptr;
        spt_candidate* cand = nullptr;
        unsigned long long* count = nullptr;
    } bufs[2];
    int cur = 0;                    // the set the read-out calls look at
    // streaming pipeline (two batches in flight)
    struct Slot {
        uint8_t* fb = nullptr;                  // device copy of the batch's filterbank
        unsigned long long* h_count = nullptr;  // pinned host word the count lands in
        cudaEvent_t copied = nullptr, done = nullptr;
        int32_t nbeam = 0;
        bool pending = false;
    } slot[2];
    int push_next = 0, pop_next = 0;
    cudaStream_t copy_stream = nullptr;
    // side streams for the DM ranges after the first (their grids fill the tail of the previous range's grid)
    cudaStream_t side[2] = {nullptr, nullptr};
    cudaEvent_t fork = nullptr, join[2] = {nullptr, nullptr};
    bool side_pending[2] = {false, false};   // side streams left un-joined by do_dedisperse(defer_join) for do_search
    cudaEvent_t wait_event = nullptr;   // when set, read-out calls wait for this event instead of the whole stream
    uint8_t* fb_pad = nullptr;      // aligned copy of an input whose rows are not 16-byte multiples
    int64_t fb_pad_stride = 0;
    uint8_t* h_fb = nullptr;        // spt_search_host: device copy of the host filterbank
    int32_t* h_dmt = nullptr;       // spt_search_host: library-owned DM transform
    cudaStream_t own_stream = nullptr;
    cudaStream_t last_stream = nullptr;     // stream of the last search / peak filter: what the read-out calls wait for
    cudaStream_t dedisp_stream = nullptr;   // stream of the last dedispersion (decimated series, launch timings)
    int32_t nbeam_dedisp = 0, nbeam_search = 0;
    bool searched = false;
    // option "profile": events around every launch of the last dedisperse [0] / search [1]
    struct Timed { int32_t kind, range; cudaEvent_t e0, e1; };
    std::vector<Timed> timed[2];
    std::vector<cudaEvent_t> event_pool;
};

static cudaEvent_t get_event(DeviceState* d) {   // nullptr when the driver cannot make another event
    cudaEvent_t e = nullptr;
    if (!d->event_pool.empty()) { e = d->event_pool.back(); d->event_pool.pop_back(); }
    else if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); e = nullptr; }
    return e;
}
static void timed_clear(DeviceState* d, int slot) {
    for (auto& t : d->timed[slot]) { d->event_pool.push_back(t.e0); d->event_pool.push_back(t.e1); }
    d->timed[slot].clear();
}
struct ScopedTimer {  // records e0 at construction and e1 at destruction when profiling is on
    DeviceState* d; cudaStream_t st; int slot; bool on;
    ScopedTimer(Plan* p, cudaStream_t s, int slot_, int kind, int range) : d(p->dev), st(s), slot(slot_), on(p->opt_profile != 0) {
        if (!on) return;
        DeviceState::Timed t{kind, range, get_event(d), get_event(d)};
        if (!t.e0 || !t.e1) {          // no event to be had: this launch goes untimed (it still runs)
            if (t.e0) d->event_pool.push_back(t.e0);
            if (t.e1) d->event_pool.push_back(t.e1);
            on = false;
            return;
        }
        cudaEventRecord(t.e0, st);
        d->timed[slot].push_back(t);
    }
    ~ScopedTimer() { if (on) cudaEventRecord(d->timed[slot].back().e1, st); }
};

template <typename T>
static int upload(T** dst, const std::vector<T>& src) {
    *dst = nullptr;
    if (src.empty()) return SPT_OK;
    SPT_CUDA(cudaMalloc((void**)dst, src.size() * sizeof(T)));
    SPT_CUDA(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return SPT_OK;
}

static void free_device(Plan* p) {
    DeviceState* d = p->dev;
    if (!d) return;
    for (RangeDev& r : d->r) {
        cudaFree(r.delay); cudaFree(r.tiles); cudaFree(r.sidx); cudaFree(r.rows); cudaFree(r.blob); cudaFree(r.skew);
        cudaFree(r.series);
        cudaFree(r.series8); cudaFree(r.cinfo); cudaFree(r.c_tiles); cudaFree(r.c_sidx); cudaFree(r.c_rows); cudaFree(r.c_blob);
        cudaFree(r.c_skew);
    }
    cudaFree(d->maxval); cudaFree(d->nout); cudaFree(d->offset); cudaFree(d->range_lo); cudaFree(d->range_hi);
    cudaFree(d->work[0]); cudaFree(d->work[1]); cudaFree(d->win_len); cudaFree(d->win_starts);
    cudaFree(d->plane); cudaFree(d->hkeys); cudaFree(d->hvals); cudaFree(d->alive[0]); cudaFree(d->alive[1]); cudaFree(d->peaks); cudaFree(d->peaks_count);
    for (auto& b : d->bufs) { cudaFree(b.sum); cudaFree(b.sumsq); cudaFree(b.cand); cudaFree(b.count); }
    for (auto& sl : d->slot) {
        cudaFree(sl.fb);
        if (sl.h_count) cudaFreeHost(sl.h_count);
        if (sl.copied) cudaEventDestroy(sl.copied);
        if (sl.done) cudaEventDestroy(sl.done);
    }
    cudaFree(d->fb_pad); cudaFree(d->h_fb); cudaFree(d->h_dmt);
    if (d->hist_stream) cudaStreamDestroy(d->hist_stream);
    if (d->hist_fork) cudaEventDestroy(d->hist_fork);
    if (d->hist_join) cudaEventDestroy(d->hist_join);
    if (d->own_stream) cudaStreamDestroy(d->own_stream);
    if (d->copy_stream) cudaStreamDestroy(d->copy_stream);
    for (int i = 0; i < 2; ++i) { if (d->side[i]) cudaStreamDestroy(d->side[i]); if (d->join[i]) cudaEventDestroy(d->join[i]); }
    if (d->fork) cudaEventDestroy(d->fork);
    timed_clear(d, 0); timed_clear(d, 1);
    for (cudaEvent_t e : d->event_pool) cudaEventDestroy(e);
    delete d;
    p->dev = nullptr;
}

static int alloc_search_bufs(Plan* p, DeviceState::SearchBufs& b) {
    const size_t n = (size_t)p->max_beams * p->ntrials;
    cudaError_t ce = cudaMalloc((void**)&b.sum, n * 8);
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&b.sumsq, n * 8);
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&b.count, 8);
    if (ce == cudaSuccess) ce = cudaMemset(b.count, 0, 8);
    if (ce == cudaSuccess && p->cand_capacity > 0)
        ce = cudaMalloc((void**)&b.cand, (size_t)p->cand_capacity * sizeof(spt_candidate));
    return ce == cudaSuccess ? SPT_OK : cuda_fail(ce, "search buffers");
}

// Every shared-memory address the kernel will form from one set of tables stays inside the region it belongs to: the variants
// inside the variant region, the gather's reads inside the variant they read, the pre-sum's raw loads (the last lane's, in
// the high half, including the words its aligned loads reach past the sample) inside the row that was staged for them.
// compute-sanitizer is not available on the GPU pool; this is the bounds check it would have made, done
// on the host for every stage of every tile.  es: bytes per element of the series the tables address.
static int check_tables(const Plan& p, const RangePlan& rp, int es) {
    const int DT = p.opt_dm_tile, kh = rp.kh;
    const int64_t rcap = kSmemDataBytes - (int64_t)rp.vcap_words * 4;
    if (rp.vcap_words <= 0 || rcap <= 0 || (kh != 224 && kh != 256)) return SPT_ERR_STATE;
    for (const TileDesc& td : rp.tiles)
        if (td.nstage < 1 || td.stage0 < 0 || (size_t)(td.stage0 + td.nstage) + 1 > rp.sidx.size() || td.ntrial < 1 || td.ntrial > DT)
            return SPT_ERR_STATE;
    for (size_t is = 0; is + 1 < rp.sidx.size(); ++is) {
        const StageIndex& si = rp.sidx[is];
        if (si.blob_words * 4u > (uint32_t)kBlobBytes || si.nrows > (uint32_t)kMaxStageRows || si.nrows < 1) return SPT_ERR_STATE;
        if ((size_t)si.blob_word0 + si.blob_words > rp.blob.size() || (size_t)si.row0 + si.nrows > rp.rows.size()) return SPT_ERR_STATE;
        const uint32_t* b = &rp.blob[si.blob_word0];
        const uint32_t ngrp = b[0];
        if (ngrp < 1 || ngrp > (uint32_t)kMaxStageGroups || b[3] + ngrp * (uint32_t)DT / 2 > si.blob_words) return SPT_ERR_STATE;
        int64_t raw_end = 0;
        for (uint32_t k = 0; k < si.nrows; ++k) {
            const RowDesc& r = rp.rows[si.row0 + k];
            if (r.nelem <= 0 || (r.nelem & 15) || (r.soff & 15) || (r.astart & 15) || r.chan < 0 || r.chan >= p.nchan) return SPT_ERR_STATE;
            raw_end = std::max<int64_t>(raw_end, (int64_t)r.soff + (int64_t)r.nelem * es);
        }
        if (raw_end > rcap) return SPT_ERR_STATE;
        const uint16_t* toff = reinterpret_cast<const uint16_t*>(b + b[3]);
        for (uint32_t g = 0; g < ngrp; ++g) {
            const uint32_t* gh = b + kBlobHdrWords + 4 * g;
            const int64_t vbase = gh[0] & 0xffffu, vlen = gh[1];
            const int nent = (int)(gh[2] & 0xffu), ntog = (int)((gh[2] >> 8) & 0xffu), ncorr = (int)((gh[2] >> 16) & 0xffu);
            const int nvar = (int)(gh[2] >> 24);
            if (vlen < kh || (vlen & 3) || nvar < 1 || nvar > kMaxVar || nent < 1 || nent > kMaxEnt || ntog > nent) return SPT_ERR_STATE;
            if (vbase + (int64_t)nvar * vlen > rp.vcap_words) return SPT_ERR_STATE;
            const uint32_t* cd = b + (gh[3] & 0xffffu);
            const uint32_t* vd = b + (gh[3] >> 16);
            const int cls = ent_class(nent);
            // the variants the pre-sum stores: whole variants of this group
            for (int k = 0; k <= ntog; ++k)
                if (vd[k] != 0xffffffffu && (vd[k] < vbase || (vd[k] - vbase) % vlen != 0 || (vd[k] - vbase) / vlen >= (uint32_t)nvar))
                    return SPT_ERR_STATE;
            for (int c = 0; c < ncorr; ++c) {
                const uint32_t dst = vd[chain_words(cls) + 2 * c];
                if (dst < vbase || (dst - vbase) % vlen != 0 || (dst - vbase) / vlen >= (uint32_t)nvar) return SPT_ERR_STATE;
            }
            // the gather: trial i reads kh words from its offset, inside one variant
            for (int i = 0; i < DT; ++i) {
                const int64_t rel = (int64_t)toff[g * DT + i] - vbase;
                if (rel < 0 || rel / vlen >= nvar || rel % vlen + kh > vlen) return SPT_ERR_STATE;
            }
            // the pre-sum's raw loads: the lane with the last four words (u0 = vlen - 4), low and high half
            for (int q = 0; q < cls; ++q) {
                const int64_t w0 = cd[2 * q] & 0x3ffffu;               // aligned word (uint8) / 8-byte unit (uint16) of sample u = 0
                const int64_t last = es == 1 ? w0 + (vlen - 4) + kh + 8 : w0 + 2 * (vlen - 4) + 2 * kh + 16;
                bool inside = false;
                for (uint32_t k = 0; k < si.nrows && !inside; ++k) {
                    const RowDesc& r = rp.rows[si.row0 + k];
                    inside = w0 >= r.soff && last <= (int64_t)r.soff + (int64_t)r.nelem * es;
                }
                if (!inside) return SPT_ERR_STATE;
            }
        }
    }
    return SPT_OK;
}

static int ensure_device(Plan* p) {
    if (p->dev) return SPT_OK;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDeviceCount");
    if (ndev < 1) { g_last_error = "no CUDA device"; return SPT_ERR_CUDA; }
    if (p->opt_kernel == 0 && !p->tiling_built) {
        const int rc = build_tiling(*p);
        if (rc != SPT_OK) return rc;
    }
    if (p->opt_kernel == 0) {
        // the tables go to the kernel only after the host-side bounds check of every shared-memory address they lead to
        // (there is no compute-sanitizer on the GPU pool to catch a table that is wrong for an untested plan shape)
        const char* skip = std::getenv("SPT_CHECK_TABLES");
        if (!(skip && skip[0] == '0'))
            for (size_t i = 0; i < p->ranges.size(); ++i) {
                if (p->ranges[i].tiles.empty()) continue;
                int rc = check_tables(*p, p->ranges[i], p->ranges[i].decim == 1 ? 1 : 2);
                if (rc == SPT_OK && i < p->compact.size() && !p->compact[i].tiles.empty()) rc = check_tables(*p, p->compact[i], 1);
                if (rc != SPT_OK) { g_last_error = "kernel tables of range " + std::to_string(i) + " fail the bounds check"; return rc; }
            }
    }
    DeviceState* d = new (std::nothrow) DeviceState();
    if (!d) return SPT_ERR_NOMEM;
    p->dev = d;
    d->r.resize(p->ranges.size());
    std::vector<int32_t> nout_all, lo_all, hi_all;
    std::vector<int64_t> off_all;
    int rc = SPT_OK;
    for (size_t i = 0; i < p->ranges.size() && rc == SPT_OK; ++i) {
        const RangePlan& rp = p->ranges[i];
        RangeDev& rd = d->r[i];
        nout_all.insert(nout_all.end(), rp.nout.begin(), rp.nout.end());
        off_all.insert(off_all.end(), rp.offset.begin(), rp.offset.end());
        lo_all.insert(lo_all.end(), (size_t)rp.ndm, rp.trial0);
        hi_all.insert(hi_all.end(), (size_t)rp.ndm, rp.trial0 + rp.ndm - 1);
        if (p->opt_kernel == 1) rc = upload(&rd.delay, rp.delay);
        else {
            if ((rc = upload(&rd.tiles, rp.tiles)) != SPT_OK) break;
            if ((rc = upload(&rd.sidx, rp.sidx)) != SPT_OK) break;
            if ((rc = upload(&rd.rows, rp.rows)) != SPT_OK) break;
            if ((rc = upload(&rd.blob, rp.blob)) != SPT_OK) break;
            if ((rc = upload(&rd.skew, rp.skew)) != SPT_OK) break;
        }
        if (rc == SPT_OK && rp.decim > 1) {
            const size_t bytes = (size_t)p->max_beams * p->nchan * rp.stride_k * sizeof(uint16_t);
            cudaError_t ce = cudaMalloc((void**)&rd.series, bytes);
            if (ce == cudaSuccess) ce = cudaMemset(rd.series, 0, bytes);
            if (ce != cudaSuccess) rc = cuda_fail(ce, "series alloc");
            if (rc == SPT_OK && p->opt_kernel == 0 && i < p->compact.size() && !p->compact[i].tiles.empty()) {
                const RangePlan& cp = p->compact[i];
                ce = cudaMalloc((void**)&rd.series8, bytes / 2);
                if (ce == cudaSuccess) ce = cudaMalloc((void**)&rd.cinfo, 4 * sizeof(uint32_t));
                if (ce != cudaSuccess) rc = cuda_fail(ce, "compact series alloc");
                if (rc == SPT_OK) rc = upload(&rd.c_tiles, cp.tiles);
                if (rc == SPT_OK) rc = upload(&rd.c_sidx, cp.sidx);
                if (rc == SPT_OK) rc = upload(&rd.c_rows, cp.rows);
                if (rc == SPT_OK) rc = upload(&rd.c_blob, cp.blob);
                if (rc == SPT_OK) rc = upload(&rd.c_skew, cp.skew);
            }
        }
    }
    if (rc == SPT_OK) rc = upload(&d->nout, nout_all);
    if (rc == SPT_OK) rc = upload(&d->offset, off_all);
    if (rc == SPT_OK) {
        cudaError_t ce = cudaMalloc((void**)&d->maxval, 2 * sizeof(uint32_t) * p->ranges.size());
        if (ce != cudaSuccess) rc = cuda_fail(ce, "maxval");
    }
    if (rc == SPT_OK) rc = upload(&d->range_lo, lo_all);
    if (rc == SPT_OK) rc = upload(&d->range_hi, hi_all);
    if (rc == SPT_OK) rc = alloc_search_bufs(p, d->bufs[0]);
    if (rc == SPT_OK) {
        cudaError_t ce = cudaStreamCreateWithFlags(&d->own_stream, cudaStreamNonBlocking);
        if (ce != cudaSuccess) rc = cuda_fail(ce, "plan stream");
    }
    if (rc == SPT_OK) {
        // the zero fills above ran on the legacy default stream, which non-blocking streams (every torch.cuda.Stream) do not
        // wait for: they must have landed before the first launch on such a stream
        cudaError_t ce = cudaStreamSynchronize(cudaStreamLegacy);
        if (ce != cudaSuccess) rc = cuda_fail(ce, "plan set-up");
    }
    if (rc != SPT_OK) free_device(p);
    return rc;
}

// defer_join: leave the side streams un-joined (d->side_pending says which carry work); the caller -- do_search with
// per_range = true, directly afterwards -- enqueues every range's search behind its dedispersion and joins then.
// tail_raw > 0 (a pushed stream segment of that many new raw samples): only the last tail_raw/decim + wmax - 1 outputs of
// every row are computed -- the window spt_segment_search reads -- and the rest of d_dmt is left alone.
static int do_dedisperse(Plan* p, const uint8_t* d_fb, int32_t nbeam, int32_t* d_dmt, cudaStream_t st,
                         bool defer_join = false, int64_t tail_raw = 0) {
    DeviceState* d = p->dev;
    const uint8_t* in = d_fb;
    int64_t in_stride = p->nsamp;
    if ((p->nsamp & 15) != 0 || (reinterpret_cast<uintptr_t>(d_fb) & 15) != 0) {
        // vector loads need 16-byte aligned rows: stage through a padded copy (zero pad)
        const int64_t pitch = (p->nsamp + 15) / 16 * 16;
        if (!d->fb_pad) {
            const size_t bytes = (size_t)p->max_beams * p->nchan * pitch;
            SPT_CUDA(cudaMalloc((void**)&d->fb_pad, bytes));
            SPT_CUDA(cudaMemsetAsync(d->fb_pad, 0, bytes, st));      // on st: ordered before the copy below on any stream
            d->fb_pad_stride = pitch;
        }
        SPT_CUDA(cudaMemcpy2DAsync(d->fb_pad, (size_t)pitch, d_fb, (size_t)p->nsamp, (size_t)p->nsamp,
                                   (size_t)nbeam * p->nchan, cudaMemcpyDeviceToDevice, st));
        // the row padding repeats the row's last sample: the bounds pass below scans whole rows, and padding zeros would
        // drag the smallest sample (the floor the packed lanes subtract) to 0 for every input like this one
        launch_fill_row_pad_u8(d->fb_pad, pitch, p->nsamp, (int64_t)nbeam * p->nchan, st);
        p->launches++;
        in = d->fb_pad;
        in_stride = pitch;
    }
    timed_clear(d, 0);
    // largest sample of every series (bounds the 16-bit lanes of the dedispersion)
    for (size_t i = 0; i < p->ranges.size(); ++i) {     // {largest, smallest} = {0, 0xffffffff}
        SPT_CUDA(cudaMemsetAsync(d->maxval + 2 * i, 0, 4, st));
        SPT_CUDA(cudaMemsetAsync(d->maxval + 2 * i + 1, 0xff, 4, st));
    }
    // Every range has a pre-pass (the bounds of a raw range, or its decimated series and their bounds: a2) and its
    // dedispersion (a3).  Unless launches are being timed one by one, the ranges after the first run on side streams:
    // they are independent, their HBM-bound pre-passes run beside the first range's dedispersion, and their
    // dedispersion grids fill the last, partly empty wave of the grid launched before them.
    const bool overlap = !p->opt_profile && p->ranges.size() > 1;
    if (overlap) {
        if (!d->fork) {
            SPT_CUDA(cudaEventCreateWithFlags(&d->fork, cudaEventDisableTiming));
            for (int i = 0; i < 2; ++i) {
                SPT_CUDA(cudaStreamCreateWithFlags(&d->side[i], cudaStreamNonBlocking));
                SPT_CUDA(cudaEventCreateWithFlags(&d->join[i], cudaEventDisableTiming));
            }
        }
        SPT_CUDA(cudaEventRecord(d->fork, st));                  // after the input staging and the resets above
        for (int i = 0; i < 2; ++i) SPT_CUDA(cudaStreamWaitEvent(d->side[i], d->fork, 0));
    }
    cudaStream_t const caller = st;
    bool used_side[2] = {false, false};
    auto stream_of = [&](size_t i) {
        if (overlap && i > 0) { used_side[(i - 1) & 1] = true; return d->side[(i - 1) & 1]; }
        return caller;
    };
    auto prepass = [&](size_t i) -> int {
        const RangePlan& rp = p->ranges[i];
        cudaStream_t s = stream_of(i);
        if (rp.decim == 1) {
            if (rp.max_nout <= 0) return SPT_OK;
            launch_max_u8(in, (int64_t)nbeam * p->nchan * in_stride, d->maxval + 2 * i, s);
            p->launches++;
            return SPT_OK;
        }
        if (rp.nsamp_k <= 0) return SPT_OK;
        ScopedTimer tm(p, s, 0, 1, (int)i);
        // The bounds of the series come from a pass of their own.  decimate_kernel can leave them as a by-product (pass maxval
        // instead of NULL), but measured on config 3 that is slower, 1.29 + 0.66 ms against 0.46 + 0.30 ms for the ranges' pre-passes:
        // two million warps each load the one running pair of bounds, and same-address loads serialise in one L2 slice.
        launch_decimate(in, in_stride, (int64_t)p->nchan * in_stride, d->r[i].series, rp.stride_k,
                        (int64_t)p->nchan * rp.stride_k, p->nchan, nbeam, rp.nsamp_k, rp.decim, nullptr, s);
        launch_max_u16(d->r[i].series, (int64_t)nbeam * p->nchan * rp.stride_k, d->maxval + 2 * i, s);
        p->launches += 2;
        if (d->r[i].series8) {               // the 8-bit copy, if the series spans less than 256 (decided on the device)
            launch_compact_u16(d->r[i].series, d->r[i].series8, (int64_t)nbeam * p->nchan * rp.stride_k, d->maxval + 2 * i,
                               d->r[i].cinfo, s);
            p->launches++;
        }
        return SPT_OK;
    };
    // launch order: the side streams' pre-passes, then the first range (pre-pass and grid), then the other grids
    for (size_t i = 1; i < p->ranges.size(); ++i) prepass(i);
    if (!p->ranges.empty()) prepass(0);
    for (size_t i = 0; i < p->ranges.size(); ++i) {
        const RangePlan& rp = p->ranges[i];
        if (rp.max_nout <= 0) continue;
        st = stream_of(i);
        const RangeDev& rd = d->r[i];
        const bool u16 = rp.decim > 1;
        const void* src = u16 ? (const void*)rd.series : (const void*)in;
        const int64_t rs = u16 ? rp.stride_k : in_stride;
        const int32_t* nout = d->nout + rp.trial0;
        const int64_t* off = d->offset + rp.trial0;
        ScopedTimer tm(p, st, 0, 2, (int)i);
        if (p->opt_kernel == 1) {
            if (u16) launch_dedisp_naive<uint16_t>((const uint16_t*)src, rs, (int64_t)p->nchan * rs, rd.delay, nout, off,
                                                   p->nchan, rp.ndm, nbeam, rp.max_nout, d_dmt, p->dmt_elems, st);
            else launch_dedisp_naive<uint8_t>((const uint8_t*)src, rs, (int64_t)p->nchan * rs, rd.delay, nout, off,
                                              p->nchan, rp.ndm, nbeam, rp.max_nout, d_dmt, p->dmt_elems, st);
        } else {
            int32_t tail = 0, tail_tiles = 0;
            if (tail_raw > 0) {
                // time tiles per DM tile, counted back from its last one, that hold the tail of some trial of the tile
                tail = (int32_t)std::min<int64_t>(tail_raw / rp.decim + p->widths.back() - 1, rp.max_nout);
                for (const TileDesc& td : rp.tiles) {
                    int32_t first = INT32_MAX;
                    for (int t = 0; t < td.ntrial; ++t) {
                        const int32_t n = rp.nout[td.trial0 + t];
                        if (n > 0) first = std::min(first, (std::max(0, n - tail) + rp.skew[(size_t)td.skew0 + t]) / (2 * rp.kh));
                    }
                    if (td.tt_last >= 0 && first != INT32_MAX) tail_tiles = std::max(tail_tiles, td.tt_last - first + 1);
                }
                if (tail_tiles <= 0) continue;
            }
            auto args_of = [&](const RangePlan& t, const void* series, const TileDesc* tiles, const StageIndex* sidx,
                               const RowDesc* rows, const uint32_t* blob, const int32_t* skew, const uint32_t* bounds) {
                TiledArgs a{};
                a.in = series; a.row_stride = rs; a.beam_stride = (int64_t)p->nchan * rs;
                a.out = d_dmt; a.out_beam_stride = p->dmt_elems;
                a.tiles = tiles; a.sidx = sidx; a.rows = rows; a.blob = blob; a.maxval = bounds; a.skew = skew;
                a.skew_max = t.skew_max; a.nout = nout; a.offset = off; a.vcap_words = t.vcap_words;
                a.ntile_dm = (int32_t)t.tiles.size(); a.ntile_t = t.ntile_t; a.nbeam = nbeam;
                a.tail = tail; a.tail_tiles = tail_tiles; a.enable = nullptr; a.enable_want = 0u;
                return a;
            };
            const TiledArgs a16 = args_of(rp, src, rd.tiles, rd.sidx, rd.rows, rd.blob, rd.skew, d->maxval + 2 * i);
            int rc;
            if (rd.series8) {
                // a decimated range runs on the 8-bit copy of its series, with the copy's tables, when the copy was made (the
                // device decided that just before), on the uint16 series otherwise: one launch, the blocks look at the flag
                const RangePlan& cp = p->compact[i];
                TiledArgs a8 = args_of(cp, rd.series8, rd.c_tiles, rd.c_sidx, rd.c_rows, rd.c_blob, rd.c_skew, rd.cinfo);
                a8.enable = rd.cinfo + 2; a8.enable_want = 1u;
                rc = launch_dedisp_dual(p->opt_dm_tile, rp.max_ent, rp.kh, a8, a16, st);
            } else {
                rc = launch_dedisp_tiled(u16, p->opt_dm_tile, rp.max_ent, rp.kh, a16, st);
            }
            if (rc != 0) { g_last_error = "dedisp_tiled: launch configuration rejected"; return SPT_ERR_CUDA; }
        }
        p->launches++;
    }
    st = caller;
    for (int i = 0; i < 2; ++i) {
        d->side_pending[i] = defer_join && used_side[i];
        if (used_side[i] && !defer_join) {                       // the caller's stream continues when every range is done
            SPT_CUDA(cudaEventRecord(d->join[i], d->side[i]));
            SPT_CUDA(cudaStreamWaitEvent(st, d->join[i], 0));
        }
    }
    SPT_CUDA(cudaGetLastError());
    d->last_stream = st;
    d->dedisp_stream = st;
    d->nbeam_dedisp = nbeam;
    return SPT_OK;
}

// The counter of the result set is reset on the caller's stream: before do_dedisperse forks when the two are fused.
static int reset_count(Plan* p, cudaStream_t st, int set) {
    SPT_CUDA(cudaMemsetAsync(p->dev->bufs[set].count, 0, 8, st));
    return SPT_OK;
}

// per_range (only right after do_dedisperse(..., defer_join = true), counter already reset): one launch per DM range on
// the stream that range was dedispersed on, so a range is searched while later ranges are still being dedispersed.
static int do_search(Plan* p, const int32_t* d_dmt, int32_t nbeam, float threshold, cudaStream_t st, int set = 0,
                     bool windowed = false, bool per_range = false) {
    DeviceState* d = p->dev;
    const DeviceState::SearchBufs& bf = d->bufs[set];
    if (!per_range) { const int rc0 = reset_count(p, st, set); if (rc0 != SPT_OK) return rc0; }
    SpsArgs a{};
    a.dmt = d_dmt;
    a.beam_stride = p->dmt_elems;
    a.nout = d->nout;
    a.offset = d->offset;
    a.ntrials = p->ntrials;
    a.nw = (int32_t)p->widths.size();
    for (int i = 0; i < a.nw; ++i) a.widths[i] = p->widths[i];
    a.threshold = (double)threshold;
    a.sum = bf.sum;
    a.sumsq = bf.sumsq;
    a.cand = bf.cand;
    a.count = bf.count;
    a.capacity = p->cand_capacity;
    a.win_len = windowed ? d->win_len : nullptr;
    a.win_starts = windowed ? d->win_starts : nullptr;
    timed_clear(d, 1);
    if (per_range && (d->side_pending[0] || d->side_pending[1])) {
        for (size_t i = 0; i < p->ranges.size(); ++i) {
            const RangePlan& rp = p->ranges[i];
            cudaStream_t s = (i > 0 && d->side_pending[(i - 1) & 1]) ? d->side[(i - 1) & 1] : st;
            a.trial0 = rp.trial0;
            a.nlaunch = rp.ndm;
            launch_sps(a, nbeam, s);
            p->launches++;
        }
        for (int i = 0; i < 2; ++i)
            if (d->side_pending[i]) {
                SPT_CUDA(cudaEventRecord(d->join[i], d->side[i]));
                SPT_CUDA(cudaStreamWaitEvent(st, d->join[i], 0));
                d->side_pending[i] = false;
            }
    } else {
        a.trial0 = 0;
        a.nlaunch = p->ntrials;
        ScopedTimer tm(p, st, 1, 3, -1);
        launch_sps(a, nbeam, st);
        p->launches++;
    }
    SPT_CUDA(cudaGetLastError());
    d->last_stream = st;
    d->nbeam_search = nbeam;
    d->searched = true;
    d->cur = set;
    d->wait_event = nullptr;
    d->peaks_valid = false;
    return SPT_OK;
}

// a2-a4 in one go: every range's search follows its own dedispersion on that range's stream.
static int do_path(Plan* p, const uint8_t* d_fb, int32_t nbeam, int32_t* d_dmt, float threshold, cudaStream_t st, int set) {
    int rc;
    if ((rc = reset_count(p, st, set)) != SPT_OK) return rc;
    if ((rc = do_dedisperse(p, d_fb, nbeam, d_dmt, st, true)) != SPT_OK) return rc;
    return do_search(p, d_dmt, nbeam, threshold, st, set, false, true);
}

// Read-out calls wait for the results they look at: the whole stream of the last plain call, or the completion event of the
// batch spt_stream_pop returned last (later batches may still be running).
static int sync_results(DeviceState* d) {
    if (d->wait_event) SPT_CUDA(cudaEventSynchronize(d->wait_event));
    else SPT_CUDA(cudaStreamSynchronize(d->last_stream));
    return SPT_OK;
}

}  // namespace spt

using namespace spt;

struct spt_plan {
    Plan p;
};

extern "C" {

int spt_plan_create(double fch1_mhz, double foff_mhz, int32_t nchan, double tsamp_s, int64_t nsamp,
                    const spt_dm_range* ranges, int32_t nranges, const int32_t* widths, int32_t nwidths,
                    int32_t max_beams, int64_t cand_capacity, spt_plan** out) {
    if (!out) return SPT_ERR_INVALID;
    *out = nullptr;
    if (!ranges || !widths || nranges < 1 || nwidths < 1 || nwidths > kMaxWidths || nchan < 1 || nsamp < 1 ||
        !(tsamp_s > 0.0) || !(fch1_mhz > 0.0) || max_beams < 1 || cand_capacity < 0)
        return SPT_ERR_INVALID;
    if (!(foff_mhz < 0.0)) return SPT_ERR_UNSUPPORTED;                       // band must be flipped
    if (!(fch1_mhz + (double)(nchan - 1) * foff_mhz > 0.0)) return SPT_ERR_INVALID;
    for (int32_t i = 0; i < nwidths; ++i)
        if (widths[i] < 1 || (i > 0 && widths[i] <= widths[i - 1])) return SPT_ERR_INVALID;
    int maxdec = 1;
    for (int32_t r = 0; r < nranges; ++r) {
        const spt_dm_range& g = ranges[r];
        if (g.ndm < 1 || !(g.dm_step > 0.0) || !(g.dm_lo >= 0.0) || g.decim < 1) return SPT_ERR_INVALID;
        if ((g.decim & (g.decim - 1)) != 0 || g.decim > 64) return SPT_ERR_UNSUPPORTED;
        if (g.decim > maxdec) maxdec = g.decim;
    }
    if ((double)nchan * 255.0 * maxdec >= 2147483648.0) return SPT_ERR_UNSUPPORTED;
    if ((double)widths[nwidths - 1] * nchan * 255.0 * maxdec >= 4294967296.0) return SPT_ERR_UNSUPPORTED;
    // Sxx = sum x^2 of a row is kept in 64 bits: a row of floor(nsamp/decim) samples of at most nchan*255*decim must fit
    for (int32_t r = 0; r < nranges; ++r) {
        const unsigned __int128 xmax = (unsigned __int128)nchan * 255u * (unsigned)ranges[r].decim;
        const unsigned __int128 worst = (unsigned __int128)(nsamp / ranges[r].decim) * xmax * xmax;
        if (worst >> 64) return SPT_ERR_UNSUPPORTED;
    }
    if (widths[nwidths - 1] > 4096 - 32) return SPT_ERR_UNSUPPORTED;
    if (nsamp >= (1ll << 31)) return SPT_ERR_UNSUPPORTED;
    spt_plan* h = new (std::nothrow) spt_plan();
    if (!h) return SPT_ERR_NOMEM;
    Plan& p = h->p;
    p.fch1 = fch1_mhz; p.foff = foff_mhz; p.tsamp = tsamp_s; p.nchan = nchan; p.nsamp = nsamp;
    p.max_beams = max_beams; p.cand_capacity = cand_capacity;
    p.widths.assign(widths, widths + nwidths);
    int rc;
    try {
        rc = build_plan(p, ranges, nranges);
    } catch (const std::bad_alloc&) {
        rc = SPT_ERR_NOMEM;
    }
    if (rc != SPT_OK) { delete h; return rc; }
    *out = h;
    return SPT_OK;
}

int spt_plan_destroy(spt_plan* plan) {
    if (!plan) return SPT_ERR_INVALID;
    free_device(&plan->p);
    delete plan;
    return SPT_OK;
}

int spt_plan_info(const spt_plan* plan, int32_t* ntrials, int64_t* dmt_elems_per_beam) {
    if (!plan) return SPT_ERR_INVALID;
    if (ntrials) *ntrials = plan->p.ntrials;
    if (dmt_elems_per_beam) *dmt_elems_per_beam = plan->p.dmt_elems;
    return SPT_OK;
}

int spt_plan_trial(const spt_plan* plan, int32_t trial, double* dm, int32_t* range, int32_t* decim, int32_t* nout,
                   int64_t* offset) {
    if (!plan) return SPT_ERR_INVALID;
    int32_t loc = 0;
    const RangePlan* rp = range_of_trial(plan->p, trial, &loc);
    if (!rp) return SPT_ERR_SHAPE;
    if (dm) *dm = rp->dm_lo + (double)loc * rp->dm_step;
    if (range) *range = (int32_t)(rp - plan->p.ranges.data());
    if (decim) *decim = rp->decim;
    if (nout) *nout = rp->nout[loc];
    if (offset) *offset = rp->offset[loc];
    return SPT_OK;
}

int spt_plan_delays(const spt_plan* plan, int32_t trial, int32_t* host_out) {
    if (!plan || !host_out) return SPT_ERR_INVALID;
    int32_t loc = 0;
    const RangePlan* rp = range_of_trial(plan->p, trial, &loc);
    if (!rp) return SPT_ERR_SHAPE;
    std::memcpy(host_out, &rp->delay[(size_t)loc * plan->p.nchan], sizeof(int32_t) * plan->p.nchan);
    return SPT_OK;
}

int spt_plan_set_option(spt_plan* plan, const char* name, int64_t value) {
    if (!plan || !name) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (!std::strcmp(name, "profile")) {
        if (value != 0 && value != 1) return SPT_ERR_INVALID;
        p.opt_profile = (int32_t)value;
        return SPT_OK;
    }
    if (!std::strcmp(name, "peaks_lookup")) {
        if (value < 0 || value > 3) return SPT_ERR_INVALID;
        p.opt_peaks_lookup = (int32_t)value;
        return SPT_OK;
    }
    if (p.dev) return SPT_ERR_STATE;
    if (!std::strcmp(name, "compact")) {
        if (value != 0 && value != 1) return SPT_ERR_INVALID;
        p.opt_compact = (int32_t)value; p.tiling_built = false;
        return SPT_OK;
    }
    if (!std::strcmp(name, "dedisp_kernel")) {
        if (value != 0 && value != 1) return SPT_ERR_INVALID;
        p.opt_kernel = (int32_t)value;
    } else if (!std::strcmp(name, "group")) {
        if (value != 1 && value != 2 && value != 4 && value != 8 && value != 12 && value != 16) return SPT_ERR_INVALID;
        p.opt_group = (int32_t)value; p.tiling_built = false;
    } else if (!std::strcmp(name, "tile_words")) {
        if (value != 0 && value != 224 && value != 256) return SPT_ERR_INVALID;
        if (value == 224 && p.opt_dm_tile != 64) return SPT_ERR_INVALID;
        p.opt_kh = (int32_t)value; p.tiling_built = false;
    } else if (!std::strcmp(name, "max_entries")) {
        if (value != 8 && value != 12 && value != 16) return SPT_ERR_INVALID;
        p.opt_max_ent = (int32_t)value; p.tiling_built = false;
    } else if (!std::strcmp(name, "skew")) {
        if (value != 0 && value != 1) return SPT_ERR_INVALID;
        p.opt_skew = (int32_t)value; p.tiling_built = false;
    } else if (!std::strcmp(name, "dm_tile")) {
        if (value != 32 && value != 64) return SPT_ERR_INVALID;
        if (value != 64 && p.opt_kh == 224) return SPT_ERR_INVALID;          // the narrow tile exists for 64-trial tiles only
        p.opt_dm_tile = (int32_t)value; p.tiling_built = false;
    } else {
        return SPT_ERR_INVALID;
    }
    return SPT_OK;
}

static int ensure_tiling(Plan& p) {
    if (p.tiling_built) return SPT_OK;
    try {
        return build_tiling(p);
    } catch (const std::bad_alloc&) {
        return SPT_ERR_NOMEM;
    }
}

int spt_plan_tiling_info(spt_plan* plan, int32_t range, int64_t* ntiles_dm, int64_t* nstages, int64_t* ngroups,
                         int64_t* nvariants, int64_t* ntiles_t, int64_t* max_stage_words) {
    if (!plan) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (range < 0 || range >= (int32_t)p.ranges.size()) return SPT_ERR_SHAPE;
    const int rc = ensure_tiling(p);
    if (rc != SPT_OK) return rc;
    const RangePlan& rp = p.ranges[range];
    {   // bounds check of every address the kernel will form from the tables (both sets of a decimated range)
        int rcc = check_tables(p, rp, rp.decim == 1 ? 1 : 2);
        if (rcc == SPT_OK && (size_t)range < p.compact.size() && !p.compact[range].tiles.empty()) rcc = check_tables(p, p.compact[range], 1);
        if (rcc != SPT_OK) return rcc;
    }
    if (ntiles_dm) *ntiles_dm = (int64_t)rp.tiles.size();
    if (nstages) *nstages = (int64_t)rp.sidx.size() - 1;   // the last entry is padding
    if (ngroups) *ngroups = rp.ngroups;
    if (nvariants) *nvariants = rp.nvariants;
    if (ntiles_t) *ntiles_t = rp.ntile_t;
    if (max_stage_words) {
        // largest shared-memory footprint of a stage: variant words + raw-row bytes, plus the fixed control area
        const int es = rp.decim == 1 ? 1 : 2;
        int64_t m = 0;
        for (size_t is = 0; is + 1 < rp.sidx.size(); ++is) {
            const StageIndex& si = rp.sidx[is];
            const uint32_t* b = &rp.blob[si.blob_word0];
            int64_t v = 0, r = 0;
            for (uint32_t k = 0; k < b[0]; ++k)
                v += (int64_t)b[kBlobHdrWords + 4 * k + 1] * (b[kBlobHdrWords + 4 * k + 2] >> 24);
            for (uint32_t k = 0; k < si.nrows; ++k) r += (int64_t)rp.rows[si.row0 + k].nelem * es;
            if (v > rp.vcap_words || r > kSmemDataBytes - (int64_t)rp.vcap_words * 4) return SPT_ERR_STATE;
            m = std::max(m, v + r / 4);
        }
        *max_stage_words = m + (kSmemCtrlBytes + 2 * kBlobBytes) / 4;
    }
    return SPT_OK;
}

int spt_plan_tiling_cost(spt_plan* plan, int32_t range, int64_t* ntasks, int64_t* task_entries, int64_t* task_variants,
                         int64_t* presum_rounds) {
    if (!plan) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (range < 0 || range >= (int32_t)p.ranges.size()) return SPT_ERR_SHAPE;
    const int rc = ensure_tiling(p);
    if (rc != SPT_OK) return rc;
    const RangePlan& rp = p.ranges[range];
    if (ntasks) *ntasks = rp.ntasks;
    if (task_entries) *task_entries = rp.task_entries;
    if (task_variants) *task_variants = rp.task_variants;
    if (presum_rounds) *presum_rounds = rp.presum_rounds;
    return SPT_OK;
}

int spt_plan_tiling_choice(spt_plan* plan, int32_t range, int32_t* tile_words, int32_t* max_entries, int32_t* group,
                           int32_t* has_compact) {
    if (!plan) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (range < 0 || range >= (int32_t)p.ranges.size()) return SPT_ERR_SHAPE;
    const int rc = ensure_tiling(p);
    if (rc != SPT_OK) return rc;
    const RangePlan& rp = p.ranges[range];
    if (tile_words) *tile_words = rp.kh;
    if (max_entries) *max_entries = rp.max_ent;
    if (group) *group = p.opt_group ? p.opt_group : (rp.max_ent > 8 ? 16 : 8);
    if (has_compact) *has_compact = ((size_t)range < p.compact.size() && !p.compact[range].tiles.empty()) ? 1 : 0;
    return SPT_OK;
}

// The delay row of trial `loc` of a range as one set of kernel tables applies it (es: bytes per element of the series the
// tables address).
static int tiling_delays_of(const Plan& p, const RangePlan* rp, int es, int32_t loc, int32_t* host_out) {
    const int DT = p.opt_dm_tile;
    const TileDesc& td = rp->tiles[loc / DT];
    const int dl = loc - td.trial0;
    for (int32_t c = 0; c < p.nchan; ++c) host_out[c] = INT32_MIN;
    for (int s = td.stage0; s < td.stage0 + td.nstage; ++s) {
        const StageIndex& si = rp->sidx[s];
        const uint32_t* b = &rp->blob[si.blob_word0];
        const uint32_t ngrp = b[0];
        const uint16_t* toff = reinterpret_cast<const uint16_t*>(b + b[3]);
        for (uint32_t g = 0; g < ngrp; ++g) {
            const uint32_t* gh = b + kBlobHdrWords + 4 * g;
            const int32_t vbase = (int32_t)(gh[0] & 0xffffu), vlen = (int32_t)gh[1];
            const int32_t nch = (int32_t)(gh[2] & 0xffu), ntog = (int32_t)((gh[2] >> 8) & 0xffu);
            const int32_t ncorr = (int32_t)((gh[2] >> 16) & 0xffu), nvar = (int32_t)(gh[2] >> 24);
            const uint32_t* cd = b + (gh[3] & 0xffffu);
            const uint32_t* vd = b + (gh[3] >> 16);
            const int32_t to = (int32_t)toff[g * DT + dl];
            const int32_t rel = to - vbase, r = rel / vlen, bb = rel - r * vlen;
            if (r < 0 || r >= nvar) return SPT_ERR_STATE;
            // the gather reads P_r[q + bb]; P_r[u] takes, of the entry at position q, the sample at its shift + u, or
            // one later when the variant takes the entry's delta.  Which deltas: from the chain word or the mask.
            uint32_t bits = 0xffffffffu;
            for (int32_t k = 0; k <= ntog; ++k)
                if (vd[k] == (uint32_t)(vbase + r * vlen)) bits = (1u << k) - 1u;
            for (int32_t c = 0; c < ncorr; ++c)
                if (vd[chain_words(ent_class(nch)) + 2 * c] == (uint32_t)(vbase + r * vlen))
                    bits = ((1u << ntog) - 1u) & ~vd[chain_words(ent_class(nch)) + 1 + 2 * c];
            if (bits == 0xffffffffu) return SPT_ERR_STATE;
            for (int pass = 0; pass < 2; ++pass)       // pass 0: base shifts; pass 1: one sample later per delta taken
                for (int32_t q = 0; q < nch; ++q) {
                    const int32_t byte = (int32_t)(cd[2 * q] & 0x3ffffu) + (int32_t)((cd[2 * q] >> 24) & 3u) * es;
                    const RowDesc* row = nullptr;
                    for (uint32_t i = 0; i < si.nrows; ++i) {
                        const RowDesc& rr = rp->rows[si.row0 + i];
                        if (byte >= rr.soff && byte < rr.soff + rr.nelem * es) { row = &rr; break; }
                    }
                    if (!row) return SPT_ERR_STATE;
                    const bool taken = (bits >> q) & 1u;
                    if (pass == 0 && (cd[2 * q] & kEntryAddBase)) {
                        if (host_out[row->chan] != INT32_MIN) return SPT_ERR_STATE;   // every channel exactly once
                        host_out[row->chan] = row->astart + (byte - row->soff) / es + bb;
                    }
                    if (pass == 1 && taken) {
                        if (host_out[row->chan] == INT32_MIN) return SPT_ERR_STATE;
                        host_out[row->chan] += 1;
                    }
                }
        }
    }
    // the tables hold the delays relative to the trial's skewed output window
    const int32_t sk = rp->skew[(size_t)td.skew0 + dl];
    for (int32_t c = 0; c < p.nchan; ++c)
        if (host_out[c] != INT32_MIN) host_out[c] += sk;
    return SPT_OK;
}

int spt_plan_tiling_delays(spt_plan* plan, int32_t trial, int32_t* host_out) {
    if (!plan || !host_out) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    int32_t loc = 0;
    const RangePlan* rp = range_of_trial(p, trial, &loc);
    if (!rp) return SPT_ERR_SHAPE;
    int rc = ensure_tiling(p);
    if (rc != SPT_OK) return rc;
    if ((rc = tiling_delays_of(p, rp, rp->decim == 1 ? 1 : 2, loc, host_out)) != SPT_OK) return rc;
    // a decimated range has a second set of tables, for the 8-bit copy of its series: it must say the same
    const size_t ri = (size_t)(rp - p.ranges.data());
    if (ri < p.compact.size() && !p.compact[ri].tiles.empty()) {
        std::vector<int32_t> again((size_t)p.nchan);
        if ((rc = tiling_delays_of(p, &p.compact[ri], 1, loc, again.data())) != SPT_OK) return rc;
        if (std::memcmp(again.data(), host_out, sizeof(int32_t) * (size_t)p.nchan) != 0) return SPT_ERR_STATE;
    }
    return SPT_OK;
}

int spt_dedisperse(spt_plan* plan, const uint8_t* d_fb, int32_t nbeam, int32_t* d_dmt, void* cuda_stream) {
    if (!plan || !d_fb || nbeam < 1) return SPT_ERR_INVALID;
    if (!d_dmt && plan->p.dmt_elems > 0) return SPT_ERR_INVALID;   // a plan whose trials are all empty has no output
    if (nbeam > plan->p.max_beams) return SPT_ERR_INVALID;
    if ((reinterpret_cast<uintptr_t>(d_dmt) & 127) != 0) return SPT_ERR_INVALID;
    int rc;
    try {
        rc = ensure_device(&plan->p);
    } catch (const std::bad_alloc&) {
        rc = SPT_ERR_NOMEM;
    }
    if (rc != SPT_OK) return rc;
    return do_dedisperse(&plan->p, d_fb, nbeam, d_dmt, (cudaStream_t)cuda_stream);
}

int spt_decimated(const spt_plan* plan, int32_t range, const uint16_t** d_ptr, int64_t* nsamp_k) {
    if (!plan || !d_ptr) return SPT_ERR_INVALID;
    const Plan& p = plan->p;
    if (range < 0 || range >= (int32_t)p.ranges.size()) return SPT_ERR_SHAPE;
    const RangePlan& rp = p.ranges[range];
    if (nsamp_k) *nsamp_k = rp.nsamp_k;
    if (rp.decim == 1) { *d_ptr = nullptr; return SPT_OK; }
    if (!p.dev || p.dev->nbeam_dedisp == 0) return SPT_ERR_STATE;
    *d_ptr = p.dev->r[range].series;
    return SPT_OK;
}

int spt_decimated_stride(const spt_plan* plan, int32_t range, int64_t* row_stride) {
    if (!plan || !row_stride) return SPT_ERR_INVALID;
    const Plan& p = plan->p;
    if (range < 0 || range >= (int32_t)p.ranges.size()) return SPT_ERR_SHAPE;
    *row_stride = p.ranges[range].stride_k;
    return SPT_OK;
}

int spt_decimated_read(spt_plan* plan, int32_t range, int32_t beam, uint16_t* host_out) {
    if (!plan || !host_out) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (range < 0 || range >= (int32_t)p.ranges.size()) return SPT_ERR_SHAPE;
    const RangePlan& rp = p.ranges[range];
    if (rp.decim == 1) return SPT_ERR_INVALID;
    if (!p.dev || p.dev->nbeam_dedisp == 0) return SPT_ERR_STATE;
    if (beam < 0 || beam >= p.dev->nbeam_dedisp) return SPT_ERR_SHAPE;
    SPT_CUDA(cudaStreamSynchronize(p.dev->dedisp_stream));
    if (rp.nsamp_k <= 0) return SPT_OK;
    const uint16_t* src = p.dev->r[range].series + (size_t)beam * p.nchan * rp.stride_k;
    SPT_CUDA(cudaMemcpy2D(host_out, (size_t)rp.nsamp_k * 2, src, (size_t)rp.stride_k * 2, (size_t)rp.nsamp_k * 2,
                          (size_t)p.nchan, cudaMemcpyDeviceToHost));
    return SPT_OK;
}

int spt_decimated_compact(spt_plan* plan, int32_t range, int32_t* in_use, uint32_t* floor_value, uint32_t* span) {
    if (!plan || !in_use) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (range < 0 || range >= (int32_t)p.ranges.size()) return SPT_ERR_SHAPE;
    *in_use = 0;
    if (floor_value) *floor_value = 0;
    if (span) *span = 0;
    if (!p.dev || p.dev->nbeam_dedisp == 0) return SPT_ERR_STATE;
    const RangeDev& rd = p.dev->r[range];
    if (!rd.series8 || p.ranges[range].nsamp_k <= 0) return SPT_OK;     // no copy for this range (decim == 1, option off, tables)
    SPT_CUDA(cudaStreamSynchronize(p.dev->dedisp_stream));
    uint32_t info[4] = {0, 0, 0, 0};
    SPT_CUDA(cudaMemcpy(info, rd.cinfo, sizeof(info), cudaMemcpyDeviceToHost));
    *in_use = info[2] == 1u ? 1 : 0;
    if (floor_value) *floor_value = info[3];
    if (span) *span = info[0];
    return SPT_OK;
}

int spt_single_pulse_search(spt_plan* plan, const int32_t* d_dmt, int32_t nbeam, float threshold, void* cuda_stream) {
    if (!plan || nbeam < 1 || nbeam > plan->p.max_beams || !(threshold == threshold)) return SPT_ERR_INVALID;
    if (!d_dmt && plan->p.dmt_elems > 0) return SPT_ERR_INVALID;
    int rc;
    try {
        rc = ensure_device(&plan->p);
    } catch (const std::bad_alloc&) {
        rc = SPT_ERR_NOMEM;
    }
    if (rc != SPT_OK) return rc;
    return do_search(&plan->p, d_dmt, nbeam, threshold, (cudaStream_t)cuda_stream);
}

int spt_search(spt_plan* plan, const uint8_t* d_fb, int32_t nbeam, int32_t* d_dmt, float threshold, void* cuda_stream) {
    if (!plan || !d_fb || nbeam < 1 || !(threshold == threshold)) return SPT_ERR_INVALID;
    if (!d_dmt && plan->p.dmt_elems > 0) return SPT_ERR_INVALID;
    if (nbeam > plan->p.max_beams) return SPT_ERR_INVALID;
    if ((reinterpret_cast<uintptr_t>(d_dmt) & 127) != 0) return SPT_ERR_INVALID;
    int rc;
    try {
        rc = ensure_device(&plan->p);
    } catch (const std::bad_alloc&) {
        rc = SPT_ERR_NOMEM;
    }
    if (rc != SPT_OK) return rc;
    return do_path(&plan->p, d_fb, nbeam, d_dmt, threshold, (cudaStream_t)cuda_stream, 0);
}

int spt_trial_stats(spt_plan* plan, int32_t beam, int32_t trial, int64_t* n, int64_t* sum, uint64_t* sumsq) {
    if (!plan) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (!p.dev || !p.dev->searched) return SPT_ERR_STATE;
    if (beam < 0 || beam >= p.dev->nbeam_search || trial < 0 || trial >= p.ntrials) return SPT_ERR_SHAPE;
    { const int rc = sync_results(p.dev); if (rc != SPT_OK) return rc; }
    int32_t loc = 0;
    const RangePlan* rp = range_of_trial(p, trial, &loc);
    if (n) *n = rp->nout[loc];
    const size_t idx = (size_t)beam * p.ntrials + trial;
    if (sum) SPT_CUDA(cudaMemcpy(sum, p.dev->bufs[p.dev->cur].sum + idx, 8, cudaMemcpyDeviceToHost));
    if (sumsq) SPT_CUDA(cudaMemcpy(sumsq, p.dev->bufs[p.dev->cur].sumsq + idx, 8, cudaMemcpyDeviceToHost));
    return SPT_OK;
}

int spt_trial_stats_all(spt_plan* plan, int32_t nbeam, int64_t* sum, uint64_t* sumsq) {
    if (!plan) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (!p.dev || !p.dev->searched) return SPT_ERR_STATE;
    if (nbeam < 1 || nbeam > p.dev->nbeam_search) return SPT_ERR_SHAPE;
    { const int rc = sync_results(p.dev); if (rc != SPT_OK) return rc; }
    const size_t bytes = (size_t)nbeam * p.ntrials * 8;
    if (sum) SPT_CUDA(cudaMemcpy(sum, p.dev->bufs[p.dev->cur].sum, bytes, cudaMemcpyDeviceToHost));
    if (sumsq) SPT_CUDA(cudaMemcpy(sumsq, p.dev->bufs[p.dev->cur].sumsq, bytes, cudaMemcpyDeviceToHost));
    return SPT_OK;
}

int spt_candidates_count(spt_plan* plan, int64_t* total, int32_t* overflowed) {
    if (!plan) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (!p.dev || !p.dev->searched) return SPT_ERR_STATE;
    { const int rc = sync_results(p.dev); if (rc != SPT_OK) return rc; }
    unsigned long long c = 0;
    SPT_CUDA(cudaMemcpy(&c, p.dev->bufs[p.dev->cur].count, 8, cudaMemcpyDeviceToHost));
    if (total) *total = (int64_t)c;
    if (overflowed) *overflowed = (int64_t)c > p.cand_capacity ? 1 : 0;
    return SPT_OK;
}

int spt_candidates_read(spt_plan* plan, spt_candidate* host_out, int64_t cap, int64_t* nwritten) {
    if (!plan || (!host_out && cap > 0) || cap < 0) return SPT_ERR_INVALID;
    int64_t total = 0;
    const int rc = spt_candidates_count(plan, &total, nullptr);
    if (rc != SPT_OK) return rc;
    int64_t n = total;
    if (n > plan->p.cand_capacity) n = plan->p.cand_capacity;
    if (n > cap) n = cap;
    if (n > 0)
        SPT_CUDA(cudaMemcpy(host_out, plan->p.dev->bufs[plan->p.dev->cur].cand, (size_t)n * sizeof(spt_candidate), cudaMemcpyDeviceToHost));
    if (nwritten) *nwritten = n;
    return SPT_OK;
}

int spt_search_host(spt_plan* plan, const uint8_t* h_fb, int32_t nbeam, float threshold, int32_t* h_dmt, int64_t* ncand,
                    int32_t* overflowed) {
    if (!plan || !h_fb || nbeam < 1 || nbeam > plan->p.max_beams) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    int rc;
    try {
        rc = ensure_device(&p);
    } catch (const std::bad_alloc&) {
        rc = SPT_ERR_NOMEM;
    }
    if (rc != SPT_OK) return rc;
    DeviceState* d = p.dev;
    const size_t fb_bytes = (size_t)p.nchan * p.nsamp;
    if (!d->h_fb) SPT_CUDA(cudaMalloc((void**)&d->h_fb, fb_bytes * p.max_beams));
    if (!d->h_dmt) SPT_CUDA(cudaMalloc((void**)&d->h_dmt, (size_t)p.dmt_elems * 4 * p.max_beams + 128));
    cudaStream_t st = d->own_stream;
    SPT_CUDA(cudaMemcpyAsync(d->h_fb, h_fb, fb_bytes * nbeam, cudaMemcpyHostToDevice, st));
    if ((rc = do_path(&p, d->h_fb, nbeam, d->h_dmt, threshold, st, 0)) != SPT_OK) return rc;
    if (h_dmt) SPT_CUDA(cudaMemcpyAsync(h_dmt, d->h_dmt, (size_t)p.dmt_elems * 4 * nbeam, cudaMemcpyDeviceToHost, st));
    int64_t total = 0;
    int32_t ovf = 0;
    if ((rc = spt_candidates_count(plan, &total, &ovf)) != SPT_OK) return rc;
    if (ncand) *ncand = total;
    if (overflowed) *overflowed = ovf;
    return SPT_OK;
}

int spt_stream_push(spt_plan* plan, const uint8_t* h_fb, int32_t nbeam, float threshold) {
    if (!plan || !h_fb || nbeam < 1 || nbeam > plan->p.max_beams || !(threshold == threshold)) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    int rc;
    try {
        rc = ensure_device(&p);
    } catch (const std::bad_alloc&) {
        rc = SPT_ERR_NOMEM;
    }
    if (rc != SPT_OK) return rc;
    DeviceState* d = p.dev;
    const int k = d->push_next;
    DeviceState::Slot& sl = d->slot[k];
    if (sl.pending) return SPT_ERR_STATE;                        // two batches are in flight: pop first
    const size_t fb_bytes = (size_t)p.nchan * p.nsamp;
    if (!d->copy_stream) SPT_CUDA(cudaStreamCreateWithFlags(&d->copy_stream, cudaStreamNonBlocking));
    if (!sl.fb) {
        SPT_CUDA(cudaMalloc((void**)&sl.fb, fb_bytes * p.max_beams));
        SPT_CUDA(cudaMallocHost((void**)&sl.h_count, 8));
        SPT_CUDA(cudaEventCreateWithFlags(&sl.copied, cudaEventDisableTiming));
        SPT_CUDA(cudaEventCreateWithFlags(&sl.done, cudaEventDisableTiming));
        if (k == 1 && !d->bufs[1].sum && (rc = alloc_search_bufs(&p, d->bufs[1])) != SPT_OK) return rc;
    }
    if (!d->h_dmt) SPT_CUDA(cudaMalloc((void**)&d->h_dmt, (size_t)p.dmt_elems * 4 * p.max_beams + 128));
    // copy engine: this batch's input, while the kernels of the previous batch run on the compute stream
    SPT_CUDA(cudaMemcpyAsync(sl.fb, h_fb, fb_bytes * nbeam, cudaMemcpyHostToDevice, d->copy_stream));
    SPT_CUDA(cudaEventRecord(sl.copied, d->copy_stream));
    cudaStream_t st = d->own_stream;
    SPT_CUDA(cudaStreamWaitEvent(st, sl.copied, 0));
    // the read-out calls keep looking at the batch popped last: everything do_search changes for them is put back,
    // also when the push fails half way
    const cudaEvent_t keep = d->wait_event;
    const int keep_cur = d->cur;
    const bool keep_searched = d->searched, keep_peaks = d->peaks_valid;
    const int32_t keep_nbeam = d->nbeam_search;
    cudaStream_t const keep_stream = d->last_stream;
    rc = do_path(&p, sl.fb, nbeam, d->h_dmt, threshold, st, k);
    d->wait_event = keep; d->cur = keep_cur; d->searched = keep_searched; d->peaks_valid = keep_peaks;
    d->nbeam_search = keep_nbeam;
    // a read-out without an event (after spt_peak_filter, or of a plain call) synchronises the stream it ran on, not ours
    if (keep_stream || keep_searched) d->last_stream = keep_stream;
    if (rc != SPT_OK) return rc;
    SPT_CUDA(cudaMemcpyAsync(sl.h_count, d->bufs[k].count, 8, cudaMemcpyDeviceToHost, st));
    SPT_CUDA(cudaEventRecord(sl.done, st));
    sl.nbeam = nbeam;
    sl.pending = true;
    d->push_next = k ^ 1;
    return SPT_OK;
}

int spt_stream_pop(spt_plan* plan, int64_t* ncand, int32_t* overflowed) {
    if (!plan) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (!p.dev) return SPT_ERR_STATE;
    DeviceState* d = p.dev;
    const int k = d->pop_next;
    DeviceState::Slot& sl = d->slot[k];
    if (!sl.pending) return SPT_ERR_STATE;                       // nothing pushed
    SPT_CUDA(cudaEventSynchronize(sl.done));
    const int64_t total = (int64_t)*sl.h_count;
    if (ncand) *ncand = total;
    if (overflowed) *overflowed = total > p.cand_capacity ? 1 : 0;
    sl.pending = false;
    d->pop_next = k ^ 1;
    d->cur = k;                                                  // read-out calls now look at this batch's results
    d->wait_event = sl.done;
    d->nbeam_search = sl.nbeam;
    d->searched = true;
    return SPT_OK;
}

int spt_peak_filter(spt_plan* plan, const int32_t* windows, int32_t nwindows, void* cuda_stream) {
    if (!plan || !windows || nwindows < 1 || nwindows > 8) return SPT_ERR_INVALID;
    for (int32_t i = 0; i < nwindows; ++i)
        if (windows[i] < 1 || (windows[i] & 1) == 0 || windows[i] > 255) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (!p.dev || !p.dev->searched) return SPT_ERR_STATE;
    DeviceState* d = p.dev;
    int64_t total = 0;
    int32_t ovf = 0;
    int rc = spt_candidates_count(plan, &total, &ovf);           // waits for the search the list comes from
    if (rc != SPT_OK) return rc;
    if (ovf) return SPT_ERR_SHAPE;                               // an incomplete list cannot be filtered
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!d->peaks_count) SPT_CUDA(cudaMalloc((void**)&d->peaks_count, 8));
    if (total > d->alive_cap) {
        cudaFree(d->alive[0]); cudaFree(d->alive[1]); cudaFree(d->peaks);
        d->alive[0] = d->alive[1] = nullptr; d->peaks = nullptr; d->alive_cap = d->peaks_cap = 0;
        SPT_CUDA(cudaMalloc((void**)&d->alive[0], (size_t)total));
        SPT_CUDA(cudaMalloc((void**)&d->alive[1], (size_t)total));
        SPT_CUDA(cudaMalloc((void**)&d->peaks, (size_t)total * sizeof(spt_candidate)));
        d->alive_cap = d->peaks_cap = total;
    }
    SPT_CUDA(cudaMemsetAsync(d->peaks_count, 0, 8, st));
    PeakArgs a{};
    a.cand = d->bufs[d->cur].cand; a.n = total; a.beam_stride = p.dmt_elems;
    a.nout = d->nout; a.offset = d->offset; a.range_lo = d->range_lo; a.range_hi = d->range_hi;
    const int32_t nbeam = d->nbeam_search;
    // Sparse list (the paper's regime): a hash table of two slots per candidate.  Dense list (a sizeable fraction of all cells):
    // a plane like the DM transform, 4 GiB at most, covering as many beams as fit and passed over the list once per slice.
    uint64_t hcap = 1024;
    while (hcap < 2 * (uint64_t)total) hcap <<= 1;
    const double plane_all = (double)nbeam * (double)p.dmt_elems * 4.0;
    const bool use_hash = p.opt_peaks_lookup == 1 || (p.opt_peaks_lookup == 0 && (double)hcap * 12.0 <= plane_all / 4.0);
    const uint8_t* in = nullptr;
    int64_t nlaunch = 0;
    if (total > 0 && use_hash) {
        if (hcap > d->hcap) {
            cudaFree(d->hkeys); cudaFree(d->hvals);
            d->hkeys = nullptr; d->hvals = nullptr; d->hcap = 0;
            SPT_CUDA(cudaMalloc((void**)&d->hkeys, (size_t)hcap * 8));
            SPT_CUDA(cudaMalloc((void**)&d->hvals, (size_t)hcap * 4));
            d->hcap = hcap;
        }
        SPT_CUDA(cudaMemsetAsync(d->hkeys, 0xff, (size_t)hcap * 8, st));
        a.hkeys = d->hkeys; a.vals = d->hvals; a.hmask = hcap - 1;
        launch_peaks_insert(a, st);
        for (int32_t i = 0; i < nwindows; ++i) {
            launch_peaks_stencil(a, windows[i], in, d->alive[i & 1], st);
            if (i + 1 < nwindows) launch_peaks_erase(a, in, d->alive[i & 1], false, st);
            in = d->alive[i & 1];
        }
        nlaunch = 2 * nwindows;
    } else if (total > 0) {
        const int64_t per_beam = p.dmt_elems * 4;
        const int32_t fit = p.opt_peaks_lookup == 3 ? 1 :
            (int32_t)std::max<int64_t>(1, std::min<int64_t>(nbeam, (4ll << 30) / std::max<int64_t>(per_beam, 1)));
        if (fit > d->plane_beams || (p.opt_peaks_lookup == 3 && d->plane_beams != 1)) {
            cudaFree(d->plane);
            d->plane = nullptr; d->plane_beams = 0;
            SPT_CUDA(cudaMalloc((void**)&d->plane, (size_t)fit * per_beam));
            SPT_CUDA(cudaMemsetAsync(d->plane, 0xff, (size_t)fit * per_beam, st));   // all empty; every call leaves it so
            d->plane_beams = fit;
        }
        a.vals = d->plane;
        for (int32_t b0 = 0; b0 < nbeam; b0 += d->plane_beams) {
            a.beam0 = b0; a.nbeam_slice = std::min(d->plane_beams, nbeam - b0);
            launch_peaks_insert(a, st);
            const uint8_t* sin = nullptr;
            for (int32_t i = 0; i < nwindows; ++i) {
                launch_peaks_stencil(a, windows[i], sin, d->alive[i & 1], st);
                if (i + 1 < nwindows) launch_peaks_erase(a, sin, d->alive[i & 1], false, st);
                sin = d->alive[i & 1];
            }
            launch_peaks_erase(a, nullptr, nullptr, true, st);
            nlaunch += 2 * nwindows + 1;
        }
        in = d->alive[(nwindows - 1) & 1];
    }
    if (total > 0) { launch_peaks_compact(a, in, d->peaks, d->peaks_count, d->peaks_cap, st); ++nlaunch; }
    p.launches += nlaunch;
    SPT_CUDA(cudaGetLastError());
    d->last_stream = st;
    d->wait_event = nullptr;
    d->peaks_valid = true;
    return SPT_OK;
}

int spt_peak_filter_static(spt_plan* plan, const spt_candidate* d_cand, int64_t n, const int32_t* windows, int32_t nwindows,
                           spt_candidate* d_peaks, uint64_t* d_count, void* cuda_stream) {
    if (!plan || !windows || nwindows < 1 || nwindows > 8 || n < 0 || !d_count || (n > 0 && (!d_cand || !d_peaks)))
        return SPT_ERR_INVALID;
    for (int32_t i = 0; i < nwindows; ++i)
        if (windows[i] < 1 || (windows[i] & 1) == 0 || windows[i] > 255) return SPT_ERR_INVALID;
    if (n > SPT_PEAKS_STATIC_MAX) {
        g_last_error = "spt_peak_filter_static: " + std::to_string((long long)n) + " records exceed the fixed working memory (" +
                       std::to_string((long long)SPT_PEAKS_STATIC_MAX) + " records at most); use spt_peak_filter";
        return SPT_ERR_UNSUPPORTED;
    }
    Plan& p = plan->p;
    if (!p.dev) return SPT_ERR_STATE;       // the plan's device tables come from its first dedispersion / search, not from here
    DeviceState* d = p.dev;
    PeakArgs a{};
    a.cand = d_cand; a.n = n; a.beam_stride = p.dmt_elems;
    a.nout = d->nout; a.offset = d->offset; a.range_lo = d->range_lo; a.range_hi = d->range_hi;
    int64_t nlaunch = 0;
    SPT_CUDA(peaks_static_filter(a, windows, nwindows, d_peaks, (unsigned long long*)d_count, (long long)n, (cudaStream_t)cuda_stream,
                                 &nlaunch));
    p.launches += nlaunch;
    return SPT_OK;
}

int spt_peaks_count(spt_plan* plan, int64_t* total) {
    if (!plan || !total) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    if (!p.dev || !p.dev->peaks_valid) return SPT_ERR_STATE;
    SPT_CUDA(cudaStreamSynchronize(p.dev->last_stream));
    unsigned long long c = 0;
    SPT_CUDA(cudaMemcpy(&c, p.dev->peaks_count, 8, cudaMemcpyDeviceToHost));
    *total = (int64_t)c;
    return SPT_OK;
}

int spt_peaks_read(spt_plan* plan, spt_candidate* host_out, int64_t cap, int64_t* nwritten) {
    if (!plan || (!host_out && cap > 0) || cap < 0) return SPT_ERR_INVALID;
    int64_t n = 0;
    const int rc = spt_peaks_count(plan, &n);
    if (rc != SPT_OK) return rc;
    if (n > cap) n = cap;
    if (n > 0) SPT_CUDA(cudaMemcpy(host_out, plan->p.dev->peaks, (size_t)n * sizeof(spt_candidate), cudaMemcpyDeviceToHost));
    if (nwritten) *nwritten = n;
    return SPT_OK;
}

int spt_corner_turn(const uint8_t* d_in, int32_t nbeam, int64_t nsamp, int32_t nchan, int32_t flip, int32_t spliced,
                    uint8_t* d_out, void* cuda_stream) {
    if (!d_in || !d_out || nbeam < 1 || nsamp < 1 || nchan < 1 || (flip != 0 && flip != 1) || (spliced != 0 && spliced != 1))
        return SPT_ERR_INVALID;
    launch_corner_turn(d_in, nbeam, nsamp, nchan, flip, spliced, d_out, nsamp, (int64_t)nchan * nsamp, 0, (cudaStream_t)cuda_stream);
    SPT_CUDA(cudaGetLastError());
    return SPT_OK;
}

int spt_segment_info(const spt_plan* plan, int64_t* min_history, int64_t* min_history_search, int64_t* granule) {
    if (!plan) return SPT_ERR_INVALID;
    const Plan& p = plan->p;
    int64_t h = 0, hs = 0, g = 16;
    const int64_t wmax = p.widths.back();
    for (const RangePlan& rp : p.ranges) {
        int32_t dmax = 0;
        for (int32_t i = 0; i < rp.ndm; ++i) dmax = std::max(dmax, rp.delay[(size_t)i * p.nchan + p.nchan - 1]);
        h = std::max<int64_t>(h, (int64_t)dmax * rp.decim);
        hs = std::max<int64_t>(hs, ((int64_t)dmax + wmax - 1) * rp.decim);   // the widest boxcar may start in the old part
        g = std::max<int64_t>(g, rp.decim);
    }
    if (min_history) *min_history = (h + g - 1) / g * g;
    if (min_history_search) *min_history_search = (hs + g - 1) / g * g;
    if (granule) *granule = g;
    return SPT_OK;
}

int spt_segment_search(spt_plan* plan, const int32_t* d_dmt, int32_t nbeam, int64_t nnew, float threshold, void* cuda_stream) {
    if (!plan || !d_dmt || nbeam < 1 || nbeam > plan->p.max_beams || !(threshold == threshold)) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    int64_t hmin = 0, hs = 0, gran = 16;
    spt_segment_info(plan, &hmin, &hs, &gran);
    if (nnew < 1 || nnew > p.nsamp || nnew % gran != 0) return SPT_ERR_INVALID;
    if (p.nsamp - nnew < hs) return SPT_ERR_SHAPE;
    int rc;
    try {
        rc = ensure_device(&p);
    } catch (const std::bad_alloc&) {
        rc = SPT_ERR_NOMEM;
    }
    if (rc != SPT_OK) return rc;
    DeviceState* d = p.dev;
    if (d->win_nnew != nnew) {
        std::vector<int32_t> len, starts;
        const int32_t wmax = p.widths.back();
        for (const RangePlan& rp : p.ranges)
            for (int32_t i = 0; i < rp.ndm; ++i) {
                const int32_t ns = (int32_t)(nnew / rp.decim);
                len.push_back(ns + wmax - 1);
                starts.push_back(ns);
            }
        cudaFree(d->win_len); cudaFree(d->win_starts);
        d->win_len = d->win_starts = nullptr;
        if ((rc = upload(&d->win_len, len)) != SPT_OK) return rc;
        if ((rc = upload(&d->win_starts, starts)) != SPT_OK) return rc;
        d->win_nnew = nnew;
    }
    return do_search(&p, d_dmt, nbeam, threshold, (cudaStream_t)cuda_stream, 0, true);
}

int spt_segment_push(spt_plan* plan, const uint8_t* d_new, int32_t nbeam, int64_t nnew, int32_t flip, int32_t spliced,
                     int32_t whole_rows, int32_t* d_dmt, void* cuda_stream) {
    if (!plan || !d_new || !d_dmt || nbeam < 1 || nbeam > plan->p.max_beams || (flip != 0 && flip != 1) ||
        (spliced != 0 && spliced != 1) || (whole_rows != 0 && whole_rows != 1))
        return SPT_ERR_INVALID;
    if ((reinterpret_cast<uintptr_t>(d_dmt) & 127) != 0) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    int64_t hmin = 0, gran = 16;
    spt_segment_info(plan, &hmin, nullptr, &gran);
    // the shift must keep the phase of every decimation and the 16-byte alignment of the rows
    if (nnew < 1 || nnew > p.nsamp || nnew % gran != 0 || p.nsamp % 16 != 0) return SPT_ERR_INVALID;
    if (p.nsamp - nnew < hmin) return SPT_ERR_SHAPE;              // not every trial would have its full sweep
    int rc;
    try {
        rc = ensure_device(&p);
    } catch (const std::bad_alloc&) {
        rc = SPT_ERR_NOMEM;
    }
    if (rc != SPT_OK) return rc;
    DeviceState* d = p.dev;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t bytes = (size_t)p.max_beams * p.nchan * p.nsamp;
    if (!d->work[0]) {
        for (int i = 0; i < 2; ++i) {
            SPT_CUDA(cudaMalloc((void**)&d->work[i], bytes));
            // the stream starts on a history of zeros; on the caller's stream, so that the history copy and the corner turn
            // below are ordered behind it whatever kind of stream that is (a plain cudaMemset runs on the legacy default
            // stream, which a non-blocking stream does not wait for)
            SPT_CUDA(cudaMemsetAsync(d->work[i], 0, bytes, st));
        }
        d->work_cur = 0;
    }
    const uint8_t* prev = d->work[d->work_cur];
    uint8_t* cur = d->work[d->work_cur ^ 1];
    const int64_t keep = p.nsamp - nnew;
    // the history moves to the front of the other buffer on a side stream while the new block is corner-turned into its
    // tail on the caller's: the two write disjoint parts of the buffer
    if (keep > 0) {
        if (!d->hist_stream) {
            SPT_CUDA(cudaStreamCreateWithFlags(&d->hist_stream, cudaStreamNonBlocking));
            SPT_CUDA(cudaEventCreateWithFlags(&d->hist_fork, cudaEventDisableTiming));
            SPT_CUDA(cudaEventCreateWithFlags(&d->hist_join, cudaEventDisableTiming));
        }
        SPT_CUDA(cudaEventRecord(d->hist_fork, st));
        SPT_CUDA(cudaStreamWaitEvent(d->hist_stream, d->hist_fork, 0));
        launch_keep_history(prev, cur, p.nsamp, nnew, keep, (int64_t)nbeam * p.nchan, d->hist_stream);
        SPT_CUDA(cudaEventRecord(d->hist_join, d->hist_stream));
    }
    launch_corner_turn(d_new, nbeam, nnew, p.nchan, flip, spliced, cur, p.nsamp, (int64_t)p.nchan * p.nsamp, keep, st);
    if (keep > 0) SPT_CUDA(cudaStreamWaitEvent(st, d->hist_join, 0));
    p.launches += keep > 0 ? 2 : 1;
    SPT_CUDA(cudaGetLastError());
    d->work_cur ^= 1;
    return do_dedisperse(&p, cur, nbeam, d_dmt, st, false, whole_rows ? 0 : nnew);
}

int spt_sift(spt_plan* plan, const spt_candidate* h_in, int64_t n, int32_t nbeam, const spt_sift_params* prm,
             spt_candidate* h_out, int64_t cap, int64_t* nwritten, int64_t* stage_counts) {
    if (!plan || !prm || (!h_in && n > 0) || n < 0 || nbeam < 1 || cap < 0 || (!h_out && cap > 0)) return SPT_ERR_INVALID;
    if (!(prm->eps > 0.0) || prm->min_pts < 1 || !(prm->time_unit_s > 0.0) || !(prm->dm_unit > 0.0)) return SPT_ERR_INVALID;
    if (nbeam > kSiftMaxBeams || n >= (1ll << 31)) return SPT_ERR_UNSUPPORTED;
    Plan& p = plan->p;
    if (nwritten) *nwritten = 0;
    if (stage_counts) stage_counts[0] = stage_counts[1] = stage_counts[2] = 0;
    if (n == 0) return SPT_OK;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); g_last_error = "no CUDA device"; return SPT_ERR_CUDA; }
    // host: order by (beam, trial, t) -- the index then breaks S/N ties towards the smaller (trial, t) -- and the plane
    std::vector<int64_t> order((size_t)n);
    for (int64_t i = 0; i < n; ++i) {
        if (h_in[i].beam < 0 || h_in[i].beam >= nbeam || h_in[i].trial < 0 || h_in[i].trial >= p.ntrials) return SPT_ERR_SHAPE;
        order[(size_t)i] = i;
    }
    std::sort(order.begin(), order.end(), [&](int64_t a, int64_t b) {
        const spt_candidate &u = h_in[a], &v = h_in[b];
        if (u.beam != v.beam) return u.beam < v.beam;
        if (u.trial != v.trial) return u.trial < v.trial;
        return u.t < v.t;
    });
    std::vector<double> x((size_t)n), y((size_t)n), dm((size_t)n), wsec((size_t)n), arr((size_t)n);
    std::vector<float> snr((size_t)n);
    std::vector<int32_t> beam((size_t)n);
    std::vector<int64_t> lo((size_t)n), hi((size_t)n);
    for (int64_t i = 0; i < n; ++i) {
        const spt_candidate& c = h_in[order[(size_t)i]];
        int32_t loc = 0;
        const RangePlan* rp = range_of_trial(p, c.trial, &loc);
        const double k = (double)rp->decim;
        dm[(size_t)i] = rp->dm_lo + (double)loc * rp->dm_step;
        arr[(size_t)i] = ((double)c.t * k) * p.tsamp;                  // arrival at the top of the band, seconds
        wsec[(size_t)i] = ((double)c.width * k) * p.tsamp;
        x[(size_t)i] = arr[(size_t)i] / prm->time_unit_s;
        y[(size_t)i] = dm[(size_t)i] / prm->dm_unit;
        snr[(size_t)i] = c.snr;
        beam[(size_t)i] = c.beam;
    }
    for (int64_t i = 0, s0 = 0; i <= n; ++i)
        if (i == n || beam[(size_t)i] != beam[(size_t)s0]) {
            for (int64_t j = s0; j < i; ++j) { lo[(size_t)j] = s0; hi[(size_t)j] = i; }
            s0 = i;
        }
    // device: one allocation for everything
    const size_t nn = (size_t)n;
    const size_t bytes = nn * (5 * 8 + 4 + 4 + 2 * 8 + 3 * 4 + 8 + 4) + 256;
    uint8_t* buf = nullptr;
    SPT_CUDA(cudaMalloc((void**)&buf, bytes));
    uint8_t* q = buf;
    auto take = [&](size_t b) { uint8_t* r = q; q += (b + 15) / 16 * 16; return r; };
    SiftArgs a{};
    double *dx = (double*)take(nn * 8), *dy = (double*)take(nn * 8), *ddm = (double*)take(nn * 8), *dw = (double*)take(nn * 8),
           *da = (double*)take(nn * 8);
    int64_t *dlo = (int64_t*)take(nn * 8), *dhi = (int64_t*)take(nn * 8);
    unsigned long long* drep = (unsigned long long*)take(nn * 8);
    float* dsnr = (float*)take(nn * 4);
    int32_t *dbeam = (int32_t*)take(nn * 4), *dcore = (int32_t*)take(nn * 4), *dpar = (int32_t*)take(nn * 4),
            *dmem = (int32_t*)take(nn * 4), *dkeep = (int32_t*)take(nn * 4);
    cudaError_t ce = cudaSuccess;
    auto up = [&](void* d, const void* h, size_t b) { if (ce == cudaSuccess) ce = cudaMemcpy(d, h, b, cudaMemcpyHostToDevice); };
    up(dx, x.data(), nn * 8); up(dy, y.data(), nn * 8); up(ddm, dm.data(), nn * 8); up(dw, wsec.data(), nn * 8);
    up(da, arr.data(), nn * 8); up(dlo, lo.data(), nn * 8); up(dhi, hi.data(), nn * 8); up(dsnr, snr.data(), nn * 4);
    up(dbeam, beam.data(), nn * 4);
    if (ce == cudaSuccess) ce = cudaMemset(drep, 0, nn * 8);
    if (ce == cudaSuccess) ce = cudaMemset(dkeep, 0, nn * 4);
    a.n = n; a.nbeam = nbeam; a.min_pts = prm->min_pts;
    a.eps2 = prm->eps * prm->eps; a.snr_min = (double)prm->snr_min; a.dm_min = prm->dm_min; a.width_max_s = prm->width_max_s;
    a.coinc_window_s = prm->coinc_window_s; a.coinc_beam_fraction = prm->coinc_beam_fraction;
    a.x = dx; a.y = dy; a.dm = ddm; a.wsec = dw; a.arrival = da; a.snr = dsnr; a.beam = dbeam; a.seg_lo = dlo; a.seg_hi = dhi;
    a.core = dcore; a.parent = dpar; a.member = dmem; a.rep = drep; a.keep = dkeep;
    std::vector<int32_t> keep(nn, 0);
    if (ce == cudaSuccess) {
        launch_sift(a, nullptr);
        p.launches += 5;
        ce = cudaGetLastError();
    }
    if (ce == cudaSuccess) ce = cudaMemcpy(keep.data(), dkeep, nn * 4, cudaMemcpyDeviceToHost);
    cudaFree(buf);
    if (ce != cudaSuccess) return cuda_fail(ce, "spt_sift");
    int64_t w = 0;
    for (int64_t i = 0; i < n; ++i) {
        const int32_t kf = keep[(size_t)i];
        if (stage_counts) { stage_counts[0] += kf & 1; stage_counts[1] += (kf >> 1) & 1; stage_counts[2] += (kf >> 2) & 1; }
        if ((kf & 4) && w < cap) h_out[w++] = h_in[order[(size_t)i]];
    }
    if (nwritten) *nwritten = w;
    return SPT_OK;
}

int spt_cutout_batch(const uint8_t* d_fb, int32_t nbeam, int32_t nchan, int64_t nsamp, double fch1_mhz, double foff_mhz,
                     double tsamp_s, const spt_cutout_params* h_cands, int32_t ncand, int32_t ndm, int32_t nt, int32_t nf,
                     int32_t* d_dds, int32_t* d_dmt, void* cuda_stream) {
    if (!d_fb || !d_dds || !d_dmt || !h_cands || ncand < 1 || nbeam < 1 || nchan < 1 || nsamp < 1 || ndm < 1 || nt < 1 || nf < 1 ||
        nchan % nf != 0 || !(tsamp_s > 0.0) || !(fch1_mhz > 0.0))
        return SPT_ERR_INVALID;
    if (!(foff_mhz < 0.0)) return SPT_ERR_UNSUPPORTED;
    if (!(fch1_mhz + (double)(nchan - 1) * foff_mhz > 0.0)) return SPT_ERR_INVALID;
    if (ndm + nf > 65535) return SPT_ERR_UNSUPPORTED;
    for (int32_t k = 0; k < ncand; ++k) {
        const spt_cutout_params& c = h_cands[k];
        if (c.tbin < 1 || c.beam < 0 || c.beam >= nbeam || !(c.dm0 >= 0.0) || !(c.ddm >= 0.0)) return SPT_ERR_INVALID;
        if ((double)nchan * 255.0 * c.tbin >= 2147483648.0) return SPT_ERR_UNSUPPORTED;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    SPT_CUDA(cudaMemsetAsync(d_dds, 0, (size_t)ncand * nf * nt * 4, st));       // the kernel adds into its outputs
    SPT_CUDA(cudaMemsetAsync(d_dmt, 0, (size_t)ncand * ndm * nt * 4, st));
    CutoutArgs a{};
    a.x = d_fb; a.nsamp = nsamp; a.beam_stride = (long long)nchan * nsamp;
    a.fch1 = fch1_mhz; a.foff = foff_mhz; a.tsamp = tsamp_s;
    a.nchan = nchan; a.ndm = ndm; a.nt = nt; a.nf = nf;
    a.dds = d_dds; a.dmt = d_dmt;
    // candidates whose bins are one sample wide and the others run different kernel instances; each kind goes in launches of
    // at most kCutoutMaxCand candidates, whose parameters travel in the kernel's parameter block
    for (int kind = 0; kind < 2; ++kind) {
        int32_t k = 0;
        while (k < ncand) {
            a.ncand = 0;
            for (; k < ncand && a.ncand < kCutoutMaxCand; ++k) {
                if ((h_cands[k].tbin > 1) != (kind == 1)) continue;
                CutoutCand& c = a.cand[a.ncand++];
                c.dm0 = h_cands[k].dm0; c.ddm = h_cands[k].ddm; c.ts = h_cands[k].ts; c.tbin = h_cands[k].tbin;
                c.beam = h_cands[k].beam; c.out = k; c.pad_ = 0;
            }
            if (a.ncand == 0) continue;
            if (launch_cutout_batch(a, st) != 0) {
                g_last_error = "spt_cutout_batch: launch failed";
                cudaGetLastError();
                return SPT_ERR_CUDA;
            }
        }
    }
    return SPT_OK;
}

int spt_cutout(const uint8_t* d_fb, int32_t nchan, int64_t nsamp, double fch1_mhz, double foff_mhz, double tsamp_s, double dm0,
               double ddm, int32_t ndm, int64_t ts, int32_t tbin, int32_t nt, int32_t nf, int32_t* d_dds, int32_t* d_dmt,
               void* cuda_stream) {
    spt_cutout_params c{};
    c.dm0 = dm0; c.ddm = ddm; c.ts = ts; c.tbin = tbin; c.beam = 0;
    return spt_cutout_batch(d_fb, 1, nchan, nsamp, fch1_mhz, foff_mhz, tsamp_s, &c, 1, ndm, nt, nf, d_dds, d_dmt, cuda_stream);
}

double spt_delta_dm(double width_s, double snr_ratio, double nu_mhz, double bw_mhz) {
    // Eq. 4 as printed; reading H notes that the derivation's own first line implies 13820
    return std::sqrt(3.14159265358979323846) / 1382.0 * width_s * (1.0 / snr_ratio) * (nu_mhz * nu_mhz * nu_mhz) / bw_mhz;
}

int spt_plan_kernel_times(spt_plan* plan, int32_t cap, int32_t* kind, int32_t* range, double* ms, int32_t* n) {
    if (!plan || !n || cap < 0) return SPT_ERR_INVALID;
    Plan& p = plan->p;
    *n = 0;
    if (!p.dev) return SPT_ERR_STATE;
    if (p.dev->nbeam_dedisp) SPT_CUDA(cudaStreamSynchronize(p.dev->dedisp_stream));
    if (p.dev->searched) SPT_CUDA(cudaStreamSynchronize(p.dev->last_stream));
    for (int slot = 0; slot < 2; ++slot)
        for (auto& t : p.dev->timed[slot]) {
            if (*n >= cap) return SPT_OK;
            float f = 0.f;
            SPT_CUDA(cudaEventElapsedTime(&f, t.e0, t.e1));
            if (kind) kind[*n] = t.kind;
            if (range) range[*n] = t.range;
            if (ms) ms[*n] = (double)f;
            ++*n;
        }
    return SPT_OK;
}

int spt_plan_launches(const spt_plan* plan, int64_t* launches) {
    if (!plan || !launches) return SPT_ERR_INVALID;
    *launches = plan->p.launches;
    return SPT_OK;
}

int spt_probe(int32_t kind, int32_t reps, double* warp_instr_per_s, double* elapsed_ms) {
    if (kind < 0 || kind > 4) return SPT_ERR_INVALID;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        g_last_error = "no CUDA device";
        return SPT_ERR_CUDA;
    }
    if (run_probe(kind, reps, warp_instr_per_s, elapsed_ms) != 0) { g_last_error = "probe failed"; return SPT_ERR_CUDA; }
    return SPT_OK;
}

const char* spt_strerror(int code) {
    switch (code) {
        case SPT_OK: return "ok";
        case SPT_ERR_INVALID: return "invalid argument";
        case SPT_ERR_UNSUPPORTED: return "unsupported configuration";
        case SPT_ERR_NOMEM: return "out of memory";
        case SPT_ERR_CUDA: return "CUDA error";
        case SPT_ERR_SHAPE: return "buffer too small or index out of range";
        case SPT_ERR_STATE: return "call out of order";
        default: return "unknown error";
    }
}

const char* spt_last_error(void) { return g_last_error.c_str(); }

}  // extern "C"
