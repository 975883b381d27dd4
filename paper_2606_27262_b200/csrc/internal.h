// internal.h -- shared declarations of libspt (host plan + CUDA launchers).  Not part of the ABI.
#pragma once

#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/spt.h"

namespace spt {

// BASELINE.json north_star (2): dt = 4.148808e3 s * DM * (f^-2 - f_top^-2), f in MHz.  (The paper prints
// 4.1488064239(11)e3; reading A2 explains why north_star's value binds.)
constexpr double kDispersionConstantS = 4.148808e3;

constexpr int kRowAlignElems = 32;  // DM-transform rows start 128-byte aligned
constexpr int kMaxWidths = 32;

// ---- tiled dedispersion kernel geometry ------------------------------------------------
// A block owns DT trials x TT = 2*H output samples; two blocks are resident per SM.  Packed 16-bit accumulator
// word q of a trial holds the outputs t0+q (low half) and t0+H+q (high half).
constexpr int kHMax = 256;           // words per trial per tile, at most: a tile is 2*kh output samples wide, kh = 224 or 256 per
                                     // DM range (RangePlan::kh; the kernel is a template on it)
constexpr int kThreads = 256;        // 8 warps
constexpr int kMaxEnt = 16;          // entries (a channel at one of its shifts) per pre-summed group, at most; the pre-sum code
                                     // exists for groups of up to 8, 12 and 16 entries (ent_class)
constexpr int kMaxVar = 16;          // variants per group
constexpr int kMaxDT = 64;           // trials per DM tile
constexpr int kMaxStageGroups = 8;   // groups per stage
constexpr int kChunkU = 128;         // variant words one warp builds per pre-sum task (4 per lane)
constexpr int kBlobBytes = 3072;     // per-stage table blob (two buffers in shared memory)
constexpr int kSmemBytes = 113 * 1024;                                   // two blocks per SM (228 KB incl. 1 KB each reserved)
constexpr int kMaxStageRows = 64;                                        // raw rows (channels) of one stage
constexpr int kSmemCtrlBytes = 64 + kMaxDT * 16 + 2 * (kMaxStageRows * 16 + 16);  // mbarrier, per-trial {row pointer, nout},
                                                                         // next stage's {RowDesc[], StageIndex} x 2
constexpr int kSmemDataBytes = kSmemBytes - kSmemCtrlBytes - 2 * kBlobBytes;  // variant region + raw-row region

// Per-stage blob, 32-bit words (copied to shared memory with one bulk copy):
//   [0] ngrp  [1] (worst-case lane interval ends here) | channels of the stage << 8  [2] ntask  [3] word offset of the trial_off table
//   [4 ..)        ngrp x { vbase | channels << 16, vlen, nent | ntog << 8 | ncorr << 16 | nvar << 24, cdesc_off | vdesc_off << 16 }
//                 (offsets inside the blob)
//   task table    ntask x { group | chunk << 8 }: warp task = kChunkU variant words of every variant of one group
//   cdesc         per group, ent_class(nent) entries of 2 words (the first nent are real, the rest repeat the first one
//                 without bit 26), in PREFIX ORDER (most-often-taken delta first; the first ntog have
//                 a delta that some trial takes); an entry is a channel at one of its shifts: bits 0-17 byte offset
//                 inside the raw region of the aligned 32-bit word (uint16 input: 8-byte unit) that holds the entry's sample
//                 at u = 0, bits 24-25 position of that sample inside it, bit 26 = the entry is the channel's smallest shift and adds
//                 it to the base sum.  The entry's delta (sample one later minus sample) moves its channel one later.
//                 Second word: what the kernel's realignment needs (uint8: bits 0-4 funnel-shift amount, bits 8-23 PRMT
//                 selector of the fifth sample; uint16: bits 0-1 = that position).
//   vdesc         per group: chain_words(ent_class(nent)) chain words, word k <= ntog = offset in the variant region of the variant "base sum
//                 + deltas of the first k entries" (0xffffffff: no trial uses it); then ncorr x { offset, mask } for the
//                 variants off the chain: all ntog deltas minus those in mask.  Headers, cdesc and vdesc are 16-byte
//                 aligned: the kernel reads them with 128-bit broadcast loads.
//   trial_off     ngrp x DT uint16 = word offset of the trial's read start in the variant region
constexpr int kBlobHdrWords = 4;
// The pre-sum code is straight-line over a fixed number of entries; a group runs the smallest instance that holds it.
constexpr int ent_class(int nent) { return nent <= 8 ? 8 : nent <= 12 ? 12 : 16; }
constexpr int chain_words(int cls) { return cls + 4; }   // cls + 1 chain words used at most, padded to 128-bit loads; corrections follow
constexpr uint32_t kEntryAddBase = 1u << 26;

struct RowDesc {            // one raw channel row of a stage; 16 bytes
    int32_t chan;
    int32_t astart;         // first element copied, relative to the tile's t0 (multiple of 16)
    int32_t nelem;          // elements to copy (multiple of 16)
    int32_t soff;           // byte offset inside the raw region (multiple of 16)
};

struct StageIndex {         // 16 bytes
    uint32_t blob_word0;    // first word of the stage's blob
    uint32_t blob_words;    // multiple of 4
    uint32_t row0;          // first RowDesc
    uint32_t nrows;
};

struct TileDesc {           // one DM tile of a range
    int32_t trial0;         // first trial (index inside the range)
    int32_t ntrial;         // <= DT
    int32_t stage0;
    int32_t nstage;
    int32_t skew0;          // first entry of the tile's DT per-trial output skews (RangePlan::skew)
    int32_t tshift;         // the block with time index i works on time tile (i - tshift) mod ntile_t: DM tiles that run
                            // together then read about the same stretch of the input (their delays differ)
    int32_t tt_last;        // last time tile in which some trial of the tile has a valid output (-1: none)
    int32_t pad_;
};

struct RangePlan {
    double dm_lo = 0, dm_step = 0;
    int32_t ndm = 0, decim = 1, trial0 = 0;
    int64_t nsamp_k = 0;         // floor(nsamp/decim)
    int64_t stride_k = 0;        // row stride (elements) of the series this range reads
    std::vector<int32_t> delay;  // [ndm][nchan]
    std::vector<int32_t> nout;   // [ndm]
    std::vector<int64_t> offset; // [ndm] int32 elements inside one beam's DM transform
    int32_t max_nout = 0;

    // tiled-kernel tables (host copies; built by build_tiling)
    std::vector<TileDesc> tiles;
    std::vector<StageIndex> sidx;
    std::vector<RowDesc> rows;
    std::vector<uint32_t> blob;
    std::vector<int32_t> skew;       // [ntiles_dm][DT]: trial i of a tile computes the outputs t0 - skew[i] + [0, kTT)
    int32_t skew_max = 0;
    int32_t vcap_words = 0;          // words of the variant region; the raw region follows it
    int32_t max_ent = 8;             // entry cap the tables were built for: selects the kernel instance
    int32_t kh = kHMax;              // packed words per trial per tile the tables were built for (tile = 2*kh outputs)
    int32_t ntile_t = 0;             // time tiles
    int64_t ngroups = 0, nvariants = 0, ncorrected = 0;   // totals, for reports (ncorrected: variants off the prefix chain)
    // work of the pre-sum over all DM tiles, for the cost model that picks the entry cap (build_tiling) and for reports:
    // warp tasks, entries processed (straight-line: the class size of each task's group), variants stored, rounds of 8 tasks
    int64_t ntasks = 0, task_entries = 0, task_variants = 0, presum_rounds = 0;
};

struct DeviceState;  // defined in api.cu

struct Plan {
    double fch1 = 0, foff = 0, tsamp = 0;
    int32_t nchan = 0;
    int64_t nsamp = 0;
    int32_t max_beams = 0;
    int64_t cand_capacity = 0;
    std::vector<int32_t> widths;
    std::vector<RangePlan> ranges;
    std::vector<RangePlan> compact;  // per range with decim > 1: the kernel tables for the 8-bit copy of its decimated series
                                     // (empty tables otherwise); built by build_tiling
    int32_t ntrials = 0;
    int64_t dmt_elems = 0;           // per beam
    // options
    int32_t opt_kernel = 0;          // 0 tiled, 1 naive
    int32_t opt_group = 0;           // channels per group, at most (0: 8 or 16, with the entry cap)
    int32_t opt_kh = 0;              // tile width in packed words: 224 or 256 (0: chosen per range by the cost model)
    int32_t opt_max_ent = 0;         // entries per group, at most: 8, 12 or 16 (0: chosen per range by the cost model)
    int32_t opt_dm_tile = 64;
    int32_t opt_profile = 0;
    int32_t opt_compact = 1;         // decimated ranges: dedisperse the 8-bit copy of the series when its values span < 256
    int32_t opt_peaks_lookup = 0;    // peak filter's S/N lookup: 0 by list density, 1 hash table, 2 dense plane, 3 dense plane of one beam
    int32_t opt_skew = 1;            // per-trial output skew inside a DM tile (0: all trials of a tile share t0)
    bool tiling_built = false;
    int64_t launches = 0;
    DeviceState* dev = nullptr;
};

// plan.cpp
int build_plan(Plan& p, const spt_dm_range* ranges, int32_t nranges);
int build_tiling(Plan& p);   // fills RangePlan::tiles/stages/groups/... for p.opt_group, p.opt_dm_tile
const RangePlan* range_of_trial(const Plan& p, int32_t trial, int32_t* local);

}  // namespace spt
