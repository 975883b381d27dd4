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

// ---- tiled dedispersion kernel geometry ---------------------------------------------
// A block owns DT trials x TT = 2*H output samples.  Packed 16-bit accumulator word q of a trial holds the
// outputs t0+q (low half) and t0+H+q (high half).
constexpr int kH = 512;              // words per trial per tile
constexpr int kTT = 2 * kH;          // output samples per tile
constexpr int kThreads = 512;        // 16 warps
constexpr int kMaxG = 8;             // channels per pre-summed group
constexpr int kSmemWords = 56 * 1024;  // 224 KB of the 227 KB a block may opt in to
constexpr int kMaxStageGroups = 32;  // groups per stage (bounds the per-stage tables kept in shared memory)
constexpr int kMaxDT = 64;           // trials per DM tile
constexpr int kTabWords = kMaxStageGroups * kMaxDT / 2;                 // trial_off slice of a stage (uint16)
constexpr int kDescWords = kMaxStageGroups * 10;                        // GroupDesc slice of a stage
constexpr int kStageDataWords = kSmemWords - kTabWords - kDescWords;    // variants + expansion rows

struct GroupDesc {          // one channel group of one (DM tile, stage); 40 bytes
    int32_t chan0;          // first channel
    int32_t nch;            // channels in the group (<= G; the last group of a band may be short)
    int32_t wlo;            // window start relative to the tile's t0, in samples, multiple of 4
    int32_t elen;           // words of each expanded channel row E_j[0 .. elen), multiple of 4
    int32_t vlen;           // words of each variant row P_r[0 .. vlen)
    int32_t nvar;           // variants R
    int32_t var0;           // index of the first variant's shift list in var_shift (x kMaxG)
    int32_t vbase;          // word offset of P_0 inside the stage's variant region
    int32_t ebase;          // word offset of E_0 inside the stage's expansion region (multiple of 4)
    int32_t pad_;
};

struct StageDesc {          // 32 bytes
    int32_t grp0;           // first GroupDesc
    int32_t ngrp;
    int32_t vwords;         // words of the variant region used by this stage
    int32_t ewords;         // words of the expansion region used by this stage
    int32_t flush;          // 1: packed accumulators must be flushed to int32 after this stage
    int32_t nvar;           // variants over all groups of the stage
    int32_t pad_[2];
};

struct TileDesc {           // one DM tile of a range
    int32_t trial0;         // first trial (index inside the range)
    int32_t ntrial;         // <= DT
    int32_t stage0;
    int32_t nstage;
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
    std::vector<StageDesc> stages;
    std::vector<GroupDesc> groups;
    std::vector<int16_t> var_shift;  // [nvariants][kMaxG] shift (>= 0) of channel j of variant r inside its E row
    std::vector<uint16_t> trial_off; // [groups.size()][DT] word offset of trial's read start inside the variant region
    int32_t ntile_t = 0;             // time tiles
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
    int32_t ntrials = 0;
    int64_t dmt_elems = 0;           // per beam
    // options
    int32_t opt_kernel = 0;          // 0 tiled, 1 naive
    int32_t opt_group = 4;
    int32_t opt_dm_tile = 64;
    int32_t opt_profile = 0;
    bool tiling_built = false;
    int64_t launches = 0;
    DeviceState* dev = nullptr;
};

// plan.cpp
int build_plan(Plan& p, const spt_dm_range* ranges, int32_t nranges);
int build_tiling(Plan& p);   // fills RangePlan::tiles/stages/groups/... for p.opt_group, p.opt_dm_tile
const RangePlan* range_of_trial(const Plan& p, int32_t trial, int32_t* local);

}  // namespace spt
