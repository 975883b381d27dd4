// plan.cpp -- host side of libspt: trial list, delay table, output geometry (a1 of SURVEY.md 8(a)) and the
// factorisation of the delay table that the tiled dedispersion kernel runs on.
//
// Delay law: PAPER.md:51-58 (Eq. 1-2), reference = highest frequency; constant and rounding per
// BASELINE.json north_star (2); readings A1-A4, B3 of DESIGN.md.  Compiled with FP contraction off.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <cstdlib>
#include <functional>
#include <map>
#include <new>
#include <system_error>
#include <thread>
#include <utility>

#include "internal.h"

namespace spt {

static inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

int build_plan(Plan& p, const spt_dm_range* ranges, int32_t nranges) {
    const double f_top = p.fch1;  // channel 0 is the reference (reading A1)
    const double inv_top = 1.0 / (f_top * f_top);
    int32_t trial0 = 0;
    int64_t off = 0;
    p.ranges.clear();
    p.ranges.reserve(nranges);
    for (int32_t r = 0; r < nranges; ++r) {
        RangePlan rp;
        rp.dm_lo = ranges[r].dm_lo;
        rp.dm_step = ranges[r].dm_step;
        rp.ndm = ranges[r].ndm;
        rp.decim = ranges[r].decim;
        rp.trial0 = trial0;
        rp.nsamp_k = p.nsamp / rp.decim;
        rp.stride_k = rp.decim == 1 ? p.nsamp : round_up(rp.nsamp_k, 16);
        rp.delay.resize((size_t)rp.ndm * p.nchan);
        rp.nout.resize(rp.ndm);
        rp.offset.resize(rp.ndm);
        const double tk = p.tsamp * (double)rp.decim;  // delays are rounded at the decimated sample period (A4)
        for (int32_t i = 0; i < rp.ndm; ++i) {
            const double dm = rp.dm_lo + (double)i * rp.dm_step;  // multiply, do not accumulate (A3)
            int32_t* row = &rp.delay[(size_t)i * p.nchan];
            for (int32_t c = 0; c < p.nchan; ++c) {
                const double f = p.fch1 + (double)c * p.foff;
                const double seconds = kDispersionConstantS * dm * (1.0 / (f * f) - inv_top);
                const double x = seconds / tk;
                if (!(x > -1.0e9 && x < 1.0e9)) return SPT_ERR_UNSUPPORTED;
                row[c] = (int32_t)std::floor(x + 0.5);
            }
            const int64_t n = rp.nsamp_k - (int64_t)row[p.nchan - 1];  // B3: every channel inside the data
            rp.nout[i] = (int32_t)std::max<int64_t>(0, std::min<int64_t>(n, rp.nsamp_k));
            rp.offset[i] = off;
            off += round_up(rp.nout[i], kRowAlignElems);
            rp.max_nout = std::max(rp.max_nout, rp.nout[i]);
            // the kernels assume what the physics guarantees for foff < 0, DM >= 0; refuse anything else
            for (int32_t c = 1; c < p.nchan; ++c)
                if (row[c] < row[c - 1]) return SPT_ERR_UNSUPPORTED;
            if (row[0] != 0) return SPT_ERR_UNSUPPORTED;
        }
        trial0 += rp.ndm;
        p.ranges.push_back(std::move(rp));
    }
    p.ntrials = trial0;
    p.dmt_elems = off;
    return SPT_OK;
}

const RangePlan* range_of_trial(const Plan& p, int32_t trial, int32_t* local) {
    for (const RangePlan& r : p.ranges)
        if (trial >= r.trial0 && trial < r.trial0 + r.ndm) {
            if (local) *local = trial - r.trial0;
            return &r;
        }
    return nullptr;
}

// -------------------------------------------------------------------------------------------------------------
// Factorisation of the delay table for the tiled kernel.
//
// For a DM tile (DT consecutive trials) and a group of up to 8 adjacent channels c0..c0+n-1 write
//     delay[d][c0+j] = dmin + b(d) + s_j + tau_j(d),      dmin = min_d delay[d][c0],  b(d) >= 0,  s_0 = tau_0 = 0,
// where s_j is the smallest delay of channel j relative to channel c0 over the tile and tau_j(d) is 0 or 1 (a group
// is halved until that holds: the true relative delay drifts by less than a sample over a tile of close trials, so
// its rounded value toggles between two neighbours).  The bit vectors tau(d) take only a few distinct values over the
// tile ("variants"), so
//     out[d][t] = sum_groups P_{r(d)}[ t - t0 + b(d) ],     P_r[u] = sum_j y[c0+j][t0 + dmin + u + s_j + tau^r_j]
// is the SAME integer sum as the definition, with every P_r built once per tile and shared by its trials.
// tau_j(d) = [theta(d) >= threshold_j] up to the slow drift, so ordered by how often they are 1 the channels form a
// chain: most variants are "the first k channels of the order take the alternate shift".  The kernel walks that chain
// with one vector add per step; a variant off the chain carries correction masks.
// -------------------------------------------------------------------------------------------------------------
namespace {

// cost model of build_range_auto (see modelled_cost)
constexpr double kCostGroup = 2.348, kCostStage = 0.876, kCostPresum = 0.02205, kPen12Wide = 1.6, kPen12Narrow = 1.5;

struct PendingVariant { int k; uint32_t plus, minus, bits; };

struct PendingEntry { int j, level; bool addbase; int ones; };   // one pre-sum entry: channel offset j at shift s_j + level

struct PendingGroup {
    int32_t chan0, nch, dmin, vlen, nvar, nent, ntog;
    std::vector<PendingEntry> ent;            // prefix order (most often taken delta first)
    std::vector<int16_t> smin, smax;          // [nch] by channel offset j
    std::vector<PendingVariant> vars;         // sorted by k
    std::vector<int> var_of;                  // [ntrial]
    std::vector<int32_t> b;                   // [ntrial]
    std::vector<RowDesc> rows;                // [nch] by channel offset j, soff relative to the group's first row
    int32_t raw_bytes, vwords, ncorrected;
};

inline int popcount32(uint32_t x) { return __builtin_popcount(x); }

}  // namespace

// Entries of a group: every channel has one entry at its smallest relative delay s_j (it adds the channel to the
// base sum); a channel whose relative delay reaches s_j + L over the tile has L entries, at s_j .. s_j+L-1, and the
// delta of the entry at level l (sample one later minus sample) moves the channel from s_j+l to s_j+l+1: bit
// "tau_j > l".  Bits sorted by how often they are set form the prefix chain.
// skew[i] (tile local): trial i's output window starts skew[i] samples early, i.e. its effective delays are
// delay - skew[i] (they may be negative); relative delays between channels do not change.
static bool make_group(const Plan& p, const RangePlan& rp, int32_t d0, int32_t ntrial, int32_t c0, int G, int max_ent, int es,
                       const int32_t* skew, PendingGroup& g) {
    g.chan0 = c0;
    int32_t dmin = INT32_MAX, dmax = INT32_MIN;
    for (int i = 0; i < ntrial; ++i) {
        const int32_t v = rp.delay[(size_t)(d0 + i) * p.nchan + c0] - skew[i];
        dmin = std::min(dmin, v); dmax = std::max(dmax, v);
    }
    g.dmin = dmin;
    const int kH = rp.kh;
    g.vlen = (int32_t)round_up(kH + (dmax - dmin), 4);
    g.b.resize(ntrial);
    for (int i = 0; i < ntrial; ++i) g.b[i] = rp.delay[(size_t)(d0 + i) * p.nchan + c0] - skew[i] - dmin;
    g.var_of.assign(ntrial, 0);
    // the group shrinks until its entries fit the kernel's registers and the variants are few (widely spaced
    // channels at high DM have a different relative delay for every trial: nothing to share)
    for (int gsize = std::min(G, p.nchan - c0);; --gsize) {
        g.nch = gsize;
        g.smin.assign(gsize, 0);
        g.smax.assign(gsize, 0);
        int nent = 0;
        bool ok = true;
        for (int j = 0; j < gsize && ok; ++j) {
            int lo = INT32_MAX, hi = INT32_MIN;
            for (int i = 0; i < ntrial; ++i) {
                const int32_t* row = &rp.delay[(size_t)(d0 + i) * p.nchan + c0];
                const int s = row[j] - row[0];
                lo = std::min(lo, s); hi = std::max(hi, s);
            }
            if (lo < 0 || hi > 30000) return false;
            g.smin[j] = (int16_t)lo; g.smax[j] = (int16_t)hi;
            nent += std::max(1, hi - lo);
            if (nent > max_ent) ok = false;
        }
        if (!ok) continue;   // gsize == 1 always passes: channel c0 relative to itself
        g.ent.clear();
        for (int j = 0; j < gsize; ++j)
            for (int l = 0; l < std::max(1, g.smax[j] - g.smin[j]); ++l) g.ent.push_back({j, l, l == 0, 0});
        for (int i = 0; i < ntrial; ++i) {
            const int32_t* row = &rp.delay[(size_t)(d0 + i) * p.nchan + c0];
            for (PendingEntry& e : g.ent)
                if (row[e.j] - row[0] - g.smin[e.j] > e.level) e.ones++;
        }
        std::stable_sort(g.ent.begin(), g.ent.end(), [](const PendingEntry& a, const PendingEntry& b) { return a.ones > b.ones; });
        int ntog = 0;
        for (const PendingEntry& e : g.ent) ntog += e.ones > 0;
        g.ntog = ntog;
        // distinct variants, as bit masks over the positions of the prefix order
        std::map<uint32_t, int> seen;
        std::vector<uint32_t> bits_of_trial(ntrial);
        for (int i = 0; i < ntrial; ++i) {
            const int32_t* row = &rp.delay[(size_t)(d0 + i) * p.nchan + c0];
            uint32_t m = 0;
            for (int q = 0; q < (int)g.ent.size(); ++q)
                if (row[g.ent[q].j] - row[0] - g.smin[g.ent[q].j] > g.ent[q].level) m |= 1u << q;
            bits_of_trial[i] = m;
            seen.emplace(m, 0);
        }
        if ((int)seen.size() > kMaxVar) continue;   // gsize == 1 has exactly one variant
        g.vars.clear();
        for (auto& kv : seen) {
            PendingVariant v{0, 0, 0, kv.first};
            int best = 1 << 30;
            for (int k = 0; k <= ntog; ++k) {
                const uint32_t pre = (1u << k) - 1u;
                const int cost = popcount32(kv.first ^ pre);
                if (cost < best) { best = cost; v.k = k; v.plus = kv.first & ~pre; v.minus = pre & ~kv.first; }
            }
            g.vars.push_back(v);
        }
        std::stable_sort(g.vars.begin(), g.vars.end(), [](const PendingVariant& a, const PendingVariant& b) { return a.k < b.k; });
        g.ncorrected = 0;
        for (size_t r = 0; r < g.vars.size(); ++r) {
            seen[g.vars[r].bits] = (int)r;
            g.ncorrected += (g.vars[r].plus | g.vars[r].minus) != 0;
        }
        for (int i = 0; i < ntrial; ++i) g.var_of[i] = seen[bits_of_trial[i]];
        break;
    }
    g.nent = (int32_t)g.ent.size();
    g.nvar = (int32_t)g.vars.size();
    g.vwords = g.nvar * g.vlen;
    g.rows.resize(g.nch);
    g.raw_bytes = 0;
    for (int j = 0; j < g.nch; ++j) {
        RowDesc& r = g.rows[j];
        r.chan = c0 + j;
        r.astart = (dmin + g.smin[j]) & ~15;
        // last element a pre-sum task touches: u = vlen-1 at the largest shift in the high half, plus the words
        // its aligned 32-bit loads reach past it
        const int32_t last = dmin + std::max<int>(g.smax[j], g.smin[j] + 1) + g.vlen + kH + 8;
        r.nelem = (int32_t)round_up(last - r.astart, 16);
        r.soff = g.raw_bytes;
        g.raw_bytes += r.nelem * es;
    }
    return true;
}

// Tables of one DM range for groups of at most G channels and max_ent entries.
// compact: tables for the 8-bit copy of a decimated series (sample - smallest sample of the series, made when that fits a
// byte): one byte per element and, like the raw input, at most 255 per sample whatever the decimation.
static int build_range(const Plan& p, RangePlan& rp, const int G, const int max_ent, const bool compact = false) {
    const int DT = p.opt_dm_tile;
    const int kTT = 2 * rp.kh;           // rp.kh is set by the caller
    rp.max_ent = max_ent;
    {
        rp.tiles.clear(); rp.sidx.clear(); rp.rows.clear(); rp.blob.clear();
        rp.ngroups = rp.nvariants = rp.ncorrected = 0;
        rp.ntasks = rp.task_entries = rp.task_variants = rp.presum_rounds = 0;
        // Output skew per trial: trial i of a DM tile computes the outputs t0 - skew[i] + [0, kTT)
        // with skew[i] = delay[i][cref] - delay[0][cref], so that at channel cref all trials of the tile read the same
        // window and elsewhere the windows spread by |delay slope(c) - delay slope(cref)| only.  cref minimises the sum
        // of the spreads over the band.
        rp.skew.assign((size_t)((rp.ndm + DT - 1) / DT) * DT, 0);
        rp.skew_max = 0;
        for (int32_t d0 = 0; d0 < rp.ndm && p.opt_skew; d0 += DT) {
            const int32_t nt = std::min(DT, rp.ndm - d0);
            int64_t best = -1;
            int32_t best_c = 0;
            for (int32_t cref = 0; cref < p.nchan; cref += std::max(1, p.nchan / 64)) {
                int64_t sum = 0;
                for (int32_t c = 0; c < p.nchan; c += 8) {
                    int32_t lo = INT32_MAX, hi = INT32_MIN;
                    for (int i = 0; i < nt; ++i) {
                        const int32_t* row = &rp.delay[(size_t)(d0 + i) * p.nchan];
                        const int32_t v = row[c] - (row[cref] - rp.delay[(size_t)d0 * p.nchan + cref]);
                        lo = std::min(lo, v); hi = std::max(hi, v);
                    }
                    sum += hi - lo;
                }
                if (best < 0 || sum < best) { best = sum; best_c = cref; }
            }
            for (int i = 0; i < DT; ++i) {
                const int ii = std::min(i, nt - 1);
                const int32_t sk = rp.delay[(size_t)(d0 + ii) * p.nchan + best_c] - rp.delay[(size_t)d0 * p.nchan + best_c];
                rp.skew[(size_t)(d0 / DT) * DT + i] = sk;      // >= 0: delays grow with DM
                rp.skew_max = std::max(rp.skew_max, sk);
            }
        }
        rp.ntile_t = (int32_t)((rp.max_nout + rp.skew_max + kTT - 1) / kTT);
        const int es = (rp.decim == 1 || compact) ? 1 : 2;
        // 16-bit lanes hold sums of at most floor(65535 / (255*decim)) channel samples
        const int lane_channels = 65535 / (255 * (compact ? 1 : rp.decim));
        if (lane_channels < 1) return SPT_ERR_UNSUPPORTED;
        // split of the data region between variants and raw rows: from the needs of the middle DM tile
        {
            const int32_t d0 = (rp.ndm / DT / 2) * DT;
            const int32_t nt = std::min(DT, rp.ndm - d0);
            int64_t vb = 0, rb = 0;
            for (int32_t c = 0; c < p.nchan;) {
                PendingGroup g;
                if (!make_group(p, rp, d0, nt, c, G, max_ent, es, &rp.skew[(size_t)(d0 / DT) * DT], g)) return SPT_ERR_UNSUPPORTED;
                vb += (int64_t)g.vwords * 4; rb += g.raw_bytes;
                c += g.nch;
            }
            int64_t v = (int64_t)((double)kSmemDataBytes * (double)vb / (double)(vb + rb));
            v = std::min<int64_t>(std::max<int64_t>(v, kSmemDataBytes / 4), (int64_t)kSmemDataBytes * 7 / 8);
            v = std::min<int64_t>(v, 65535 * 4);
            rp.vcap_words = (int32_t)(v / 16 * 4);
        }
        const int64_t rcap_bytes = kSmemDataBytes - (int64_t)rp.vcap_words * 4;

        for (int32_t d0 = 0; d0 < rp.ndm; d0 += DT) {
            TileDesc td{};
            td.skew0 = (d0 / DT) * DT;
            td.trial0 = d0;
            td.ntrial = std::min(DT, rp.ndm - d0);
            td.tshift = rp.delay[(size_t)(d0 + td.ntrial / 2) * p.nchan + p.nchan / 2] / kTT;   // median delay over the channels
            td.tt_last = -1;
            for (int i = 0; i < td.ntrial; ++i)
                if (rp.nout[d0 + i] > 0)
                    td.tt_last = std::max(td.tt_last, (rp.nout[d0 + i] - 1 + rp.skew[(size_t)td.skew0 + i]) / kTT);
            td.stage0 = (int32_t)rp.sidx.size();
            std::vector<PendingGroup> open;
            auto blob_words_of = [&](const std::vector<PendingGroup>& gs, const PendingGroup* extra) {
                int64_t w = kBlobHdrWords + 4;
                auto one = [&](const PendingGroup& g) {
                    w += 4 + (g.vlen + kChunkU - 1) / kChunkU + 2 * ent_class(g.nent) + chain_words(ent_class(g.nent)) + 2 * g.ncorrected + 3 + DT / 2;
                };
                for (const PendingGroup& g : gs) one(g);
                if (extra) one(*extra);
                return w;
            };
            auto close_stage = [&](bool flush) {
                if (open.empty()) return;
                StageIndex si;
                si.blob_word0 = (uint32_t)rp.blob.size();
                si.row0 = (uint32_t)rp.rows.size();
                const size_t ngrp = open.size();
                std::vector<uint32_t> hdr(kBlobHdrWords + 4 * ngrp), tasks, cdesc, vdesc;
                std::vector<uint16_t> toff;
                int32_t vbase = 0, rbase = 0;
                for (size_t k = 0; k < ngrp; ++k)
                    for (int ch = 0; ch < (open[k].vlen + kChunkU - 1) / kChunkU; ++ch)
                        tasks.push_back((uint32_t)k | ((uint32_t)ch << 8));
                const uint32_t ntask = (uint32_t)tasks.size();
                while ((hdr.size() + tasks.size()) % 4) tasks.push_back(0xffffffffu);   // 128-bit loads of the descriptors
                const uint32_t cdesc0 = (uint32_t)(hdr.size() + tasks.size());
                for (size_t k = 0; k < ngrp; ++k) {
                    PendingGroup& g = open[k];
                    const uint32_t my_cdesc = cdesc0 + (uint32_t)cdesc.size();
                    for (int j = 0; j < g.nch; ++j) {
                        RowDesc r = g.rows[j];
                        r.soff += rbase;
                        rp.rows.push_back(r);
                    }
                    for (const PendingEntry& en : g.ent) {
                        const RowDesc& r = g.rows[en.j];
                        const int32_t e0 = g.dmin + g.smin[en.j] + en.level - r.astart;   // element of the entry's u = 0 sample
                        const uint32_t byte = (uint32_t)(rbase + r.soff + e0 * es);
                        // uint8: aligned 32-bit word + byte position; uint16: aligned 8-byte unit + sample position in it
                        const uint32_t a0 = es == 1 ? (byte & 3u) : ((byte >> 1) & 3u);
                        cdesc.push_back((es == 1 ? (byte & ~3u) : (byte & ~7u)) | (a0 << 24) | (en.addbase ? kEntryAddBase : 0u));
                        // second word, ready for the kernel: uint8: funnel-shift amount and the PRMT selector of sample 4
                        cdesc.push_back(es == 1 ? (a0 * 8u) | ((a0 * 0x1111u + 0x4400u) << 8) : a0);
                    }
                    for (int q = g.nent; q < ent_class(g.nent); ++q) {   // padding: straight-line code in the kernel; deltas never taken
                        const uint32_t c0 = cdesc[cdesc.size() - 2 * (size_t)g.nent], c1 = cdesc[cdesc.size() - 2 * (size_t)g.nent + 1];
                        cdesc.push_back(c0 & ~kEntryAddBase);
                        cdesc.push_back(c1);
                    }
                    hdr[kBlobHdrWords + 4 * k + 0] = (uint32_t)vbase | ((uint32_t)g.nch << 16);
                    hdr[kBlobHdrWords + 4 * k + 1] = (uint32_t)g.vlen;
                    hdr[kBlobHdrWords + 4 * k + 2] = (uint32_t)g.nent | ((uint32_t)g.ntog << 8) | ((uint32_t)g.ncorrected << 16) | ((uint32_t)g.nvar << 24);
                    hdr[kBlobHdrWords + 4 * k + 3] = my_cdesc;                     // vdesc offset patched below
                    for (int i = 0; i < DT; ++i) {
                        const int ii = std::min(i, td.ntrial - 1);  // unused trial slots alias the last valid trial
                        toff.push_back((uint16_t)(vbase + g.var_of[ii] * g.vlen + g.b[ii]));
                    }
                    vbase += g.vwords;
                    rbase += g.raw_bytes;
                    rp.ngroups++; rp.nvariants += g.nvar; rp.ncorrected += g.ncorrected;
                    const int64_t nt = (g.vlen + kChunkU - 1) / kChunkU;
                    rp.ntasks += nt; rp.task_entries += nt * ent_class(g.nent); rp.task_variants += nt * g.nvar;
                }
                const uint32_t vdesc0 = cdesc0 + (uint32_t)cdesc.size();
                vbase = 0;
                for (size_t k = 0; k < ngrp; ++k) {
                    PendingGroup& g = open[k];
                    hdr[kBlobHdrWords + 4 * k + 3] |= (vdesc0 + (uint32_t)vdesc.size()) << 16;
                    // chain: the variant that is exactly "first k deltas taken", k = 0..ntog (or none)
                    for (int k2 = 0; k2 <= g.ntog; ++k2) {
                        uint32_t dst = 0xffffffffu;
                        for (int r = 0; r < g.nvar; ++r)
                            if (g.vars[r].k == k2 && !(g.vars[r].plus | g.vars[r].minus)) dst = (uint32_t)(vbase + r * g.vlen);
                        vdesc.push_back(dst);
                    }
                    for (int k2 = g.ntog + 1; k2 < chain_words(ent_class(g.nent)); ++k2) vdesc.push_back(0xffffffffu);   // whole 128-bit loads
                    // off the chain: destination and the mask of the deltas NOT taken (subtracted from the full sum)
                    for (int r = 0; r < g.nvar; ++r)
                        if (g.vars[r].plus | g.vars[r].minus) {
                            vdesc.push_back((uint32_t)(vbase + r * g.vlen));
                            vdesc.push_back(~g.vars[r].bits & ((1u << g.ntog) - 1u));
                        }
                    while (vdesc.size() % 4) vdesc.push_back(0);
                    vbase += g.vwords;
                }
                int nch_stage = 0;
                for (const PendingGroup& g : open) nch_stage += g.nch;
                hdr[0] = (uint32_t)ngrp; hdr[1] = (flush ? 1u : 0u) | ((uint32_t)nch_stage << 8); hdr[2] = ntask;
                rp.presum_rounds += (ntask + kThreads / 32 - 1) / (kThreads / 32);
                while ((vdesc0 + vdesc.size()) % 4) vdesc.push_back(0);   // trial_off rows are read with 128-bit loads
                hdr[3] = vdesc0 + (uint32_t)vdesc.size();
                rp.blob.insert(rp.blob.end(), hdr.begin(), hdr.end());
                rp.blob.insert(rp.blob.end(), tasks.begin(), tasks.end());
                rp.blob.insert(rp.blob.end(), cdesc.begin(), cdesc.end());
                rp.blob.insert(rp.blob.end(), vdesc.begin(), vdesc.end());
                for (size_t i = 0; i < toff.size(); i += 2)
                    rp.blob.push_back((uint32_t)toff[i] | ((uint32_t)(i + 1 < toff.size() ? toff[i + 1] : 0) << 16));
                while ((rp.blob.size() - si.blob_word0) % 4) rp.blob.push_back(0);
                si.blob_words = (uint32_t)(rp.blob.size() - si.blob_word0);
                si.nrows = (uint32_t)(rp.rows.size() - si.row0);
                rp.sidx.push_back(si);
                open.clear();
            };
            // all groups of the tile first, then the cut into stages
            std::vector<PendingGroup> all;
            for (int32_t c = 0; c < p.nchan;) {
                PendingGroup g;
                if (!make_group(p, rp, d0, td.ntrial, c, std::min(G, lane_channels), max_ent, es, &rp.skew[(size_t)(d0 / DT) * DT], g))
                    return SPT_ERR_UNSUPPORTED;
                c += g.nch;
                if (g.vwords > rp.vcap_words || g.raw_bytes > rcap_bytes || blob_words_of({}, &g) * 4 > kBlobBytes)
                    return SPT_ERR_UNSUPPORTED;  // one group must fit a stage
                all.push_back(std::move(g));
            }
            // A stage costs ceil(tasks / warps) pre-sum rounds plus a fixed overhead (barriers, bulk-copy issue, tables) of
            // about one round; its groups must fit shared memory and the table blob, and its channels one worst-case lane
            // interval (the kernel widens the lanes between stages, never inside one).  Take, from every starting group,
            // the feasible prefix with the lowest cost per channel: 15 tasks in two rounds beat 18 tasks in three.
            constexpr int kWarps = kThreads / 32;
            constexpr double kStageOverheadRounds = 1.0;
            for (size_t i0 = 0; i0 < all.size();) {
                int64_t v = 0, r = 0, words = kBlobHdrWords + 4;
                int nch = 0, tasks = 0;
                size_t best_n = 1;
                double best_cost = 1e300;
                for (size_t n = 1; i0 + n <= all.size() && n <= (size_t)kMaxStageGroups; ++n) {
                    const PendingGroup& g = all[i0 + n - 1];
                    v += g.vwords; r += g.raw_bytes; nch += g.nch;
                    words += 4 + (g.vlen + kChunkU - 1) / kChunkU + 2 * ent_class(g.nent) + chain_words(ent_class(g.nent)) + 2 * g.ncorrected + 3 + DT / 2;
                    tasks += (g.vlen + kChunkU - 1) / kChunkU;
                    if (n > 1 && (v > rp.vcap_words || r > rcap_bytes || words * 4 > kBlobBytes || nch > lane_channels || nch > kMaxStageRows)) break;
                    const double cost = ((tasks + kWarps - 1) / kWarps + kStageOverheadRounds) / nch;
                    if (cost <= best_cost) { best_cost = cost; best_n = n; }
                }
                for (size_t n = 0; n < best_n; ++n) open.push_back(std::move(all[i0 + n]));
                close_stage(false);
                i0 += best_n;
            }
            td.nstage = (int32_t)rp.sidx.size() - td.stage0;
            rp.tiles.push_back(td);
        }
        // a stage's transaction also fetches the NEXT stage's index and a fixed-size slice of its rows: pad the arrays
        rp.sidx.push_back(StageIndex{0, 0, 0, 0});
        rp.rows.resize(rp.rows.size() + kMaxStageRows, RowDesc{0, 0, 0, 0});
    }
    return SPT_OK;
}

// Modelled time of a range's launch, in ms per beam up to a common factor ("Entry cap and tile
// width"): per time tile the gather costs per group in proportion to the tile width, the stage loop per stage, the pre-sum
// per entry processed and variant stored; the 12- and 16-entry pre-sum instances run slower per unit of work than the
// 8-entry one (register pressure: fewer loads in flight).  Constants fitted to eight measured range-0 launches -- configs 3
// and 6 at tile widths 224 / 256 and caps 8 / 12 -- which the model reproduces within 0.3 ms (1.5 %).
static double modelled_cost(const RangePlan& rp) {
    const bool wide = rp.kh >= 256;
    const double pen = rp.max_ent <= 8 ? 1.0 : rp.max_ent <= 12 ? (wide ? kPen12Wide : kPen12Narrow) : (wide ? 2.2 : 2.0);
    const double nstage = (double)rp.sidx.size() - 1.0;
    const double tile = kCostGroup * (double)rp.ngroups * ((double)rp.kh / 256.0) + kCostStage * nstage +
                        kCostPresum * pen * (double)(rp.task_entries + rp.task_variants);
    return 1e-6 * (double)rp.ntile_t * tile;
}

static int build_range_auto(const Plan& p, RangePlan& rp, bool compact);

int build_tiling(Plan& p) {
    p.compact.clear();
    p.compact.resize(p.ranges.size());
    // the ranges are independent of each other: one thread each (every thread touches only its own RangePlan entries)
    auto build_one = [&p](size_t i) -> int {
        const int rc = build_range_auto(p, p.ranges[i], false);
        if (rc != SPT_OK) return rc;
        if (p.ranges[i].decim > 1 && p.opt_compact) {
            // second set of tables for the 8-bit copy of the decimated series (the delay table is shared by value: a few MB)
            // Both sets run in one kernel instance, so they share tile width and entry cap: the copy's choice (it is the set
            // that runs on well-behaved data), and the same DM tiles and skews, so that a block does the same tile either way.
            // The uint16 rows are twice as large, so the copy's choice may not build for them (build_range_auto may have
            // rejected exactly that combination): the range then keeps the tables chosen for the uint16 series alone and
            // has no 8-bit copy -- a working plan, one launch on the uint16 series -- instead of failing the whole plan.
            RangePlan own = p.ranges[i];
            p.compact[i] = p.ranges[i];
            bool ok = build_range_auto(p, p.compact[i], true) == SPT_OK;
            if (ok && (p.compact[i].max_ent != p.ranges[i].max_ent || p.compact[i].kh != p.ranges[i].kh)) {
                const int G = p.opt_group ? p.opt_group : (p.compact[i].max_ent > 8 ? 16 : 8);
                p.ranges[i].kh = p.compact[i].kh;
                ok = build_range(p, p.ranges[i], G, p.compact[i].max_ent, false) == SPT_OK;
            }
            if (ok && (p.compact[i].ntile_t != p.ranges[i].ntile_t || p.compact[i].tiles.size() != p.ranges[i].tiles.size() ||
                       p.compact[i].skew != p.ranges[i].skew))
                ok = false;
            if (!ok) {
                p.ranges[i] = std::move(own);
                p.compact[i] = RangePlan();
            }
        }
        return SPT_OK;
    };
    std::vector<int> rcs(p.ranges.size(), SPT_OK);
    auto guarded = [&](size_t i) {
        try {
            rcs[i] = build_one(i);
        } catch (const std::bad_alloc&) {
            rcs[i] = SPT_ERR_NOMEM;
        }
    };
    {
        std::vector<std::thread> workers;
        for (size_t i = 1; i < p.ranges.size(); ++i) {
            try {
                workers.emplace_back(guarded, i);
            } catch (const std::system_error&) {
                guarded(i);
            }
        }
        if (!p.ranges.empty()) guarded(0);
        for (auto& t : workers) t.join();
    }
    for (int rc : rcs)
        if (rc != SPT_OK) return rc;
    p.tiling_built = true;
    return SPT_OK;
}

// Tile width and entry cap of one range: what the caller fixed (A/B runs, tests), else the cheapest by the model of
// {256, 224 words} x {8, 12 entries} -- wide tiles and small groups for long sweeps (every channel of a group toggles
// within a DM tile, the pre-sum dominates), narrower tiles and larger groups where sweeps are short (a variant plus its
// small halo then fills two pre-sum tasks instead of spilling into a third).
static int build_range_auto(const Plan& p, RangePlan& rp, const bool compact) {
    const int khs[2] = {256, 224};
    const int caps[2] = {8, 12};
    // the candidates the options leave, in the order the choice prefers on equal cost ...
    struct Cand { int kh, use_cap, G; bool last; RangePlan plan; int rc; };
    std::vector<Cand> cands;
    for (int kh : khs) {
        if (p.opt_kh != 0 && kh != p.opt_kh) continue;
        if (p.opt_kh == 0 && kh != 256 && p.opt_dm_tile != 64) continue;     // the narrow tile exists for 64-trial tiles only
        for (int cap : caps) {
            if (p.opt_max_ent != 0 && cap != p.opt_max_ent && !(p.opt_max_ent == 16 && cap == 12)) continue;
            const int use_cap = (p.opt_max_ent == 16) ? 16 : cap;
            if (p.opt_max_ent == 0 && p.opt_group != 0 && p.opt_group <= 8 && cap > 8) continue;
            const int G = p.opt_group ? p.opt_group : (use_cap > 8 ? 16 : 8);
            cands.push_back(Cand{kh, use_cap, G, kh == khs[1] && cap == caps[1], RangePlan(), SPT_OK});
        }
    }
    // ... each built on its own thread (a plan is built per band; the tables of one candidate of the config-3
    // plan take about a second, and build_range only reads the plan and writes its own RangePlan)
    auto build_one = [&](Cand& c) {
        try {
            c.plan = rp;
            c.plan.kh = c.kh;
            c.rc = build_range(p, c.plan, c.G, c.use_cap, compact);
        } catch (const std::bad_alloc&) {
            c.rc = SPT_ERR_NOMEM;
        }
    };
    {
        std::vector<std::thread> workers;
        for (size_t i = 1; i < cands.size(); ++i) {
            try {
                workers.emplace_back(build_one, std::ref(cands[i]));
            } catch (const std::system_error&) {
                build_one(cands[i]);                                          // no more threads: build it here
            }
        }
        if (!cands.empty()) build_one(cands[0]);
        for (auto& t : workers) t.join();
    }
    bool have = false;
    double best = 0.0;
    RangePlan keep;
    for (Cand& c : cands) {
        if (c.rc != SPT_OK) {
            if (!have && c.last) return c.rc;
            continue;
        }
        // a margin for the decimated uint16 series, whose pre-sum the constants fit less well: stay with the default there
        double cost = modelled_cost(c.plan);
        if (!(c.kh == 256 && c.use_cap == 8)) cost *= (rp.decim == 1 || compact) ? 1.03 : 1.10;
        if (!have || cost < best) { best = cost; keep = std::move(c.plan); have = true; }
    }
    if (!have) return SPT_ERR_UNSUPPORTED;
    rp = std::move(keep);
    return SPT_OK;
}

}  // namespace spt
