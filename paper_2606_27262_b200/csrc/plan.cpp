// plan.cpp -- host side of libspt: trial list, delay table, output geometry (a1 of SURVEY.md 8(a)) and the
// factorisation of the delay table that the tiled dedispersion kernel runs on.
//
// Delay law: PAPER.md:51-58 (Eq. 1-2), reference = highest frequency; constant and rounding per
// BASELINE.json north_star (2); readings A1-A4, B3 of DESIGN.md.  Compiled with FP contraction off.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
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
// For a DM tile (DT consecutive trials) and a group of G adjacent channels c0..c0+G-1 write
//     delay[d][c0+j] = dmin + b(d) + rho_j(d),      dmin = min_d delay[d][c0],  b(d) >= 0,  rho_0 = 0.
// Over the DT trials the vector rho(d) takes only a handful of distinct values ("variants": each rho_j toggles
// between floor and ceil of the slowly varying true relative delay), so
//     out[d][t] = sum_groups P_{r(d)}[ t - t0 + b(d) ],     P_r[u] = sum_j y[c0+j][t0 + dmin + u + rho^r_j]
// is the SAME integer sum as the definition, with every P_r built once per tile and shared by the trials.
// The kernel builds all P_r of a group in one sweep over the (channel, shift) pairs the variants use: the most
// used shift of a channel is its "base" pair (added for every variant), every other shift a "delta" pair that
// replaces the base for the variants in its mask.
// -------------------------------------------------------------------------------------------------------------
namespace {

struct PendingGroup {
    int32_t chan0, nch, dmin, vlen, nvar;
    std::vector<std::vector<int16_t>> vars;   // [nvar][nch] rho
    std::vector<int> var_of;                  // [ntrial]
    std::vector<int32_t> b;                   // [ntrial]
    std::vector<RowDesc> rows;                // [nch], soff relative to the group's first row
    int32_t raw_bytes, vwords, npairs;
};

}  // namespace

static bool make_group(const Plan& p, const RangePlan& rp, int32_t d0, int32_t ntrial, int32_t c0, int G, int es,
                       PendingGroup& g) {
    g.chan0 = c0;
    int32_t dmin = INT32_MAX, dmax = 0;
    for (int i = 0; i < ntrial; ++i) {
        const int32_t v = rp.delay[(size_t)(d0 + i) * p.nchan + c0];
        dmin = std::min(dmin, v); dmax = std::max(dmax, v);
    }
    g.dmin = dmin;
    g.vlen = kH + (dmax - dmin);
    g.b.resize(ntrial);
    for (int i = 0; i < ntrial; ++i) g.b[i] = rp.delay[(size_t)(d0 + i) * p.nchan + c0] - dmin;
    g.var_of.assign(ntrial, 0);
    // distinct relative-delay vectors of the tile's trials; the group is halved until they are few (widely spaced
    // channels at high DM have a different vector for every trial: nothing to share)
    for (int gsize = std::min(G, p.nchan - c0);; gsize >>= 1) {
        std::map<std::vector<int16_t>, int> seen;
        g.vars.clear();
        g.nch = gsize;
        for (int i = 0; i < ntrial; ++i) {
            const int32_t* row = &rp.delay[(size_t)(d0 + i) * p.nchan + c0];
            std::vector<int16_t> rho(gsize, 0);
            for (int j = 0; j < gsize; ++j) {
                const int s = row[j] - row[0];
                if (s > 30000) return false;
                rho[j] = (int16_t)s;
            }
            auto it = seen.find(rho);
            if (it == seen.end()) {
                it = seen.emplace(rho, (int)g.vars.size()).first;
                g.vars.push_back(rho);
            }
            g.var_of[i] = it->second;
        }
        if (gsize == 1 || (int)g.vars.size() <= kMaxVar) break;
    }
    g.nvar = (int32_t)g.vars.size();
    g.vwords = g.nvar * g.vlen;
    g.rows.resize(g.nch);
    g.raw_bytes = 0;
    g.npairs = 0;
    for (int j = 0; j < g.nch; ++j) {
        int rmin = INT32_MAX, rmax = 0;
        std::vector<int> shifts;
        for (auto& v : g.vars) {
            rmin = std::min<int>(rmin, v[j]); rmax = std::max<int>(rmax, v[j]);
            if (std::find(shifts.begin(), shifts.end(), (int)v[j]) == shifts.end()) shifts.push_back(v[j]);
        }
        g.npairs += (int32_t)shifts.size();
        RowDesc& r = g.rows[j];
        r.chan = c0 + j;
        r.astart = (dmin + rmin) & ~15;
        const int32_t last = dmin + rmax + (g.vlen - 1) + kH;   // last element any valid output can need
        r.nelem = (int32_t)((last + 1 + kRowSlack - r.astart + 15) / 16 * 16);
        r.soff = g.raw_bytes;
        g.raw_bytes += r.nelem * es;
    }
    return true;
}

int build_tiling(Plan& p) {
    const int G = p.opt_group, DT = p.opt_dm_tile;
    for (RangePlan& rp : p.ranges) {
        rp.tiles.clear(); rp.sidx.clear(); rp.rows.clear(); rp.blob.clear();
        rp.ngroups = rp.nvariants = rp.npairs = 0;
        rp.ntile_t = (int32_t)((rp.max_nout + kTT - 1) / kTT);
        const int es = rp.decim == 1 ? 1 : 2;
        // 16-bit lanes hold sums of at most floor(65535 / (255*decim)) channel samples
        const int lane_channels = 65535 / (255 * rp.decim);
        if (lane_channels < 1) return SPT_ERR_UNSUPPORTED;
        // split of the data region between variants and raw rows: from the needs of the middle DM tile
        {
            const int32_t d0 = (rp.ndm / DT / 2) * DT;
            const int32_t nt = std::min(DT, rp.ndm - d0);
            int64_t vb = 0, rb = 0;
            for (int32_t c = 0; c < p.nchan;) {
                PendingGroup g;
                if (!make_group(p, rp, d0, nt, c, G, es, g)) return SPT_ERR_UNSUPPORTED;
                vb += (int64_t)g.vwords * 4; rb += g.raw_bytes;
                c += g.nch;
            }
            int64_t v = (int64_t)((double)kSmemDataBytes * (double)vb / (double)(vb + rb));
            v = std::min<int64_t>(std::max<int64_t>(v, kSmemDataBytes / 4), (int64_t)kSmemDataBytes * 7 / 8);
            v = std::min<int64_t>(v, 65535 * 4);
            rp.vcap_words = (int32_t)(v / 16 * 4);
        }
        const int64_t rcap_bytes = std::min<int64_t>(kSmemDataBytes - (int64_t)rp.vcap_words * 4, 1 << 17);

        for (int32_t d0 = 0; d0 < rp.ndm; d0 += DT) {
            TileDesc td;
            td.trial0 = d0;
            td.ntrial = std::min(DT, rp.ndm - d0);
            td.stage0 = (int32_t)rp.sidx.size();
            std::vector<PendingGroup> open;
            int64_t open_v = 0, open_r = 0, open_pairs = 0;
            int since_flush = 0;
            auto blob_words_of = [&](size_t ngrp, int64_t npairs) {
                return (int64_t)kBlobHdrWords + 4 * (int64_t)ngrp + npairs + (int64_t)ngrp * DT / 2;
            };
            auto close_stage = [&](bool flush) {
                if (open.empty()) {
                    if (flush && (int32_t)rp.sidx.size() > td.stage0) {
                        rp.blob[rp.sidx.back().blob_word0 + 1] = 1;
                        since_flush = 0;
                    }
                    return;
                }
                StageIndex si;
                si.blob_word0 = (uint32_t)rp.blob.size();
                si.row0 = (uint32_t)rp.rows.size();
                const size_t ngrp = open.size();
                std::vector<uint32_t> hdr(kBlobHdrWords + 4 * ngrp), pairs;
                std::vector<uint16_t> toff;
                int32_t vbase = 0, rbase = 0;
                for (size_t k = 0; k < ngrp; ++k) {
                    PendingGroup& g = open[k];
                    const uint32_t pair0 = (uint32_t)pairs.size();
                    for (int j = 0; j < g.nch; ++j) {
                        RowDesc r = g.rows[j];
                        r.soff += rbase;
                        rp.rows.push_back(r);
                        // shifts of this channel, most used first (= base pair)
                        std::vector<std::pair<int, int>> cnt;  // (shift, variants using it)
                        for (auto& v : g.vars) {
                            auto it = std::find_if(cnt.begin(), cnt.end(), [&](auto& x) { return x.first == v[j]; });
                            if (it == cnt.end()) cnt.push_back({v[j], 1}); else it->second++;
                        }
                        std::stable_sort(cnt.begin(), cnt.end(), [](auto& a, auto& b) { return a.second > b.second; });
                        for (size_t q = 0; q < cnt.size(); ++q) {
                            const int s = cnt[q].first;
                            const uint32_t off = (uint32_t)(r.soff + (g.dmin + s - r.astart) * es);
                            uint32_t mask = 0;
                            if (q > 0)
                                for (int v = 0; v < g.nvar; ++v) if (g.vars[v][j] == s) mask |= 1u << v;
                            pairs.push_back(off | (q == 0 ? kPairBaseBit : 0u) | (mask << 20));
                        }
                    }
                    hdr[kBlobHdrWords + 4 * k + 0] = (uint32_t)vbase;
                    hdr[kBlobHdrWords + 4 * k + 1] = (uint32_t)g.vlen;
                    hdr[kBlobHdrWords + 4 * k + 2] = pair0 | ((uint32_t)(pairs.size() - pair0) << 16);
                    hdr[kBlobHdrWords + 4 * k + 3] = (uint32_t)g.nvar;
                    for (int i = 0; i < DT; ++i) {
                        const int ii = std::min(i, td.ntrial - 1);  // unused trial slots alias the last valid trial
                        toff.push_back((uint16_t)(vbase + g.var_of[ii] * g.vlen + g.b[ii]));
                    }
                    vbase += g.vwords;
                    rbase += g.raw_bytes;
                    rp.ngroups++; rp.nvariants += g.nvar;
                }
                rp.npairs += (int64_t)pairs.size();
                hdr[0] = (uint32_t)ngrp; hdr[1] = flush ? 1u : 0u; hdr[2] = (uint32_t)pairs.size(); hdr[3] = 0;
                rp.blob.insert(rp.blob.end(), hdr.begin(), hdr.end());
                rp.blob.insert(rp.blob.end(), pairs.begin(), pairs.end());
                for (size_t i = 0; i < toff.size(); i += 2)
                    rp.blob.push_back((uint32_t)toff[i] | ((uint32_t)(i + 1 < toff.size() ? toff[i + 1] : 0) << 16));
                while ((rp.blob.size() - si.blob_word0) % 4) rp.blob.push_back(0);
                si.blob_words = (uint32_t)(rp.blob.size() - si.blob_word0);
                si.nrows = (uint32_t)(rp.rows.size() - si.row0);
                rp.sidx.push_back(si);
                if (flush) since_flush = 0;
                open.clear();
                open_v = open_r = open_pairs = 0;
            };
            for (int32_t c = 0; c < p.nchan;) {
                PendingGroup g;
                if (!make_group(p, rp, d0, td.ntrial, c, G, es, g)) return SPT_ERR_UNSUPPORTED;
                c += g.nch;
                if (g.vwords > rp.vcap_words || g.raw_bytes > rcap_bytes ||
                    blob_words_of(1, g.npairs) * 4 > kBlobBytes)
                    return SPT_ERR_UNSUPPORTED;  // one group must fit a stage
                if (since_flush + g.nch > lane_channels) close_stage(true);
                else if (open_v + g.vwords > rp.vcap_words || open_r + g.raw_bytes > rcap_bytes ||
                         (int)open.size() >= kMaxStageGroups ||
                         blob_words_of(open.size() + 1, open_pairs + g.npairs) * 4 > kBlobBytes)
                    close_stage(false);
                open_v += g.vwords; open_r += g.raw_bytes; open_pairs += g.npairs;
                since_flush += g.nch;
                open.push_back(std::move(g));
            }
            close_stage(true);
            td.nstage = (int32_t)rp.sidx.size() - td.stage0;
            rp.tiles.push_back(td);
        }
    }
    p.tiling_built = true;
    return SPT_OK;
}

}  // namespace spt
