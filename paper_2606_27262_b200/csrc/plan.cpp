// plan.cpp -- host side of libspt: trial list, delay table, output geometry (a1 of SURVEY.md 8(a)) and the
// factorisation of the delay table that the tiled dedispersion kernel runs on.
//
// Delay law: PAPER.md:51-58 (Eq. 1-2), reference = highest frequency; constant and rounding per
// BASELINE.json north_star (2); readings A1-A4, B3 of DESIGN.md.  Compiled with FP contraction off.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>

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
// -------------------------------------------------------------------------------------------------------------
int build_tiling(Plan& p) {
    const int G = p.opt_group, DT = p.opt_dm_tile;
    for (RangePlan& rp : p.ranges) {
        rp.tiles.clear(); rp.stages.clear(); rp.groups.clear(); rp.var_shift.clear(); rp.trial_off.clear();
        rp.ntile_t = (int32_t)((rp.max_nout + kTT - 1) / kTT);
        // 16-bit lanes hold sums of at most floor(65535 / (255*decim)) channel samples
        const int lane_channels = 65535 / (255 * rp.decim);
        if (lane_channels < 1) return SPT_ERR_UNSUPPORTED;
        for (int32_t d0 = 0; d0 < rp.ndm; d0 += DT) {
            TileDesc td;
            td.trial0 = d0;
            td.ntrial = std::min(DT, rp.ndm - d0);
            td.stage0 = (int32_t)rp.stages.size();
            StageDesc st{}; st.grp0 = (int32_t)rp.groups.size();
            int64_t st_words = 0;      // variant + expansion words of the open stage
            int32_t st_vwords = 0;     // variant words of the open stage
            int since_flush = 0;       // channels accumulated in the packed lanes since the last flush
            auto close_stage = [&](bool flush) {
                if (st.ngrp == 0) {
                    if (flush && (int32_t)rp.stages.size() > td.stage0) { rp.stages.back().flush = 1; since_flush = 0; }
                    return;
                }
                st.flush = flush ? 1 : 0;
                rp.stages.push_back(st);
                if (flush) since_flush = 0;
                st = StageDesc{}; st.grp0 = (int32_t)rp.groups.size();
                st_words = 0;
                st_vwords = 0;
            };
            for (int32_t c_next = 0; c_next < p.nchan;) {
                GroupDesc gd{};
                gd.chan0 = c_next;
                int32_t dmin = INT32_MAX, dmax = 0;
                for (int i = 0; i < td.ntrial; ++i) {
                    const int32_t v = rp.delay[(size_t)(d0 + i) * p.nchan + gd.chan0];
                    dmin = std::min(dmin, v); dmax = std::max(dmax, v);
                }
                gd.wlo = dmin & ~3;
                const int a0 = dmin - gd.wlo;
                gd.vlen = kH + (dmax - dmin);
                // distinct relative-delay vectors of the tile's trials; the group is halved until they are few
                // (widely spaced channels at high DM have a different vector for every trial: no reuse to exploit)
                std::vector<std::vector<int16_t>> vars;
                std::vector<int> var_of(td.ntrial);
                int maxshift = 0;
                for (int gsize = std::min(G, p.nchan - c_next);; gsize >>= 1) {
                    std::map<std::vector<int16_t>, int> seen;
                    vars.clear();
                    maxshift = 0;
                    gd.nch = gsize;
                    for (int i = 0; i < td.ntrial; ++i) {
                        const int32_t* row = &rp.delay[(size_t)(d0 + i) * p.nchan + gd.chan0];
                        std::vector<int16_t> rho(kMaxG, 0);
                        for (int j = 0; j < gd.nch; ++j) {
                            const int s = a0 + (row[j] - row[0]);
                            if (s > 32000) return SPT_ERR_UNSUPPORTED;
                            rho[j] = (int16_t)s;
                            maxshift = std::max(maxshift, s);
                        }
                        auto it = seen.find(rho);
                        if (it == seen.end()) {
                            it = seen.emplace(rho, (int)vars.size()).first;
                            vars.push_back(rho);
                        }
                        var_of[i] = it->second;
                    }
                    if (gsize == 1 || (int)vars.size() <= 2 * gsize + 2) break;
                }
                c_next += gd.nch;
                gd.nvar = (int32_t)vars.size();
                gd.elen = (int32_t)round_up(gd.vlen + maxshift, 4);
                const int64_t vneed = (int64_t)gd.nvar * gd.vlen;
                const int64_t need = vneed + (int64_t)gd.nch * gd.elen;
                if (need + 4 > kStageDataWords) return SPT_ERR_UNSUPPORTED;  // one group must fit a stage
                if (since_flush + gd.nch > lane_channels) close_stage(true);
                else if (st_words + need + 4 > kStageDataWords || st.ngrp >= kMaxStageGroups ||
                         st_vwords + vneed > 65535) close_stage(false);
                gd.var0 = (int32_t)(rp.var_shift.size() / kMaxG);
                for (auto& v : vars) rp.var_shift.insert(rp.var_shift.end(), v.begin(), v.end());
                gd.vbase = st_vwords;
                gd.ebase = st.ewords;
                for (int i = 0; i < DT; ++i) {
                    const int ii = std::min(i, td.ntrial - 1);  // unused trial slots alias the last valid trial
                    const int32_t b = rp.delay[(size_t)(d0 + ii) * p.nchan + gd.chan0] - dmin;
                    rp.trial_off.push_back((uint16_t)(gd.vbase + var_of[ii] * gd.vlen + b));
                }
                rp.groups.push_back(gd);
                st.ngrp += 1;
                st.ewords += gd.nch * gd.elen;
                st.nvar += gd.nvar;
                st_words += need;
                st_vwords += (int32_t)vneed;
                st.vwords = st_vwords;
                since_flush += gd.nch;
            }
            close_stage(true);
            td.nstage = (int32_t)rp.stages.size() - td.stage0;
            rp.tiles.push_back(td);
        }
    }
    p.tiling_built = true;
    return SPT_OK;
}

}  // namespace spt
