/*
 * oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct CPU statement of what the SPOTLIGHT search hot path computes
 * (arxiv/paper_2606_27262), written from the paper so that a reader can check it by eye.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call anything in oracle/.  It shares no code, header, table or constant with the
 * CUDA path (paper_2606_27262_b200/csrc) and neither includes the other.
 *
 * Where the paper is silent the readings of SURVEY.md section 8(c) are taken; every one is listed in
 * DESIGN.md ("Readings").  Parity status: every function below is pinned by tests/test_oracle_*.py
 * (closed forms in exact rational arithmetic, invariants, brute force on tiny inputs, the worked
 * sqrt(N - w) boxcar example, injected-burst recovery); none is "parity unpinned".  The S/N
 * normalisation, the best-width rule and the candidate rule are READINGS (the paper gives only the
 * principle) -- pinned for self-consistency, not against the authors' implementation.
 *
 * Integer results are exact by definition (any order of the same integer sums is the same number);
 * floating point is IEEE double throughout, compiled with -ffp-contract=off.
 *
 * OpenMP, where used, only distributes INDEPENDENT trials over threads; no sum is blocked, fused or
 * reordered.
 */
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <map>
#include <tuple>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

/* Dispersion constant.  The paper prints D = 4.1488064239(11)e3 MHz^2 pc^-1 cm^3 s;
 * BASELINE.json north_star (2) fixes 4.148808e3 for this build and binds (reading A2). */
const double kDispersionConstant = 4.148808e3;

}  // namespace

extern "C" {

/* Threads the batch entry points will use (for the "cores" figure of the reported CPU baseline). */
int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------------
 * A. Plan and delay table -- PAPER.md:51-58 (Eq. 1-2), 76-78 (plan = sub-ranges with their own step).
 *
 *   f_c   = fch1 + c*foff            (c = 0 is the highest frequency and the reference)
 *   DM_i  = dm_lo + i*dm_step        (multiply, do not accumulate)
 *   x     = (D * DM_i * (1/f_c^2 - 1/f_top^2)) / (tsamp * k)       [samples of the k-decimated rate]
 *   delay = floor(x + 0.5)           (round half up; the paper says only "the appropriate time delay",
 *                                     PAPER.md:80; north_star: "rounded to integer samples")
 * ---------------------------------------------------------------------------------------------- */
int orc_delay_table(double fch1, double foff, int32_t nchan, double tsamp, double dm_lo, double dm_step,
                    int32_t ndm, int32_t decim, int32_t* delay /* [ndm][nchan] */) {
    if (!delay || nchan <= 0 || ndm <= 0 || decim <= 0 || !(foff < 0.0) || !(tsamp > 0.0)) return -1;
    const double ftop = fch1;
    for (int32_t i = 0; i < ndm; ++i) {
        const double dm = dm_lo + (double)i * dm_step;
        for (int32_t c = 0; c < nchan; ++c) {
            const double f = fch1 + (double)c * foff;
            const double x = (kDispersionConstant * dm * (1.0 / (f * f) - 1.0 / (ftop * ftop))) / (tsamp * (double)decim);
            delay[(size_t)i * nchan + c] = (int32_t)std::floor(x + 0.5);
        }
    }
    return 0;
}

/* Valid output length of a trial: nout = max(0, floor(nsamp/k) - delay[lowest channel]) (reading B3:
 * only samples for which every channel is inside the data are defined; no wrap, no padding). */
int orc_nout(const int32_t* delay /* [ndm][nchan] */, int32_t ndm, int32_t nchan, int64_t nsamp, int32_t decim,
             int32_t* nout /* [ndm] */) {
    if (!delay || !nout || decim <= 0) return -1;
    const int64_t nk = nsamp / decim;
    for (int32_t i = 0; i < ndm; ++i) {
        int64_t n = nk - (int64_t)delay[(size_t)i * nchan + (nchan - 1)];
        nout[i] = (int32_t)(n > 0 ? n : 0);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * B1. Time decimation by k (not in the paper; BASELINE.json north_star (3), reading B1):
 *   y[c][j] = sum_{m<k} x[c][k*j + m],  j < floor(nsamp/k); the trailing nsamp mod k samples are dropped.
 *   A sum, not a mean: integers stay exact and S/N is scale free.
 * ---------------------------------------------------------------------------------------------- */
int orc_decimate(const uint8_t* x /* [nchan][nsamp] */, int32_t nchan, int64_t nsamp, int32_t k,
                 uint16_t* y /* [nchan][nsamp/k] */) {
    if (!x || !y || nchan <= 0 || nsamp <= 0 || k <= 0 || k > 257) return -1;
    const int64_t nk = nsamp / k;
    for (int32_t c = 0; c < nchan; ++c)
        for (int64_t j = 0; j < nk; ++j) {
            uint32_t s = 0;
            for (int32_t m = 0; m < k; ++m) s += x[(size_t)c * nsamp + (size_t)(k * j + m)];
            y[(size_t)c * nk + j] = (uint16_t)s;
        }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * B2. Brute-force incoherent dedispersion -- PAPER.md:80 ("shifting each channel ... by the appropriate
 * time delay"), PAPER.md:90 (output = DM transform, one row per trial):
 *   out[d][t] = sum_c y[c][t + delay[d][c]],   t in [0, nout[d])
 * Lower frequencies arrive later, so the read is forward in time.  Rows are written back to back:
 * row d starts at rowoff[d] (caller supplied; rowoff[d+1] - rowoff[d] >= nout[d]).
 * ---------------------------------------------------------------------------------------------- */
int orc_dedisperse_u16(const uint16_t* y /* [nchan][nk] */, int32_t nchan, int64_t nk,
                       const int32_t* delay /* [ndm][nchan] */, int32_t ndm, const int32_t* nout,
                       const int64_t* rowoff, int32_t* out) {
    if (!y || !delay || !nout || !rowoff || !out) return -1;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int32_t d = 0; d < ndm; ++d) {
        int32_t* row = out + rowoff[d];
        const int64_t n = nout[d];
        for (int64_t t = 0; t < n; ++t) row[t] = 0;
        for (int32_t c = 0; c < nchan; ++c) {
            const uint16_t* src = y + (size_t)c * nk + delay[(size_t)d * nchan + c];
            for (int64_t t = 0; t < n; ++t) row[t] += (int32_t)src[t];
        }
    }
    return 0;
}

int orc_dedisperse_u8(const uint8_t* x /* [nchan][nsamp] */, int32_t nchan, int64_t nsamp,
                      const int32_t* delay /* [ndm][nchan] */, int32_t ndm, const int32_t* nout,
                      const int64_t* rowoff, int32_t* out) {
    if (!x || !delay || !nout || !rowoff || !out) return -1;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int32_t d = 0; d < ndm; ++d) {
        int32_t* row = out + rowoff[d];
        const int64_t n = nout[d];
        for (int64_t t = 0; t < n; ++t) row[t] = 0;
        for (int32_t c = 0; c < nchan; ++c) {
            const uint8_t* src = x + (size_t)c * nsamp + delay[(size_t)d * nchan + c];
            for (int64_t t = 0; t < n; ++t) row[t] += (int32_t)src[t];
        }
    }
    return 0;
}

/* One output sample, straight from the definition (for sampled parity at full size). */
int orc_dedisperse_point_u8(const uint8_t* x, int32_t nchan, int64_t nsamp, const int32_t* delay_row /* [nchan] */,
                            int32_t k, int64_t t, int32_t* out) {
    if (!x || !delay_row || !out || k <= 0) return -1;
    int64_t acc = 0;
    for (int32_t c = 0; c < nchan; ++c) {
        const int64_t j = t + delay_row[c];                      /* decimated sample index */
        for (int32_t m = 0; m < k; ++m) {
            const int64_t s = (int64_t)k * j + m;
            if (s < 0 || s >= nsamp) return -2;
            acc += x[(size_t)c * nsamp + s];
        }
    }
    *out = (int32_t)acc;
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * C1. Per-trial statistics (reading C1): exact integer sums over the whole valid series,
 *   mu = Sx/N,  sigma^2 = (N*Sxx - Sx^2)/N^2  (population variance, no clipping).
 * ---------------------------------------------------------------------------------------------- */
int orc_stats(const int32_t* x, int64_t n, int64_t* sum, uint64_t* sumsq) {
    if (!x || !sum || !sumsq || n < 0) return -1;
    int64_t s = 0;
    uint64_t q = 0;
    for (int64_t t = 0; t < n; ++t) {
        s += x[t];
        q += (uint64_t)((int64_t)x[t] * (int64_t)x[t]);
    }
    *sum = s;
    *sumsq = q;
    return 0;
}

int orc_mean_sigma(int64_t n, int64_t sum, uint64_t sumsq, double* mu, double* sigma) {
    if (!mu || !sigma) return -1;
    if (n <= 0) { *mu = 0.0; *sigma = 0.0; return 0; }
    const unsigned __int128 a = (unsigned __int128)(uint64_t)n * (unsigned __int128)sumsq;
    const __int128 s = (__int128)sum;
    const unsigned __int128 b = (unsigned __int128)(s * s);
    const unsigned __int128 num = a >= b ? a - b : 0;     /* N*Sxx - Sx^2 >= 0 (Cauchy-Schwarz) */
    *mu = (double)sum / (double)n;
    *sigma = std::sqrt((double)num / ((double)n * (double)n));
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * C3-C4. Boxcar filter and S/N -- PAPER.md:94: "the convolution of any signal with a boxcar is the
 * cumulative sum of the input signal across the boxcar width", several trial widths.
 *   S_w[t]   = sum_{j<w} x[t+j],  t in [0, N-w]                      (start aligned)
 *   snr_w[t] = (S_w[t] - w*mu) / (sigma*sqrt(w)) = (N*S_w[t] - w*Sx) / (N*sigma*sqrt(w))
 * The numerator is formed in exact integers (reading C4).  sigma == 0 or N < 2 -> S/N == 0.
 * ---------------------------------------------------------------------------------------------- */
int orc_boxcar_snr(const int32_t* x, int64_t n, int32_t w, double* snr /* [n-w+1] */) {
    if (!x || !snr || w < 1) return -1;
    if (w > n) return 0;
    int64_t sum; uint64_t sumsq; double mu, sigma;
    orc_stats(x, n, &sum, &sumsq);
    orc_mean_sigma(n, sum, sumsq, &mu, &sigma);
    for (int64_t t = 0; t + w <= n; ++t) {
        int64_t S = 0;
        for (int32_t j = 0; j < w; ++j) S += x[t + j];
        if (sigma > 0.0 && n >= 2) {
            const int64_t num = n * S - (int64_t)w * sum;
            snr[t] = (double)num / ((double)n * sigma * std::sqrt((double)w));
        } else {
            snr[t] = 0.0;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * C5 + D1. Best width per sample and candidates (readings C5, D1):
 *   best[t] = max over the valid widths (w <= N - t), scanned in increasing w with strict '>'
 *             (exact tie -> the smaller width);  defined for t in [0, N - wmin].
 *   candidate at every t with best[t] >= threshold (inclusive); no peak filtering here (that is the
 *   separate, optional stage of PAPER.md:96).
 * The boxcar sums come from the exact int64 cumulative sum C[t] = sum_{u<t} x[u]: S_w[t] = C[t+w] - C[t]
 * (PAPER.md:94's "cumulative sum"; same integers as the literal loop in orc_boxcar_snr, which a test checks).
 * widths must be strictly increasing and >= 1.
 * Outputs (any may be NULL): best_snr/best_w of length max(0, N - wmin + 1).
 * ---------------------------------------------------------------------------------------------- */
int orc_best_width(const int32_t* x, int64_t n, const int32_t* widths, int32_t nw,
                   double* best_snr, int32_t* best_w) {
    if (!x || !widths || nw < 1) return -1;
    for (int32_t i = 0; i < nw; ++i)
        if (widths[i] < 1 || (i > 0 && widths[i] <= widths[i - 1])) return -1;
    const int64_t nbest = n - widths[0] + 1;
    if (nbest <= 0) return 0;
    int64_t sum; uint64_t sumsq; double mu, sigma;
    orc_stats(x, n, &sum, &sumsq);
    orc_mean_sigma(n, sum, sumsq, &mu, &sigma);
    std::vector<int64_t> C((size_t)n + 1);
    C[0] = 0;
    for (int64_t t = 0; t < n; ++t) C[t + 1] = C[t] + x[t];
    const bool live = sigma > 0.0 && n >= 2;
    for (int64_t t = 0; t < nbest; ++t) {
        double b = 0.0;
        int32_t bw = widths[0];
        bool first = true;
        for (int32_t i = 0; i < nw; ++i) {
            const int32_t w = widths[i];
            if (t + w > n) break;
            double s = 0.0;
            if (live) {
                const int64_t S = C[t + w] - C[t];
                const int64_t num = n * S - (int64_t)w * sum;
                s = (double)num / ((double)n * sigma * std::sqrt((double)w));
            }
            if (first || s > b) { b = s; bw = w; first = false; }
        }
        if (best_snr) best_snr[t] = b;
        if (best_w) best_w[t] = bw;
    }
    return 0;
}

/* S/N of one given width at one sample (for the near-tie rule of the candidate comparison). */
int orc_snr_at(const int32_t* x, int64_t n, int32_t w, int64_t t, double* snr) {
    if (!x || !snr || w < 1 || t < 0 || t + w > n) return -1;
    int64_t sum; uint64_t sumsq; double mu, sigma;
    orc_stats(x, n, &sum, &sumsq);
    orc_mean_sigma(n, sum, sumsq, &mu, &sigma);
    int64_t S = 0;
    for (int32_t j = 0; j < w; ++j) S += x[t + j];
    if (sigma > 0.0 && n >= 2) {
        const int64_t num = n * S - (int64_t)w * sum;
        *snr = (double)num / ((double)n * sigma * std::sqrt((double)w));
    } else {
        *snr = 0.0;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Whole-plane single-pulse search over a DM transform with ragged rows (independent trials in
 * parallel).  Per trial: stats, best[], candidates (best >= threshold).
 * Pass 1 (cand_* == NULL): counts only.  cand arrays must hold rowcount-prefix layout:
 *   candidates of trial d go to [candoff[d], candoff[d] + count[d]) in increasing t.
 * ---------------------------------------------------------------------------------------------- */
int orc_search_plane(const int32_t* dmt, int32_t ntrial, const int64_t* rowoff, const int32_t* nout,
                     const int32_t* widths, int32_t nw, double threshold,
                     int64_t* sum /* [ntrial] */, uint64_t* sumsq /* [ntrial] */, int64_t* count /* [ntrial] */,
                     const int64_t* candoff, int32_t* cand_t, int32_t* cand_w, double* cand_snr) {
    if (!dmt || !rowoff || !nout || !widths || !count) return -1;
    int bad = 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int32_t d = 0; d < ntrial; ++d) {
        const int64_t n = nout[d];
        const int32_t* x = dmt + rowoff[d];
        int64_t s = 0; uint64_t q = 0;
        orc_stats(x, n, &s, &q);
        if (sum) sum[d] = s;
        if (sumsq) sumsq[d] = q;
        const int64_t nbest = n - widths[0] + 1;
        int64_t cnt = 0;
        if (nbest > 0) {
            std::vector<double> b((size_t)nbest);
            std::vector<int32_t> bw((size_t)nbest);
            if (orc_best_width(x, n, widths, nw, b.data(), bw.data()) != 0) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
                bad = 1;
            }
            for (int64_t t = 0; t < nbest; ++t)
                if (b[t] >= threshold) {
                    if (cand_t && candoff) {
                        const int64_t o = candoff[d] + cnt;
                        cand_t[o] = (int32_t)t;
                        cand_w[o] = bw[t];
                        cand_snr[o] = b[t];
                    }
                    ++cnt;
                }
        }
        count[d] = cnt;
    }
    return bad ? -1 : 0;
}

/* ------------------------------------------------------------------------------------------------
 * E. Peak filtering of the candidate plane -- PAPER.md:96: "Peaks are filtered out by sliding a window across
 * the candidates in the DM-time plane.  From each window, the peak with the highest S/N is picked, and all
 * others are rejected.  Two different stencils are used: a 3x3 window, and an 11x11 window."
 * Reading E: the plane of one beam and one DM range has axes (trial index, sample index of the
 * range's own rate); the window of odd size P is centred on each candidate in turn (it slides by one cell); a
 * candidate is kept iff no OTHER live candidate of the same beam and range inside its window is stronger, where
 * stronger = larger S/N, or equal S/N and smaller (trial, t) in that order -- so exactly one of an exact tie
 * survives.  Stencils are applied one after the other by calling this once per window: `alive` is both input
 * (only live candidates compete) and output.
 * Plain form: for every candidate, every cell of its window is looked up in an ordered map.
 * ---------------------------------------------------------------------------------------------- */
int orc_peak_filter(int64_t n, const int32_t* beam, const int32_t* trial, const int32_t* t, const double* snr,
                    const int32_t* range_of_trial /* [ntrial] */, int32_t ntrial, int32_t window, uint8_t* alive /* [n] in/out */) {
    if (n < 0 || window < 1 || (window & 1) == 0 || !alive || (n > 0 && (!beam || !trial || !t || !snr || !range_of_trial))) return -1;
    const int32_t h = (window - 1) / 2;
    std::map<std::tuple<int32_t, int32_t, int32_t>, int64_t> at;   /* (beam, trial, t) -> index, live candidates only */
    for (int64_t i = 0; i < n; ++i) {
        if (trial[i] < 0 || trial[i] >= ntrial) return -1;
        if (alive[i] && !at.emplace(std::make_tuple(beam[i], trial[i], t[i]), i).second) return -2;   /* duplicate cell */
    }
    std::vector<uint8_t> out((size_t)n, 0);
    for (int64_t i = 0; i < n; ++i) {
        if (!alive[i]) continue;
        bool beaten = false;
        for (int32_t dd = trial[i] - h; dd <= trial[i] + h && !beaten; ++dd) {
            if (dd < 0 || dd >= ntrial || range_of_trial[dd] != range_of_trial[trial[i]]) continue;
            for (int32_t tt = t[i] - h; tt <= t[i] + h; ++tt) {
                if (dd == trial[i] && tt == t[i]) continue;
                auto it = at.find(std::make_tuple(beam[i], dd, tt));
                if (it == at.end()) continue;
                const int64_t j = it->second;
                const bool stronger = snr[j] > snr[i] ||
                                      (snr[j] == snr[i] && (trial[j] < trial[i] || (trial[j] == trial[i] && t[j] < t[i])));
                if (stronger) { beaten = true; break; }
            }
        }
        out[(size_t)i] = beaten ? 0 : 1;
    }
    for (int64_t i = 0; i < n; ++i) alive[i] = out[(size_t)i];
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * H. Candidate cut-outs -- PAPER.md:116 ("candies ... extracts two features from this data: the dedispersed dynamic
 * spectrum, and the DM transform.  The former is created at the candidate's detected DM, while the latter is created at
 * a narrow DM range centred around that DM"), Eq. 4 for the half-width of that range.  Reading H: integers,
 * no normalisation; time bins of tbin raw samples, nt of them, the window starting at raw sample ts (may lie partly
 * outside the data: samples outside contribute 0); nf frequency bands of nchan/nf adjacent channels;
 *   dds[f][j] = sum_{c in band f} sum_{m<tbin} x[c][ts + j*tbin + m + delay(dm0, c)]
 *   dmt[i][j] = sum_c            sum_{m<tbin} x[c][ts + j*tbin + m + delay(DM_i, c)],  DM_i = (dm0 - ddm) + i*step,
 *   step = (2*ddm)/(ndm-1) (ndm > 1), delays at full time resolution as in section A.
 * ---------------------------------------------------------------------------------------------- */
int orc_cutout(const uint8_t* x /* [nchan][nsamp] */, int32_t nchan, int64_t nsamp, double fch1, double foff, double tsamp,
               double dm0, double ddm, int32_t ndm, int64_t ts, int32_t tbin, int32_t nt, int32_t nf,
               int32_t* dds /* [nf][nt] */, int32_t* dmt /* [ndm][nt] */) {
    if (!x || !dds || !dmt || nchan < 1 || ndm < 1 || tbin < 1 || nt < 1 || nf < 1 || nchan % nf != 0) return -1;
    std::vector<int32_t> d0((size_t)nchan), di((size_t)nchan);
    if (orc_delay_table(fch1, foff, nchan, tsamp, dm0, 1.0, 1, 1, d0.data()) != 0) return -1;
    const int32_t per = nchan / nf;
    auto at = [&](int32_t c, int64_t s) -> int32_t { return (s < 0 || s >= nsamp) ? 0 : (int32_t)x[(size_t)c * nsamp + s]; };
    for (int32_t f = 0; f < nf; ++f)
        for (int32_t j = 0; j < nt; ++j) {
            int32_t acc = 0;
            for (int32_t c = f * per; c < (f + 1) * per; ++c)
                for (int32_t m = 0; m < tbin; ++m) acc += at(c, ts + (int64_t)j * tbin + m + d0[c]);
            dds[(size_t)f * nt + j] = acc;
        }
    const double step = ndm > 1 ? (2.0 * ddm) / (double)(ndm - 1) : 0.0;
    for (int32_t i = 0; i < ndm; ++i) {
        if (orc_delay_table(fch1, foff, nchan, tsamp, (dm0 - ddm) + (double)i * step, 1.0, 1, 1, di.data()) != 0) return -1;
        for (int32_t j = 0; j < nt; ++j) {
            int32_t acc = 0;
            for (int32_t c = 0; c < nchan; ++c)
                for (int32_t m = 0; m < tbin; ++m) acc += at(c, ts + (int64_t)j * tbin + m + di[c]);
            dmt[(size_t)i * nt + j] = acc;
        }
    }
    return 0;
}

/* Eq. 4 (clean form at PAPER.md:244): dDM = sqrt(pi)/C * W_s * (S/S(dDM)) * nu_MHz^3 / dnu_MHz with the
 * printed C = 1382.  (The derivation's own first line, from Eq. A3, gives C = 13820: DESIGN.md reading H.) */
double orc_delta_dm(double width_s, double snr_ratio_inverse, double nu_mhz, double bw_mhz, double constant) {
    return std::sqrt(3.14159265358979323846) / constant * width_s * snr_ratio_inverse * (nu_mhz * nu_mhz * nu_mhz) / bw_mhz;
}

}  // extern "C"
