/*
 * synth.c -- seeded synthetic uGMRT-shaped filterbanks (input generator only).
 *
 * This file is the ONE piece of code that serves both the CUDA path and the
 * oracle: it makes the bytes they are both fed.  It holds none of the search
 * arithmetic (no delay table, no dedispersion, no boxcar, no S/N).  The only
 * physics in here is what a *signal* needs: a dispersed burst sweeps across the
 * band following the cold-plasma law (Eq. 1-2), so the
 * generator places the burst in channel c at the sample nearest to
 * t0 + Dconst*DM*(f_c^-2 - f_top^-2)/tsamp.
 *
 * Data shape follows the paper: 8-bit samples, channel 0 = highest frequency,
 * 1.31072 ms sampling.  Layout: [chan][time], time
 * contiguous (BASELINE.json north_star: "nchan x nsamp per beam").
 *
 * Noise is counter based: sample (seed, beam, chan, t) does not depend on the
 * thread count or on the order of generation.
 *     key  = mix64(mix64(seed) ^ mix64(beam * 0x9E3779B97F4A7C15 + chan))
 *     pair p = t >> 1 :  h1 = mix64(key + p * 0xD1B54A32D192ED03), h2 = mix64(h1 ^ 0x8CB92BA72F3D8DD7)
 *     u1 = ((h1 >> 11) + 1) * 2^-53  in (0,1],  u2 = (h2 >> 11) * 2^-53 in [0,1)
 *     r = sqrt(-2 ln u1);  g(2p) = r cos(2 pi u2);  g(2p+1) = r sin(2 pi u2)      (Box-Muller)
 * Signal terms are added in double BEFORE quantisation:
 *     x = clip(floor(mean + std*g + signal + 0.5), 0, 255)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SYNTH_DCONST 4.148808e3 /* s MHz^2 pc^-1 cm^3 -- BASELINE.json north_star (2) */

typedef struct {
    double dm;      /* pc cm^-3 */
    double amp;     /* counts added per channel per sample while the burst is on */
    int64_t t0;     /* start sample in the top channel */
    int32_t width;  /* samples */
    int32_t pad_;
} synth_burst;

typedef struct {
    double offset;  /* constant counts added to the channel */
    double amp;     /* sinusoid amplitude (counts) */
    double period;  /* samples */
    double phase;   /* radians */
    int32_t chan;
    int32_t pad_;
} synth_tone;

typedef struct {
    double amp;     /* counts added to ALL channels (zero-DM broadband spike) */
    int64_t t0;
    int32_t dur;
    int32_t pad_;
} synth_spike;

static inline uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

static void noise_row(double* g, int64_t nsamp, uint64_t key) {
    const double two53 = 1.0 / 9007199254740992.0;
    const double twopi = 6.283185307179586476925286766559;
    int64_t npair = (nsamp + 1) >> 1;
    for (int64_t p = 0; p < npair; ++p) {
        uint64_t h1 = mix64(key + (uint64_t)p * 0xD1B54A32D192ED03ULL);
        uint64_t h2 = mix64(h1 ^ 0x8CB92BA72F3D8DD7ULL);
        double u1 = (double)((h1 >> 11) + 1) * two53;
        double u2 = (double)(h2 >> 11) * two53;
        double r = sqrt(-2.0 * log(u1));
        double a = twopi * u2;
        g[2 * p] = r * cos(a);
        if (2 * p + 1 < nsamp) g[2 * p + 1] = r * sin(a);
    }
}

/* Sample offset of a burst of dispersion measure dm in channel frequency f (MHz). */
static inline int64_t sweep_samples(double dm, double f, double ftop, double tsamp) {
    double dt = SYNTH_DCONST * dm * (1.0 / (f * f) - 1.0 / (ftop * ftop)); /* seconds */
    return (int64_t)floor(dt / tsamp + 0.5);
}

int synth_sweep_samples(double dm, double fch1, double foff, int32_t chan, double tsamp, int64_t* out) {
    if (!out) return -1;
    *out = sweep_samples(dm, fch1 + (double)chan * foff, fch1, tsamp);
    return 0;
}

/*
 * Fill out[nchan][nsamp] (uint8) for one beam.  Returns 0, or -1 on bad arguments / out of memory.
 */
int synth_filterbank(uint8_t* out, int32_t nchan, int64_t nsamp, double fch1, double foff, double tsamp,
                     double mean, double std, uint64_t seed, uint64_t beam,
                     const synth_burst* bursts, int32_t nbursts,
                     const synth_tone* tones, int32_t ntones,
                     const synth_spike* spikes, int32_t nspikes, int32_t nthreads) {
    if (!out || nchan <= 0 || nsamp <= 0 || nbursts < 0 || ntones < 0 || nspikes < 0) return -1;
    int failed = 0;
    /* the zero-DM spikes hit every channel at the same samples: build their time profile once */
    double* spike_profile = NULL;
    if (nspikes > 0) {
        spike_profile = (double*)calloc((size_t)nsamp, sizeof(double));
        if (!spike_profile) return -1;
        for (int32_t s = 0; s < nspikes; ++s)
            for (int64_t t = spikes[s].t0; t < spikes[s].t0 + spikes[s].dur; ++t)
                if (t >= 0 && t < nsamp) spike_profile[t] += spikes[s].amp;
    }
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#pragma omp parallel num_threads(nthreads)
#endif
    {
        double* v = (double*)malloc((size_t)nsamp * sizeof(double));
        if (!v) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
            failed = 1;
        }
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 4)
#endif
        for (int32_t c = 0; c < nchan; ++c) {
            if (!v) continue;
            uint64_t key = mix64(mix64(seed) ^ mix64(beam * 0x9E3779B97F4A7C15ULL + (uint64_t)c));
            noise_row(v, nsamp, key);
            for (int64_t t = 0; t < nsamp; ++t) v[t] = mean + std * v[t];
            double f = fch1 + (double)c * foff;
            for (int32_t b = 0; b < nbursts; ++b) {
                int64_t ts = bursts[b].t0 + sweep_samples(bursts[b].dm, f, fch1, tsamp);
                for (int64_t t = ts; t < ts + bursts[b].width; ++t)
                    if (t >= 0 && t < nsamp) v[t] += bursts[b].amp;
            }
            for (int32_t k = 0; k < ntones; ++k) {
                if (tones[k].chan != c) continue;
                const double twopi = 6.283185307179586476925286766559;
                for (int64_t t = 0; t < nsamp; ++t)
                    v[t] += tones[k].offset + tones[k].amp * sin(twopi * (double)t / tones[k].period + tones[k].phase);
            }
            if (spike_profile)
                for (int64_t t = 0; t < nsamp; ++t) v[t] += spike_profile[t];
            uint8_t* row = out + (size_t)c * (size_t)nsamp;
            for (int64_t t = 0; t < nsamp; ++t) {
                double q = floor(v[t] + 0.5);
                row[t] = (uint8_t)(q < 0.0 ? 0.0 : (q > 255.0 ? 255.0 : q));
            }
        }
        free(v);
    }
    free(spike_profile);
    return failed ? -1 : 0;
}

/* Order-sensitive 64-bit checksum of a buffer (recorded with every generated input). */
uint64_t synth_checksum(const uint8_t* buf, int64_t n) {
    uint64_t h = 0xCBF29CE484222325ULL;
    int64_t i = 0;
    for (; i + 8 <= n; i += 8) {
        uint64_t w;
        memcpy(&w, buf + i, 8);
        h = mix64(h ^ w);
    }
    for (; i < n; ++i) h = mix64(h ^ buf[i]);
    return h;
}
