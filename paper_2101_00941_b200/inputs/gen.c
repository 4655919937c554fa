/*
 * Seeded synthetic filterbank generator (input side only).
 *
 * This file belongs to the INPUT GENERATOR module.  It holds none of the
 * method's arithmetic (no dedispersion, no statistics, no boxcars): it only
 * turns (seed, sample index) into an 8-bit noise sample.  Both the CUDA path
 * and the CPU oracle are fed from buffers written here; neither links it.
 *
 * Noise model: the value at flat
 * index i = t*nchans + c is
 *     x_i = Q_m( u_i ),   u_i = top 32 bits of mix64(seed, i)
 * where Q_m is the quantile function of clip(rint(m + 16 z), 0, 255), z~N(0,1),
 * given as a table cdf[255] of 32-bit thresholds computed by the Python side in
 * double precision: x = #{ v in 0..254 : u >= cdf[v] }.  Everything here is
 * integer arithmetic, so every compiler / thread count gives the same bytes.
 */
#include <stdint.h>
#include <stddef.h>

static inline uint64_t mix64(uint64_t seed, uint64_t i)
{
    /* counter-based: SplitMix64 finaliser applied to seed*phi + i */
    uint64_t z = seed * 0x9E3779B97F4A7C15ull + i;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static inline uint8_t quantile(const uint32_t *cdf, uint32_t u)
{
    /* binary search: number of thresholds <= u, thresholds non-decreasing */
    int lo = 0, hi = 255;               /* answer in [0,255] */
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (u >= cdf[mid]) lo = mid + 1; else hi = mid;
    }
    return (uint8_t)lo;
}

/* 32-bit uniform for flat index i (exported so Python can patch pulses). */
uint32_t aain_uniform32(uint64_t seed, uint64_t i)
{
    return (uint32_t)(mix64(seed, i) >> 32);
}

/*
 * Fill out[0..n) with noise samples for flat indices first..first+n.
 * lut16[65536]: for the top 16 bits of u, the sample value if the whole bucket
 * maps to one value, else 0xFFFF (then the binary search decides).
 */
void aain_fill_noise(uint8_t *out, uint64_t first, uint64_t n, uint64_t seed,
                     const uint32_t *cdf, const uint16_t *lut16)
{
    #pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k) {
        uint32_t u = (uint32_t)(mix64(seed, first + (uint64_t)k) >> 32);
        uint16_t q = lut16[u >> 16];
        out[k] = (q != 0xFFFFu) ? (uint8_t)q : quantile(cdf, u);
    }
}

/* One sample through a given table (used for the few pulse-carrying samples). */
uint8_t aain_sample(uint64_t seed, uint64_t i, const uint32_t *cdf)
{
    return quantile(cdf, (uint32_t)(mix64(seed, i) >> 32));
}

/*
 * Re-draw samples t in [t_first, t_first+w) of channel c through table cdf
 * (a table for a shifted mean): out[t*nchans + c].  Used for pulse injection.
 */
void aain_patch(uint8_t *buf, uint64_t nchans, uint64_t nsamp, uint64_t c,
                int64_t t_first, int64_t w, uint64_t seed, const uint32_t *cdf)
{
    for (int64_t t = t_first; t < t_first + w; ++t) {
        if (t < 0 || (uint64_t)t >= nsamp) continue;
        uint64_t i = (uint64_t)t * nchans + c;
        buf[i] = quantile(cdf, (uint32_t)(mix64(seed, i) >> 32));
    }
}
