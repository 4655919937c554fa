/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU statement of what the hot path computes:
 * brute-force incoherent dedispersion of 8-bit filterbank data followed by the
 * single-pulse search (boxcar S/N over a width list, robust per-block mean and
 * sigma, threshold, one candidate per (DM, time)).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it.  It shares no code, header, table or helper with the CUDA path
 * (paper_2101_00941_b200/csrc) and knows nothing of chunks, streams or tiles:
 * it works on the whole observation (or on a plain sub-range of output
 * samples) exactly in the order of SURVEY.md §8(c) steps 1-8.
 *
 * What defines each step.  The paper names the two phases --
 * "dedispersion of data and single pulse searching" --
 * but gives no formula; the arithmetic is fixed by BASELINE.json:north_star
 * (delay formula, exact integer sums, S/N tolerances) and by the readings
 * A1-A16 of SURVEY.md §8(c), restated in DESIGN.md "Readings".
 *
 * Parity pins (tests/test_oracle_pins.py): delay closed forms and spot values;
 * DM=0 row == plain channel sum; constant input; single-impulse brute force;
 * python-loop brute force on tiny inputs; statistics vs numpy on un-clipped
 * data and vs a python restatement of the clipping; S/N of an injected boxcar
 * vs its closed form; candidate rule vs python loops.
 * Parity unpinned against the paper (the paper fixes none of them): the choice
 * of estimator (A8), the norm-block length (A9), the candidate definition
 * (A11), the peak rule (A17, aaor_find_peaks), the per-width statistics (A18,
 * aaor_series_stats / aaor_sps_row2), the packing of other bit depths (A19,
 * aaor_bin_u16 and the unpackers of __init__.py) and the grid of long widths
 * (A20, aaor_sps_row2).  They are conventions of this build, pinned only to
 * their own written definition: python-loop brute force, exact fractions,
 * closed forms, hand-made cases (tests/test_oracle_pins.py).
 *
 * Floating point: double everywhere, no FMA contraction (compile with
 * -ffp-contract=off), statistics from exact integer sums so that the only
 * roundings are the ones written below.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- steps 1-2: channel frequencies and integer delays --------------------
 * f_c = f_top + c*foff  (channel centres, A2);  DM_i = dm_low + i*dm_step;
 * delta(c,i) = floor(v + 0.5),
 *   v = ((4.148808e3*DM_i) * (1/(f_c*f_c) - 1/(f_top*f_top))) / (tsamp*bin)
 * (north_star: "delay(c,DM) = round(4.148808e3*DM*(f_c^-2 - f_top^-2)/tsamp) in
 * double"; binned ranges measure the delay in binned samples, A6).
 * out[i*nchans + c]. */
void aaor_delays(int nchans, double f_top, double foff, double tsamp, int bin,
                 double dm_low, double dm_step, int ndms, int64_t *out)
{
    double ts = tsamp * (double)bin;
    for (int i = 0; i < ndms; ++i) {
        double dm = dm_low + (double)i * dm_step;
        for (int c = 0; c < nchans; ++c) {
            double f = f_top + (double)c * foff;
            double g = 1.0 / (f * f) - 1.0 / (f_top * f_top);
            double v = ((4.148808e3 * dm) * g) / ts;
            out[(size_t)i * nchans + c] = (int64_t)floor(v + 0.5);
        }
    }
}

/* ---- step 4: binned, channel-major input ----------------------------------
 * y[c][k] = sum_{i<bin} x[(bin*(tau_first+k) + i)][c],  k = 0..ntau-1,
 * x time-major [nsamp][nchans] (A1), integer sum before delaying (A6).
 * Samples past the end of the observation must not be asked for. */
int aaor_bin(const uint8_t *x, uint64_t nsamp, int nchans, int bin,
             uint64_t tau_first, uint64_t ntau, uint32_t *y)
{
    if ((tau_first + ntau) * (uint64_t)bin > nsamp) return -1;
    #pragma omp parallel for schedule(static)
    for (int c = 0; c < nchans; ++c)
        for (uint64_t k = 0; k < ntau; ++k) {
            uint32_t s = 0;
            for (int i = 0; i < bin; ++i)
                s += x[((tau_first + k) * (uint64_t)bin + (uint64_t)i) * (uint64_t)nchans + (uint64_t)c];
            y[(size_t)c * ntau + k] = s;
        }
    return 0;
}

/* The same for 16-bit samples (x time-major [nsamp][nchans] uint16): inputs of other bit depths (DESIGN.md reading
 * A19: 4-bit samples packed two per byte, low nibble = even channel; 16-bit little-endian words) are widened to
 * uint16 by the caller and binned here.  Sums stay below 2^32 (65535 * bin, bin <= 128). */
int aaor_bin_u16(const uint16_t *x, uint64_t nsamp, int nchans, int bin,
                 uint64_t tau_first, uint64_t ntau, uint32_t *y)
{
    if ((tau_first + ntau) * (uint64_t)bin > nsamp) return -1;
    #pragma omp parallel for schedule(static)
    for (int c = 0; c < nchans; ++c)
        for (uint64_t k = 0; k < ntau; ++k) {
            uint32_t s = 0;
            for (int i = 0; i < bin; ++i)
                s += x[((tau_first + k) * (uint64_t)bin + (uint64_t)i) * (uint64_t)nchans + (uint64_t)c];
            y[(size_t)c * ntau + k] = s;
        }
    return 0;
}

/* ---- step 5: dedispersion ---------------------------------------------------
 * D[i][k] = sum_c y[c][(tau_first + k) + delta(c,i) - y_first],  k = 0..ntau-1,
 * where row c of y holds binned samples y_first .. y_first+ny-1.
 * Exact integer sums (A7: 255*nchans*bin < 2^32 is checked by the caller). */
int aaor_dedisperse(const uint32_t *y, int nchans, uint64_t y_first, uint64_t ny,
                    const int64_t *delays, int ndms,
                    uint64_t tau_first, uint64_t ntau, uint32_t *D)
{
    int bad = 0;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < ndms; ++i) {
        uint32_t *row = D + (size_t)i * ntau;
        memset(row, 0, ntau * sizeof(uint32_t));
        for (int c = 0; c < nchans; ++c) {
            int64_t dl = delays[(size_t)i * nchans + c];
            int64_t first = (int64_t)tau_first + dl - (int64_t)y_first;
            if (first < 0 || (uint64_t)first + ntau > ny) {
                #pragma omp atomic write
                bad = 1;
                continue;
            }
            const uint32_t *src = y + (size_t)c * ny + (size_t)first;
            for (uint64_t k = 0; k < ntau; ++k) row[k] += src[k];
        }
    }
    return bad ? -1 : 0;
}

/* ---- step 6: robust mean and sigma of one norm block ----------------------
 * Plain pass over all n samples, then exactly three passes that keep the
 * samples with |x - mu| <= 3 sigma (latest mu, sigma; chosen among ALL n samples
 * each time) and recompute.  Population sigma, no bias correction (A8).
 * Each (mu, sigma) comes from exact integer sums m = #, S1 = sum x, S2 = sum x^2:
 *     mu = S1/m,   sigma = sqrt( (m*S2 - S1^2) / (m*m) )
 * with m*S2 - S1^2 formed exactly in 128-bit integers and rounded once. */
static void moments(uint64_t m, uint64_t S1, unsigned __int128 S2, double *mu, double *sigma)
{
    unsigned __int128 N = (unsigned __int128)m * S2 - (unsigned __int128)S1 * S1;
    double dm = (double)m;
    *mu = (double)S1 / dm;
    *sigma = sqrt((double)N / (dm * dm));
}

void aaor_block_stats(const uint32_t *d, uint64_t n, double *mu_out, double *sigma_out,
                      uint64_t *nsel_out)
{
    /* the sum of squares is kept in 128 bits: 16-bit input on thousands of channels passes 2^64 (65536 samples of
     * 2^28 each); wherever it stays below 2^64 the value is the same as before */
    uint64_t m = 0, S1 = 0;
    unsigned __int128 S2 = 0;
    double mu = 0.0, sigma = 0.0;
    for (uint64_t k = 0; k < n; ++k) { m++; S1 += d[k]; S2 += (uint64_t)d[k] * d[k]; }
    if (m) moments(m, S1, S2, &mu, &sigma);
    for (int pass = 0; pass < 3 && m; ++pass) {
        double lim = 3.0 * sigma;
        m = 0; S1 = 0; S2 = 0;
        for (uint64_t k = 0; k < n; ++k)
            if (fabs((double)d[k] - mu) <= lim) { m++; S1 += d[k]; S2 += (uint64_t)d[k] * d[k]; }
        if (m) moments(m, S1, S2, &mu, &sigma);
    }
    *mu_out = mu; *sigma_out = sigma; *nsel_out = m;
}

/* ---- step 6 on a series of 64-bit values (the boxcar series of one width, reading A18) -----------------
 * Same estimator as aaor_block_stats: a plain pass and three 3-sigma-clip passes, population sigma, from exact
 * integer sums (128-bit sum of squares, 128-bit numerator rounded once). */
void aaor_series_stats(const uint64_t *v, uint64_t n, double *mu_out, double *sigma_out, uint64_t *nsel_out)
{
    uint64_t m = 0, S1 = 0;
    unsigned __int128 S2 = 0;
    double mu = 0.0, sigma = 0.0;
    for (uint64_t k = 0; k < n; ++k) { m++; S1 += v[k]; S2 += (unsigned __int128)v[k] * v[k]; }
    if (m) moments(m, S1, S2, &mu, &sigma);
    for (int pass = 0; pass < 3 && m; ++pass) {
        double lim = 3.0 * sigma;
        m = 0; S1 = 0; S2 = 0;
        for (uint64_t k = 0; k < n; ++k)
            if (fabs((double)v[k] - mu) <= lim) { m++; S1 += v[k]; S2 += (unsigned __int128)v[k] * v[k]; }
        if (m) moments(m, S1, S2, &mu, &sigma);
    }
    *mu_out = mu; *sigma_out = sigma; *nsel_out = m;
}

/* Reading A20 (decimated long boxcars): widths above wdec are looked at on a coarser time grid, as in a search that
 * halves the time resolution while it doubles the width: dec(w) = the smallest power of two with w / dec(w) <= wdec
 * (1 if wdec <= 0 or w <= wdec); the boxcar of width w is evaluated only at tau with tau mod dec(w) == 0 (tau = the
 * absolute binned sample index).  The sums themselves stay exact. */
static uint64_t width_dec(uint64_t w, int wdec)
{
    uint64_t dec = 1;
    if (wdec > 0)
        while (w > (uint64_t)wdec * dec) dec *= 2;
    return dec;
}

/* ---- steps 6-8 for one dedispersed row --------------------------------------
 * d[0..d_count) holds D[row][d_first .. d_first+d_count).  nout = number of valid
 * output samples of the row's range, L = norm-block length in binned samples.
 * Emits one candidate per tau in [tau_a, tau_b) (tau_a on a block boundary):
 *   for every width w with tau + w <= nout (and tau on the width's grid, A20):  B_w = sum_{i<w} D[tau+i],
 *   sigma_mode 0 (A10): S_w = (B_w - w*mu_k) / (sigma_k*sqrt(w)),  k = block containing tau   (A9)
 *   sigma_mode 1 (A18): S_w = (B_w - mu_{k,w}) / sigma_{k,w}, (mu, sigma)_{k,w} = the robust statistics (A8) of the
 *                boxcar series of width w itself over the block: B_w[t] for the t of block k on the width's grid with
 *                t + w <= nout; a width with sigma_{k,w} = 0 or fewer than 32 such t is skipped
 *   w* = argmax_w S_w (ties -> smallest w);  emit iff S_{w*} >= thr, sigma_k > 0
 *   and the block has n_k >= 32 samples                                    (A11, A13)
 * Returns the number found (may exceed max_out; only max_out are stored) or -1
 * if d does not cover what is needed. */
int64_t aaor_sps_row2(const uint32_t *d, uint64_t d_first, uint64_t d_count,
                      uint64_t nout, uint64_t L,
                      const int32_t *widths, int nwidths, double thr,
                      uint64_t tau_a, uint64_t tau_b, int wdec, int sigma_mode,
                      uint64_t *out_tau, int32_t *out_w, double *out_snr, int64_t max_out)
{
    int64_t found = 0;
    if (tau_b > nout) tau_b = nout;
    if (tau_a % L != 0) return -1;
    double *wmu = (double *)malloc(sizeof(double) * (size_t)(nwidths > 0 ? nwidths : 1));
    double *wsg = (double *)malloc(sizeof(double) * (size_t)(nwidths > 0 ? nwidths : 1));
    uint64_t *series = sigma_mode ? (uint64_t *)malloc(sizeof(uint64_t) * (size_t)L) : NULL;
    for (uint64_t b0 = tau_a; b0 < tau_b; b0 += L) {
        uint64_t b1 = b0 + L < nout ? b0 + L : nout;       /* block [b0, b1) */
        uint64_t n_k = b1 - b0, nsel;
        double mu, sigma;
        if (b0 < d_first || b1 > d_first + d_count) { found = -1; break; }
        aaor_block_stats(d + (b0 - d_first), n_k, &mu, &sigma, &nsel);
        if (!(sigma > 0.0) || n_k < 32) continue;
        if (sigma_mode) {
            int bad = 0;
            for (int j = 0; j < nwidths; ++j) {
                uint64_t w = (uint64_t)widths[j], dec = width_dec(w, wdec), ns = 0, dummy;
                for (uint64_t t = b0; t < b1; ++t) {
                    if (t % dec != 0 || t + w > nout) continue;
                    if (t + w > d_first + d_count) { bad = 1; break; }
                    uint64_t B = 0;
                    for (uint64_t i = 0; i < w; ++i) B += d[t + i - d_first];
                    series[ns++] = B;
                }
                if (bad) break;
                wmu[j] = 0.0; wsg[j] = 0.0;
                if (ns >= 32) aaor_series_stats(series, ns, &wmu[j], &wsg[j], &dummy);
            }
            if (bad) { found = -1; break; }
        }
        uint64_t e = b1 < tau_b ? b1 : tau_b;
        int fail = 0;
        for (uint64_t tau = b0; tau < e && !fail; ++tau) {
            double best = 0.0; int32_t best_w = 0;
            for (int j = 0; j < nwidths; ++j) {
                uint64_t w = (uint64_t)widths[j];
                if (tau + w > nout) continue;
                if (tau % width_dec(w, wdec) != 0) continue;
                if (tau + w > d_first + d_count) { fail = 1; break; }
                int64_t B = 0;
                for (uint64_t i = 0; i < w; ++i) B += d[tau + i - d_first];
                double S;
                if (sigma_mode) {
                    if (!(wsg[j] > 0.0)) continue;
                    S = ((double)B - wmu[j]) / wsg[j];
                } else {
                    S = ((double)B - (double)w * mu) / (sigma * sqrt((double)w));
                }
                if (best_w == 0 || S > best) { best = S; best_w = (int32_t)w; }
            }
            if (!fail && best_w != 0 && best >= thr) {
                if (found < max_out) { out_tau[found] = tau; out_w[found] = best_w; out_snr[found] = best; }
                found++;
            }
        }
        if (fail) { found = -1; break; }
    }
    free(wmu); free(wsg); free(series);
    return found;
}

/* The search of steps 6-8 as BASELINE.json states it: every width at every tau, white-noise scaling. */
int64_t aaor_sps_row(const uint32_t *d, uint64_t d_first, uint64_t d_count,
                     uint64_t nout, uint64_t L,
                     const int32_t *widths, int nwidths, double thr,
                     uint64_t tau_a, uint64_t tau_b,
                     uint64_t *out_tau, int32_t *out_w, double *out_snr, int64_t max_out)
{
    return aaor_sps_row2(d, d_first, d_count, nout, L, widths, nwidths, thr, tau_a, tau_b, 0, 0, out_tau, out_w, out_snr, max_out);
}

/* ---- peak finding (reading A17) on a list sorted by (dm_index, t_start) ------------------------------------
 * keep[i] = 1 iff no neighbour beats candidate i.  Neighbours: |dm' - dm| <= 1 and the boxcars overlap or touch in
 * raw samples (t' <= t + w and t <= t' + w').  c' beats c iff snr' > snr, or snr' == snr and (dm', t') < (dm, t).
 * The definition is the all-pairs loop of oracle.find_peaks (python); this is the same test with the pairs that cannot
 * be neighbours left out: other rows than dm-1, dm, dm+1, and starts outside [t - wmax, t + w] (wmax = the largest
 * width in the list).  Pinned against the all-pairs loop on random lists. */
typedef struct { uint32_t dm_index, t_start, width; float snr; } aaor_cand;

void aaor_find_peaks(const aaor_cand *c, int64_t n, uint8_t *keep)
{
    uint64_t wmax = 0;
    for (int64_t i = 0; i < n; ++i) if (c[i].width > wmax) wmax = c[i].width;
    #pragma omp parallel for schedule(dynamic, 1024)
    for (int64_t i = 0; i < n; ++i) {
        keep[i] = 1;
        for (int dd = -1; dd <= 1 && keep[i]; ++dd) {
            int64_t dm = (int64_t)c[i].dm_index + dd;
            if (dm < 0) continue;
            int64_t t_lo = (int64_t)c[i].t_start - (int64_t)wmax, t_hi = (int64_t)c[i].t_start + (int64_t)c[i].width;
            /* first record with (dm_index, t_start) >= (dm, t_lo) */
            int64_t a = 0, b = n;
            while (a < b) {
                int64_t m = (a + b) / 2;
                if ((int64_t)c[m].dm_index < dm || ((int64_t)c[m].dm_index == dm && (int64_t)c[m].t_start < t_lo)) a = m + 1; else b = m;
            }
            for (int64_t j = a; j < n && (int64_t)c[j].dm_index == dm && (int64_t)c[j].t_start <= t_hi; ++j) {
                if (j == i) continue;
                if ((int64_t)c[i].t_start > (int64_t)c[j].t_start + (int64_t)c[j].width) continue;      /* not touching */
                int beats = c[j].snr > c[i].snr ||
                            (c[j].snr == c[i].snr && (c[j].dm_index < c[i].dm_index ||
                                                      (c[j].dm_index == c[i].dm_index && c[j].t_start < c[i].t_start)));
                if (beats) { keep[i] = 0; break; }
            }
        }
    }
}

int aaor_num_threads(void)
{
    int n = 1;
    #pragma omp parallel
    {
        #pragma omp single
        n =
#ifdef _OPENMP
            omp_get_num_threads();
#else
            1;
#endif
    }
    return n;
}
