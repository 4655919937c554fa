// Single-pulse search of one dedispersed sub-chunk.
//
// One CTA per (normalisation block, DM row):
//   1. robust mean / sigma: a plain pass and three 3-sigma-clip passes, each reducing the EXACT
//      integer sums (count, sum x, sum x^2); mu and sigma are formed from them with one rounding
//      each (128-bit integer numerator), so they equal the oracle's bit for bit;
//   2. boxcars: the block is processed in tiles; a block-wide prefix sum of each tile (warp
//      shuffles) gives B_w[tau] = P[tau+w] - P[tau] exactly for every width; an integer
//      pre-filter B_w >= floor(w mu + thr sigma sqrt w) - 1 discards almost every sample, the
//      survivors get the double-precision S/N of every width, the arg-max (ties -> smallest
//      width) and the threshold test;
//   3. candidates are appended to THIS STREAM's private list with one atomicAdd per warp
//      (warp-aggregated), so only candidates ever cross the host link.
// HBM-bound: the block (<= 256 KB) is read once from HBM and four more times from L2.
#include "aa_internal.h"

namespace aa {

namespace {

constexpr int NT = 256;
constexpr int TT = 2048;   // taus per tile

__device__ __forceinline__ double u128_to_double(unsigned __int128 v)
{
    // round-to-nearest-even conversion: keep the top 64 bits, fold the rest into a sticky bit
    const uint64_t hi = (uint64_t)(v >> 64);
    if (hi == 0) return __ull2double_rn((uint64_t)v);
    const int s = 64 - __clzll((long long)hi);
    uint64_t top = (uint64_t)(v >> s);
    const unsigned __int128 mask = (((unsigned __int128)1) << s) - 1;
    if ((v & mask) != 0) top |= 1ull;
    return ldexp(__ull2double_rn(top), s);
}

__device__ __forceinline__ uint64_t warp_sum(uint64_t v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

struct Shared {
    uint64_t red[5][NT / 32];
    double mu, sigma;
    uint64_t m;
    long long bthr[kMaxWidths];
    double den[kMaxWidths];
    unsigned long long warp_tot[NT / 32];
    int w[kMaxWidths];        // widths (a dynamically indexed kernel parameter would go through the ADU pipe)
    int dec[kMaxWidths];      // time grid of each width (reading A20): 1, or a power of two for widths above wdec
    // reading A18 (sigma_mode 1): the width's own robust mean and sigma, and the exact sums they are made from
    double wmu[kMaxWidths], wsg[kMaxWidths];
    uint64_t wacc[kMaxWidths][NT / 32][4];     // per width and warp: count, sum B, sum B^2 (low 64 bits, high 64 bits)
    uint64_t wcnt0[kMaxWidths];                // boxcars of the width in the block (first pass)
    int wdone[kMaxWidths];                     // the width's statistics are final (or it has none)
};

// BIG: the block's sum of squares may pass 2^64 (16-bit input on thousands of channels): every thread keeps its part
// as (low 64 bits, carries), the parts are added as three sums that cannot overflow and joined in 128 bits.
template <typename ACC, bool BIG = false>
__global__ void __launch_bounds__(NT) sps_kernel(const SpsArgs a, const __grid_constant__ WidthTable wt)
{
    extern __shared__ __align__(16) uint8_t dyn[];
    ACC *P = reinterpret_cast<ACC *>(dyn);          // exclusive prefix sums of the current tile
    __shared__ Shared sh;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d = blockIdx.y;
    if (tid < kMaxWidths) { sh.w[tid] = wt.w[tid]; sh.dec[tid] = wt.dec[tid]; }
    const int64_t b0 = (int64_t)blockIdx.x * a.block_len;
    int64_t b1 = b0 + a.block_len;
    if (b1 > a.nout_left) b1 = a.nout_left;
    if (b0 >= b1 || b0 >= a.nemit) return;
    const int64_t n_k = b1 - b0;
    const uint32_t *row = a.D + (size_t)d * a.pitch;

    // ---- 1. statistics ------------------------------------------------------------------
    double mu = 0.0, sigma = 0.0;
    for (int pass = 0; pass < 4; ++pass) {
        const double lim = __dmul_rn(3.0, sigma);
        uint64_t m = 0, S1 = 0, S2 = 0, carry = 0;
        for (int64_t i = b0 + tid; i < b1; i += NT) {
            const uint32_t x = row[i];
            const bool sel = (pass == 0) || (fabs(__dsub_rn((double)x, mu)) <= lim);
            if (sel) {
                m += 1;
                S1 += x;
                const uint64_t sq = (uint64_t)x * x;
                S2 += sq;
                if (BIG) carry += S2 < sq;
            }
        }
        m = warp_sum(m); S1 = warp_sum(S1);
        if (BIG) {
            const uint64_t lo = warp_sum(S2 & 0xFFFFFFFFull), hi = warp_sum(S2 >> 32);
            carry = warp_sum(carry);
            if (lane == 0) { sh.red[2][warp] = lo; sh.red[3][warp] = hi; sh.red[4][warp] = carry; }
        } else {
            S2 = warp_sum(S2);
            if (lane == 0) sh.red[2][warp] = S2;
        }
        if (lane == 0) { sh.red[0][warp] = m; sh.red[1][warp] = S1; }
        __syncthreads();
        if (tid == 0) {
            m = S1 = 0;
            unsigned __int128 S2w = 0;
            for (int w = 0; w < NT / 32; ++w) {
                m += sh.red[0][w]; S1 += sh.red[1][w];
                S2w += sh.red[2][w];
                if (BIG) S2w += ((unsigned __int128)sh.red[3][w] << 32) + ((unsigned __int128)sh.red[4][w] << 64);
            }
            sh.m = m;
            if (m) {
                const unsigned __int128 N = (unsigned __int128)m * S2w - (unsigned __int128)S1 * S1;
                const double dm = __ull2double_rn(m);
                sh.mu = __ddiv_rn(__ull2double_rn(S1), dm);
                sh.sigma = __dsqrt_rn(__ddiv_rn(u128_to_double(N), __dmul_rn(dm, dm)));
            }
        }
        __syncthreads();
        const uint64_t msel = sh.m;
        if (msel) { mu = sh.mu; sigma = sh.sigma; }
        __syncthreads();
        if (!msel) break;
    }
    if (!(sigma > 0.0) || n_k < 32) return;

    const int64_t e = b1 < a.nemit ? b1 : (int64_t)a.nemit;     // taus [b0, e) may emit
    const int64_t navail = a.ncols < a.nout_left ? (int64_t)a.ncols : a.nout_left;
    const int halo = a.wmax - 1;
    const int ept = (TT + halo + 1 + NT - 1) / NT;              // scan slots per thread (covers P[0..TT+halo])
    const bool measured = a.sigma_mode != 0;                    // reading A18

    // block-wide exclusive prefix sum of row[ts .. ts+n_in) into P[0 .. n_in]; returns n_in
    auto build_prefix = [&](int64_t ts) -> int64_t {
        int64_t n_in = navail - ts;
        if (n_in > TT + halo) n_in = TT + halo;
        {
            const int64_t i0 = (int64_t)tid * ept;
            ACC run = 0;
            for (int k = 0; k < ept; ++k) {
                const int64_t i = i0 + k;
                if (i < n_in) run += (ACC)row[ts + i];
            }
            unsigned long long incl = (unsigned long long)run;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                unsigned long long v = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += v;
            }
            if (lane == 31) sh.warp_tot[warp] = incl;
            __syncthreads();
            unsigned long long base = 0;
            for (int w = 0; w < warp; ++w) base += sh.warp_tot[w];
            ACC pre = (ACC)(base + incl - (unsigned long long)run);   // exclusive prefix of this thread
            for (int k = 0; k < ept; ++k) {
                const int64_t i = i0 + k;
                if (i <= n_in) P[i] = pre;
                if (i < n_in) pre += (ACC)row[ts + i];
            }
            __syncthreads();
        }
        return n_in;
    };

    // ---- 2a. reading A18: robust statistics of every width's own boxcar series over the block ----------------------
    // The series of width w is B_w[t] for the t of the block on the width's grid (A20) with t + w <= nout.  The block does
    // not fit shared memory here (64-bit sums, or a block no cluster takes), so each of the four passes of the estimator
    // sweeps the block tile by tile through the same prefix sums as the search and adds up the exact integers
    // (count, sum B, sum B^2 in 128 bits) of all widths at once; mu_w, sigma_w are formed as for the block itself.
    if (measured) {
        if (tid < kMaxWidths) {
            sh.wmu[tid] = 0.0; sh.wsg[tid] = 0.0; sh.wcnt0[tid] = 0;
            sh.wdone[tid] = tid < a.nwidths ? 0 : 1;
        }
        __syncthreads();
        for (int pass = 0; pass < 4; ++pass) {
            for (int i = tid; i < kMaxWidths * (NT / 32) * 4; i += NT) (&sh.wacc[0][0][0])[i] = 0;
            bool open = false;
            for (int j = 0; j < a.nwidths; ++j) open |= !sh.wdone[j];
            __syncthreads();
            if (!open) break;                                   // uniform
            for (int64_t ts = b0; ts < b1; ts += TT) {
                const int64_t n_in = build_prefix(ts);
                for (int j = 0; j < a.nwidths; ++j) {
                    if (sh.wdone[j]) continue;                  // uniform
                    const int w = sh.w[j];
                    const uint32_t gm = (uint32_t)(sh.dec[j] - 1);
                    const double wm = sh.wmu[j], lim = __dmul_rn(3.0, sh.wsg[j]);
                    uint64_t m = 0, S1 = 0;
                    unsigned __int128 S2 = 0;
                    for (int q = 0; q < TT / NT; ++q) {
                        const int tl = q * NT + tid;
                        const int64_t tau = ts + tl;
                        if (tau < b1 && tau + w <= a.nout_left && tl + w <= n_in && ((a.tau0 + (uint32_t)tau) & gm) == 0) {
                            const uint64_t B = (uint64_t)(ACC)(P[tl + w] - P[tl]);
                            if (pass == 0 || fabs(__dsub_rn((double)B, wm)) <= lim) {
                                m += 1;
                                S1 += B;
                                S2 += (unsigned __int128)B * B;
                            }
                        }
                    }
                    m = warp_sum(m); S1 = warp_sum(S1);
                    const uint64_t lo = (uint64_t)S2;
                    const uint64_t l0 = warp_sum(lo & 0xFFFFFFFFull), l1 = warp_sum(lo >> 32), hi = warp_sum((uint64_t)(S2 >> 64));
                    if (lane == 0) {
                        uint64_t *acc = sh.wacc[j][warp];
                        const unsigned __int128 cur = ((unsigned __int128)acc[3] << 64 | acc[2]) + (unsigned __int128)l0 +
                                                      ((unsigned __int128)l1 << 32) + ((unsigned __int128)hi << 64);
                        acc[0] += m; acc[1] += S1; acc[2] = (uint64_t)cur; acc[3] = (uint64_t)(cur >> 64);
                    }
                }
                __syncthreads();                                // the next tile overwrites P
            }
            if (tid < a.nwidths && !sh.wdone[tid]) {
                uint64_t m = 0, S1 = 0;
                unsigned __int128 S2 = 0;
                for (int wp = 0; wp < NT / 32; ++wp) {
                    m += sh.wacc[tid][wp][0]; S1 += sh.wacc[tid][wp][1];
                    S2 += ((unsigned __int128)sh.wacc[tid][wp][3] << 64) | sh.wacc[tid][wp][2];
                }
                if (pass == 0) sh.wcnt0[tid] = m;
                if (m == 0 || sh.wcnt0[tid] < 32) {
                    sh.wdone[tid] = 1;                          // fewer than 32 boxcars: no statistics; an empty clip keeps the last ones
                } else {
                    const unsigned __int128 N = (unsigned __int128)m * S2 - (unsigned __int128)S1 * S1;
                    const double dm = __ull2double_rn(m);
                    sh.wmu[tid] = __ddiv_rn(__ull2double_rn(S1), dm);
                    sh.wsg[tid] = __dsqrt_rn(__ddiv_rn(u128_to_double(N), __dmul_rn(dm, dm)));
                }
            }
            __syncthreads();
        }
    }

    // ---- 2. per-width constants ---------------------------------------------------------
    if (tid < a.nwidths) {
        if (measured) {
            const double sg = sh.wcnt0[tid] >= 32 ? sh.wsg[tid] : 0.0;
            const bool ok = sg > 0.0;
            sh.den[tid] = ok ? sg : 0.0;
            // B >= floor(mu_w + thr sigma_w) - 1 is necessary for S >= thr; a width without statistics never hits
            sh.bthr[tid] = ok ? __double2ll_rd(sh.wmu[tid] + a.thr * sg) - 1 : 0x7FFFFFFFFFFFFFFFll;
        } else {
            const double w = (double)sh.w[tid];
            const double den = __dmul_rn(sigma, __dsqrt_rn(w));
            sh.den[tid] = den;
            sh.bthr[tid] = __double2ll_rd(w * mu + a.thr * den) - 1;
        }
    }
    __syncthreads();

    for (int64_t ts = b0; ts < e; ts += TT) {
        build_prefix(ts);
        // boxcars
        for (int q = 0; q < TT / NT; ++q) {
            const int tl = q * NT + tid;                 // tau within the tile
            const int64_t tau = ts + tl;                 // tau within the sub-chunk
            bool has = false;
            int best_w = 0;
            double best = 0.0;
            if (tau < e) {
                const ACC p0 = P[tl];
                bool any = false;
                const uint32_t tabs = a.tau0 + (uint32_t)tau;          // absolute binned sample: the grids of A20 live on it
                for (int j = 0; j < a.nwidths; ++j) {
                    const int w = sh.w[j];
                    if (tau + w <= a.nout_left && (tabs & (uint32_t)(sh.dec[j] - 1)) == 0) {
                        const long long B = (long long)(ACC)(P[tl + w] - p0);
                        any |= (B >= sh.bthr[j]);
                    }
                }
                if (any) {
                    for (int j = 0; j < a.nwidths; ++j) {
                        const int w = sh.w[j];
                        if (tau + w > a.nout_left || (tabs & (uint32_t)(sh.dec[j] - 1)) != 0) continue;
                        const long long B = (long long)(ACC)(P[tl + w] - p0);
                        double S;
                        if (measured) {
                            const double sg = sh.den[j];
                            if (!(sg > 0.0)) continue;
                            S = __ddiv_rn(__dsub_rn((double)B, sh.wmu[j]), sg);
                        } else {
                            S = __ddiv_rn(__dsub_rn((double)B, __dmul_rn((double)w, mu)), sh.den[j]);
                        }
                        if (best_w == 0 || S > best) { best = S; best_w = w; }
                    }
                    has = (best_w != 0) && (best >= a.thr);
                }
            }
            // warp-aggregated append to this stream's private list
            const unsigned mask = __ballot_sync(0xffffffffu, has);
            if (mask) {
                uint32_t base = 0;
                const int leader = __ffs(mask) - 1;
                if (lane == leader) base = atomicAdd(a.count, (uint32_t)__popc(mask));
                base = __shfl_sync(0xffffffffu, base, leader);
                if (has) {
                    const uint32_t slot = base + __popc(mask & ((1u << lane) - 1));
                    if (slot < a.cap) {
                        aa_candidate c;
                        c.dm_index = a.dm_base + (uint32_t)d;
                        c.t_start = (a.tau0 + (uint32_t)tau) * a.bin;
                        c.width = (uint32_t)best_w * a.bin;
                        c.snr = (float)best;
                        a.cands[slot] = c;
                    }
                }
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// Cluster variant (32-bit boxcar sums, block_len % (4 C) == 0): the normalisation block of one DM row
// is split over a thread-block cluster of C CTAs, each keeping its segment (<= kSegMax samples plus the
// boxcar tail) in shared memory, so the dedispersed series is read from HBM exactly once:
//   load     one cp.async.bulk (TMA 1-D) of the segment + tail onto an mbarrier;
//   stats    the four passes run on shared memory; the 3-sigma selection |x - mu| <= 3 sigma (double, as
//            in the oracle) is turned into the exact integer interval [lo, hi] it selects, the partial
//            sums (m, sum x, sum x^2: exact integers) of every CTA are written into every CTA's shared
//            memory (DSMEM) and added in rank order after a cluster barrier, so all CTAs form the same
//            mu and sigma, bit for bit the single-CTA values;
//   boxcars  in-place exclusive prefix sum of segment + tail (mod 2^32; differences are exact), then four
//            taus per thread: B_w = P[tau+w] - P[tau] against the integer pre-filter; survivors take the
//            same double-precision path as the generic kernel.
constexpr int NT2 = 256;
constexpr int kSegMax = 16384;
constexpr int kMaxCluster = 8;

struct SharedC {
    uint64_t red[5][NT2 / 32];
    uint64_t part[2][kMaxCluster][4];   // [parity of the reduction][rank] partial sums, written by the CTA of that rank
    uint64_t bar;                       // mbarrier of the bulk load
    double mu, sigma;
    uint64_t m;
    uint32_t lo, hi;
    int empty;
    uint32_t thr_u[kMaxWidths];
    double den[kMaxWidths];             // sigma sqrt(w) (A10) or the width's own sigma (A18)
    double wmu[kMaxWidths];             // A18: the width's own mean
    int w[kMaxWidths];
    int dec[kMaxWidths];
    uint32_t warp_tot[NT2 / 32];
    uint4 wl[kMaxWidths + 1];           // (width, pre-filter threshold, grid, -): multiples of 4 first, then the others, then coarse grids
    int na, nu, nd;
};

__device__ __forceinline__ bool clip_pred(double x, double mu, double lim)
{
    return fabs(__dsub_rn(x, mu)) <= lim;
}

// The integers x in [0, 2^32) with |x - mu| <= lim (evaluated as the oracle does, in double) form an
// interval, because the rounded difference is monotone in x.  Returns false if it is empty.
__device__ bool clip_interval(double mu, double lim, uint32_t &lo, uint32_t &hi)
{
    const double top = 4294967295.0;
    double l = ceil(mu - lim), h = floor(mu + lim);
    if (l < 0.0) l = 0.0;
    if (h > top) h = top;
    if (!(l <= top) || !(h >= 0.0)) return false;
    for (int it = 0; it < 4 && l > 0.0 && clip_pred(l - 1.0, mu, lim); ++it) l -= 1.0;
    for (int it = 0; it < 8 && l < top && !clip_pred(l, mu, lim); ++it) l += 1.0;
    for (int it = 0; it < 4 && h < top && clip_pred(h + 1.0, mu, lim); ++it) h += 1.0;
    for (int it = 0; it < 8 && h > 0.0 && !clip_pred(h, mu, lim); ++it) h -= 1.0;
    if (!clip_pred(l, mu, lim) || !clip_pred(h, mu, lim) || l > h) return false;
    lo = (uint32_t)l;
    hi = (uint32_t)h;
    return true;
}

__device__ __forceinline__ uint32_t cluster_rank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void st_cluster_u64(const void *local, uint32_t rank, uint64_t v)
{
    uint32_t a = (uint32_t)__cvta_generic_to_shared(local), r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    asm volatile("st.shared::cluster.u64 [%0], %1;" ::"r"(r), "l"(v) : "memory");
}

// Exact moments over the whole cluster.  Every thread brings its part (count, sum, sum of squares as low 64 bits plus
// carries); the CTA's totals go to every CTA's shared memory (DSMEM), are added in rank order after a cluster barrier,
// and mu = S1 / m, sigma = sqrt((m S2 - S1^2) / m^2) are formed from the 128-bit integers with one rounding each, so
// all CTAs hold bit-identical values, equal to the oracle's.  `turn` alternates the DSMEM slot: the barrier of one
// reduction separates the reads of the previous one from the writes of the next.  Returns the count.
__device__ __forceinline__ uint64_t cluster_moments(SharedC &sh, int C, uint32_t rank, int &turn, uint64_t m, uint64_t S1, uint64_t S2,
                                                    uint64_t carry, double &mu, double &sigma)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    m = warp_sum(m); S1 = warp_sum(S1);
    const uint64_t lo = warp_sum(S2 & 0xFFFFFFFFull), hi = warp_sum(S2 >> 32);
    carry = warp_sum(carry);
    if (lane == 0) { sh.red[0][warp] = m; sh.red[1][warp] = S1; sh.red[2][warp] = lo; sh.red[3][warp] = hi; sh.red[4][warp] = carry; }
    __syncthreads();
    const int slot = turn & 1;
    ++turn;
    if (tid == 0) {
        m = S1 = 0;
        unsigned __int128 S2w = 0;
        for (int w = 0; w < NT2 / 32; ++w) {
            m += sh.red[0][w]; S1 += sh.red[1][w];
            S2w += (unsigned __int128)sh.red[2][w] + ((unsigned __int128)sh.red[3][w] << 32) + ((unsigned __int128)sh.red[4][w] << 64);
        }
        if (C > 1) {
            for (int r = 0; r < C; ++r) {
                st_cluster_u64(&sh.part[slot][rank][0], (uint32_t)r, m);
                st_cluster_u64(&sh.part[slot][rank][1], (uint32_t)r, S1);
                st_cluster_u64(&sh.part[slot][rank][2], (uint32_t)r, (uint64_t)S2w);
                st_cluster_u64(&sh.part[slot][rank][3], (uint32_t)r, (uint64_t)(S2w >> 64));
            }
        } else {
            sh.part[slot][0][0] = m; sh.part[slot][0][1] = S1; sh.part[slot][0][2] = (uint64_t)S2w; sh.part[slot][0][3] = (uint64_t)(S2w >> 64);
        }
    }
    if (C > 1) cluster_sync_all(); else __syncthreads();
    if (tid == 0) {
        m = S1 = 0;
        unsigned __int128 S2w = 0;
        for (int r = 0; r < C; ++r) {
            m += sh.part[slot][r][0]; S1 += sh.part[slot][r][1];
            S2w += (unsigned __int128)sh.part[slot][r][2] + ((unsigned __int128)sh.part[slot][r][3] << 64);
        }
        sh.m = m;
        if (m) {
            const unsigned __int128 N = (unsigned __int128)m * S2w - (unsigned __int128)S1 * S1;
            const double dm = __ull2double_rn(m);
            sh.mu = __ddiv_rn(__ull2double_rn(S1), dm);
            sh.sigma = __dsqrt_rn(__ddiv_rn(u128_to_double(N), __dmul_rn(dm, dm)));
        }
    }
    __syncthreads();
    const uint64_t msel = sh.m;
    if (msel) { mu = sh.mu; sigma = sh.sigma; }
    __syncthreads();
    return msel;
}

// SMALL: every boxcar sum is below 2^31 (maxsample nchans bin wmax < 2^31), so the pre-filter B >= th is the sign of
// (th - 1) - B and costs one 3-input add and one OR per (tau, width).
template <bool SMALL>
__global__ void __launch_bounds__(NT2) sps_cluster_kernel(const SpsArgs a, const __grid_constant__ WidthTable wt, const int C, const int seg)
{
    extern __shared__ __align__(16) uint8_t dyn[];
    uint32_t *X = reinterpret_cast<uint32_t *>(dyn);     // segment + tail; later its exclusive prefix sums
    __shared__ SharedC sh;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d = blockIdx.y;
    const uint32_t rank = C > 1 ? cluster_rank() : 0u;
    const int64_t blk = blockIdx.x / C;
    if (tid < kMaxWidths) { sh.w[tid] = wt.w[tid]; sh.dec[tid] = wt.dec[tid]; }
    const int64_t b0 = blk * a.block_len;
    int64_t b1 = b0 + a.block_len;
    if (b1 > a.nout_left) b1 = a.nout_left;
    if (b0 >= b1 || b0 >= a.nemit) return;               // uniform over the cluster
    const int64_t n_k = b1 - b0;
    const uint32_t *row = a.D + (size_t)d * a.pitch;
    const int64_t s0 = b0 + (int64_t)rank * seg;         // first column of this CTA's segment
    const int64_t navail = a.ncols < a.nout_left ? (int64_t)a.ncols : a.nout_left;
    const int halo = a.wmax - 1;
    int64_t n_in = navail - s0;                          // columns this CTA holds: segment + boxcar tail
    if (n_in > seg + halo) n_in = seg + halo;
    if (n_in < 0) n_in = 0;
    int64_t n_own = b1 - s0;                             // columns of the block inside the segment
    if (n_own > seg) n_own = seg;
    if (n_own < 0) n_own = 0;
    const bool measured = a.sigma_mode != 0;             // reading A18

    // ---- load -------------------------------------------------------------------------------
    const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&sh.bar);
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (C > 1) cluster_sync_all();                       // every CTA of the cluster runs before DSMEM is written
    if (n_in > 0) {
        if (tid == 0) {
            // whole 16-byte pieces; the row pitch leaves room past the last column
            const uint32_t bytes = (uint32_t)((n_in + 3) / 4 * 16);
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                             (uint32_t)__cvta_generic_to_shared(X)),
                         "l"(row + s0), "r"(bytes), "r"(bar)
                         : "memory");
        }
        uint32_t ok = 0;
        while (!ok)
            asm volatile(
                "{\n\t.reg .pred p;\n\t"
                "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\t"
                "selp.u32 %0, 1, 0, p;\n\t}"
                : "=r"(ok)
                : "r"(bar)
                : "memory");
    }

    // ---- 1. statistics of the block (A8) -------------------------------------------------------
    double mu = 0.0, sigma = 0.0;
    int turn = 0;
    const int n4 = (int)(n_own / 4);
    for (int pass = 0; pass < 4; ++pass) {
        uint32_t lo = 0u, span = 0xFFFFFFFFu;
        bool run = true;
        if (pass > 0) {
            if (tid == 0) {
                uint32_t l = 0, h = 0;
                sh.empty = clip_interval(mu, __dmul_rn(3.0, sigma), l, h) ? 0 : 1;
                sh.lo = l;
                sh.hi = h;
            }
            __syncthreads();
            run = !sh.empty;
            lo = sh.lo;
            span = sh.hi - lo;
        }
        uint64_t m = 0, S1 = 0, S2 = 0;
        if (pass == 0) {                                  // every sample: no selection
            uint32_t mc = 0;
            for (int i = tid; i < n4; i += NT2) {
                const uint4 v = reinterpret_cast<const uint4 *>(X)[i];
                S1 += (uint64_t)v.x + v.y;
                S1 += (uint64_t)v.z + v.w;
                S2 += (uint64_t)v.x * v.x;
                S2 += (uint64_t)v.y * v.y;
                S2 += (uint64_t)v.z * v.z;
                S2 += (uint64_t)v.w * v.w;
                mc += 4;
            }
            for (int i = 4 * n4 + tid; i < n_own; i += NT2) {
                const uint32_t x = X[i];
                mc += 1;
                S1 += x;
                S2 += (uint64_t)x * x;
            }
            m = mc;
        } else if (run) {
            uint32_t mc = 0;
            for (int i = tid; i < n4; i += NT2) {
                const uint4 v = reinterpret_cast<const uint4 *>(X)[i];
                const uint32_t xs[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const bool sel = (xs[k] - lo) <= span;
                    const uint32_t x = sel ? xs[k] : 0u;
                    mc += sel ? 1u : 0u;
                    S1 += x;
                    S2 += (uint64_t)x * x;
                }
            }
            for (int i = 4 * n4 + tid; i < n_own; i += NT2) {
                const uint32_t x = X[i];
                if ((x - lo) <= span) {
                    mc += 1;
                    S1 += x;
                    S2 += (uint64_t)x * x;
                }
            }
            m = mc;
        }
        // (the launcher sends blocks whose sum of squares could pass 2^64 to the generic kernel: no carries here)
        if (!cluster_moments(sh, C, rank, turn, m, S1, S2, 0, mu, sigma)) break;
    }
    if (!(sigma > 0.0) || n_k < 32) return;

    // ---- 2. exclusive prefix sums in place: X[i] <- sum_{j<i} X[j], i <= n_in; constant beyond ------
    {
        const int total = seg + halo + 8;                 // slots the boxcar loop may read
        int chunk = (int)((n_in + 1 + NT2 - 1) / NT2);    // slots 0 .. n_in
        chunk |= 1;                                       // odd stride: conflict-free
        const int64_t i0 = (int64_t)tid * chunk;
        const bool inside = i0 + chunk <= n_in;           // the whole chunk holds data: no per-element tests
        uint32_t run = 0;
        if (inside) {
#pragma unroll 5
            for (int k = 0; k < chunk; ++k) run += X[i0 + k];
        } else {
            for (int k = 0; k < chunk; ++k)
                if (i0 + k < n_in) run += X[i0 + k];
        }
        uint32_t incl = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        if (lane == 31) sh.warp_tot[warp] = incl;
        __syncthreads();
        uint32_t pre = incl - run;
        for (int w = 0; w < warp; ++w) pre += sh.warp_tot[w];
        if (inside) {
            uint32_t *xp = X + i0;
#pragma unroll 5
            for (int k = 0; k < chunk; ++k) {
                const uint32_t x = xp[k];
                xp[k] = pre;
                pre += x;
            }
            if (i0 + chunk == n_in) xp[chunk] = pre;
        } else {
            for (int k = 0; k < chunk; ++k) {
                const int64_t i = i0 + k;
                if (i < n_in) {
                    const uint32_t x = X[i];
                    X[i] = pre;
                    pre += x;
                } else if (i == n_in) {
                    X[i] = pre;
                }
            }
        }
        __syncthreads();
        const uint32_t last = X[n_in];
        for (int64_t i = n_in + 1 + tid; i < total; i += NT2) X[i] = last;
        __syncthreads();
    }

    // ---- 3. per-width constants ---------------------------------------------------------------
    const uint32_t tabs0 = a.tau0 + (uint32_t)s0;          // absolute binned sample of X[0]: a multiple of 4
    if (measured) {
        // reading A18: the robust statistics (A8) of each width's own boxcar series over the block, on the width's
        // grid (A20), from the prefix sums: B = X[t + w] - X[t] (exact modulo 2^32: every sum is below 2^32)
        for (int j = 0; j < a.nwidths; ++j) {
            const int w = sh.w[j];
            const uint32_t gm = (uint32_t)(sh.dec[j] - 1);
            int64_t nv = a.nout_left - s0 - w + 1;        // columns t of this segment with t + w <= nout
            if (nv > n_own) nv = n_own;
            double wm = 0.0, ws = 0.0;
            uint64_t cnt0 = 0;
            for (int pass = 0; pass < 4; ++pass) {
                uint32_t lo = 0u, span = 0xFFFFFFFFu;
                bool run = true;
                if (pass > 0) {
                    if (tid == 0) {
                        uint32_t l = 0, h = 0;
                        sh.empty = clip_interval(wm, __dmul_rn(3.0, ws), l, h) ? 0 : 1;
                        sh.lo = l;
                        sh.hi = h;
                    }
                    __syncthreads();
                    run = !sh.empty;
                    lo = sh.lo;
                    span = sh.hi - lo;
                }
                uint64_t m = 0, S1 = 0, S2 = 0, carry = 0;
                if (run) {
                    for (int64_t t = tid; t < nv; t += NT2) {
                        if ((tabs0 + (uint32_t)t) & gm) continue;
                        const uint32_t B = X[t + w] - X[t];
                        if ((B - lo) <= span) {
                            m += 1;
                            S1 += B;
                            const uint64_t sq = (uint64_t)B * B;
                            S2 += sq;
                            carry += S2 < sq;
                        }
                    }
                }
                const uint64_t got = cluster_moments(sh, C, rank, turn, m, S1, S2, carry, wm, ws);
                if (pass == 0) cnt0 = got;
                if (!got || cnt0 < 32) break;              // uniform over the cluster
            }
            if (tid == 0) {
                const bool ok = cnt0 >= 32 && ws > 0.0;
                sh.wmu[j] = wm;
                sh.den[j] = ok ? ws : 0.0;
                // B >= floor(mu_w + thr sigma_w) - 1 is necessary for S >= thr; a width without statistics never hits
                const long long bt = ok ? __double2ll_rd(wm + a.thr * ws) - 1 : 0x7FFFFFFFFFFFll;
                sh.thr_u[j] = bt <= 0 ? 0u : (bt >= 0xFFFFFFFFll ? 0xFFFFFFFFu : (uint32_t)bt);
            }
        }
        __syncthreads();
    } else {
        if (tid < a.nwidths) {
            const double w = (double)sh.w[tid];
            const double den = __dmul_rn(sigma, __dsqrt_rn(w));
            sh.den[tid] = den;
            // B >= floor(w mu + thr sigma sqrt w) - 1 is necessary for S >= thr; clamped to the 32-bit sums
            const long long bt = __double2ll_rd(w * mu + a.thr * den) - 1;
            sh.thr_u[tid] = bt <= 0 ? 0u : (bt >= 0xFFFFFFFFll ? 0xFFFFFFFFu : (uint32_t)bt);
        }
        __syncthreads();
    }
    if (tid == 0) {
        // SMALL: th - 1 as a signed number, B >= th  <=>  (th - 1) - B < 0; th above every possible B -> never
        auto enc = [&](uint32_t th) { return SMALL ? (th == 0u ? 0xFFFFFFFFu : (th > 0x7FFFFFFFu ? 0x7FFFFFFFu : th - 1u)) : th; };
        int n = 0;
        for (int j = 0; j < a.nwidths; ++j)
            if (sh.dec[j] == 1 && (sh.w[j] & 3) == 0) sh.wl[n++] = make_uint4((uint32_t)sh.w[j], enc(sh.thr_u[j]), 1u, 0u);
        sh.na = n;
        for (int j = 0; j < a.nwidths; ++j)
            if (sh.dec[j] == 1 && (sh.w[j] & 3) != 0) sh.wl[n++] = make_uint4((uint32_t)sh.w[j], enc(sh.thr_u[j]), 1u, 0u);
        sh.nu = n - sh.na;
        for (int j = 0; j < a.nwidths; ++j)
            if (sh.dec[j] > 1) sh.wl[n++] = make_uint4((uint32_t)sh.w[j], enc(sh.thr_u[j]), (uint32_t)sh.dec[j], 0u);
        sh.nd = n - sh.na - sh.nu;
    }
    __syncthreads();

    const int64_t n_emit = n_own;                         // taus [0, n_emit) of this segment may emit (blocks tile the sub-chunk)
    if (n_emit <= 0) return;                              // nothing after this point is cluster-wide

    // ---- 4. boxcars, eight taus per thread -----------------------------------------------------------
    // (two groups of four, NT2 groups apart, so that every 16-byte access of a warp is contiguous)
    const int ngroups = (int)((n_emit + 3) / 4);
    const int nw = a.nwidths, na = sh.na, nu = sh.nu, nd = sh.nd;
    constexpr int GB = 4 * NT2;                          // distance of the second group in samples
    for (int g0 = 0; g0 < ngroups; g0 += 2 * NT2) {
        const int g = g0 + tid;
        uint32_t any = 0;
        uint32_t f0 = 0, f1 = 0, f2 = 0, f3 = 0, f4 = 0, f5 = 0, f6 = 0, f7 = 0;   // SMALL: sign bits collect the hits
        if (g < ngroups) {
            const bool two = g + NT2 < ngroups;          // else the second group repeats the first
            const uint32_t *xg = X + 4 * g;
            const int gb = two ? GB : 0;
            const uint4 pa = *reinterpret_cast<const uint4 *>(xg), pb = *reinterpret_cast<const uint4 *>(xg + gb);
            // widths that are multiples of 4: aligned 16-byte loads
#pragma unroll 2
            for (int j = 0; j < na; ++j) {
                const uint4 wt2 = sh.wl[j];
                const uint32_t th = wt2.y;
                const uint4 qa = *reinterpret_cast<const uint4 *>(xg + wt2.x);
                const uint4 qb = *reinterpret_cast<const uint4 *>(xg + wt2.x + gb);
                if (SMALL) {
                    f0 |= th + pa.x - qa.x; f1 |= th + pa.y - qa.y; f2 |= th + pa.z - qa.z; f3 |= th + pa.w - qa.w;
                    f4 |= th + pb.x - qb.x; f5 |= th + pb.y - qb.y; f6 |= th + pb.z - qb.z; f7 |= th + pb.w - qb.w;
                    continue;
                }
                any |= ((qa.x - pa.x) >= th ? 1u : 0u) | ((qa.y - pa.y) >= th ? 2u : 0u) | ((qa.z - pa.z) >= th ? 4u : 0u) |
                       ((qa.w - pa.w) >= th ? 8u : 0u) | ((qb.x - pb.x) >= th ? 16u : 0u) | ((qb.y - pb.y) >= th ? 32u : 0u) |
                       ((qb.z - pb.z) >= th ? 64u : 0u) | ((qb.w - pb.w) >= th ? 128u : 0u);
            }
            // the others: the aligned pieces around tau + w, shifted by w mod 4 (uniform)
#pragma unroll 1
            for (int j = na; j < na + nu; ++j) {
                const uint4 wt2 = sh.wl[j];
                const uint32_t th = wt2.y;
                const int r = (int)(wt2.x & 3u);
                const uint32_t *xq = xg + (wt2.x - (uint32_t)r);
                const uint4 q0 = *reinterpret_cast<const uint4 *>(xq), q1 = *reinterpret_cast<const uint4 *>(xq + 4),
                            q2 = *reinterpret_cast<const uint4 *>(xq + gb), q3 = *reinterpret_cast<const uint4 *>(xq + gb + 4);
                uint32_t v0, v1, v2, v3, v4, v5, v6, v7;
                if (r == 1) { v0 = q0.y; v1 = q0.z; v2 = q0.w; v3 = q1.x; v4 = q2.y; v5 = q2.z; v6 = q2.w; v7 = q3.x; }
                else if (r == 2) { v0 = q0.z; v1 = q0.w; v2 = q1.x; v3 = q1.y; v4 = q2.z; v5 = q2.w; v6 = q3.x; v7 = q3.y; }
                else { v0 = q0.w; v1 = q1.x; v2 = q1.y; v3 = q1.z; v4 = q2.w; v5 = q3.x; v6 = q3.y; v7 = q3.z; }
                if (SMALL) {
                    f0 |= th + pa.x - v0; f1 |= th + pa.y - v1; f2 |= th + pa.z - v2; f3 |= th + pa.w - v3;
                    f4 |= th + pb.x - v4; f5 |= th + pb.y - v5; f6 |= th + pb.z - v6; f7 |= th + pb.w - v7;
                    continue;
                }
                any |= ((v0 - pa.x) >= th ? 1u : 0u) | ((v1 - pa.y) >= th ? 2u : 0u) | ((v2 - pa.z) >= th ? 4u : 0u) |
                       ((v3 - pa.w) >= th ? 8u : 0u) | ((v4 - pb.x) >= th ? 16u : 0u) | ((v5 - pb.y) >= th ? 32u : 0u) |
                       ((v6 - pb.z) >= th ? 64u : 0u) | ((v7 - pb.w) >= th ? 128u : 0u);
            }
            // widths on a coarser grid (A20): grid 2 looks at taus 0 and 2 of a group, grid 4 and beyond at tau 0, and
            // only in the groups that start on the grid (tabs0 and GB are multiples of 4 and of every grid up to 1024)
#pragma unroll 1
            for (int j = na + nu; j < na + nu + nd; ++j) {
                const uint4 wt2 = sh.wl[j];
                const uint32_t th = wt2.y, grid = wt2.z;
                const uint32_t ga = tabs0 + 4u * (uint32_t)g;
                const bool ok_a = grid <= 4u || !(ga & (grid - 1u)), ok_b = grid <= 4u || !((ga + (uint32_t)gb) & (grid - 1u));
                if (!ok_a && !ok_b) continue;
                const uint32_t *xq = xg + wt2.x;
                const uint32_t a0 = xq[0], b0 = xq[gb];
                if (SMALL) {
                    if (ok_a) f0 |= th + pa.x - a0;
                    if (ok_b) f4 |= th + pb.x - b0;
                } else {
                    any |= (ok_a && (a0 - pa.x) >= th ? 1u : 0u) | (ok_b && (b0 - pb.x) >= th ? 16u : 0u);
                }
                if (grid == 2u) {
                    const uint32_t a2 = xq[2], b2 = xq[gb + 2];
                    if (SMALL) { f2 |= th + pa.z - a2; f6 |= th + pb.z - b2; }
                    else any |= ((a2 - pa.z) >= th ? 4u : 0u) | ((b2 - pb.z) >= th ? 64u : 0u);
                }
            }
        }
        if (SMALL)
            any = (f0 >> 31) | (f1 >> 31) << 1 | (f2 >> 31) << 2 | (f3 >> 31) << 3 | (f4 >> 31) << 4 | (f5 >> 31) << 5 |
                  (f6 >> 31) << 6 | (f7 >> 31) << 7;
        if (g < ngroups && g + NT2 >= ngroups) any &= 15u;   // the repeated group is not evaluated twice
        if (!__any_sync(0xffffffffu, any != 0)) continue;
#pragma unroll 1
        for (int k = 0; k < 8; ++k) {
            if (!__any_sync(0xffffffffu, (any >> k) & 1u)) continue;
            const int tl = 4 * (g + (k >> 2) * NT2) + (k & 3);
            const int64_t tau = s0 + tl;                  // column inside the sub-chunk
            bool has = false;
            int best_w = 0;
            double best = 0.0;
            if (((any >> k) & 1u) && tl < n_emit) {
                const uint32_t p0 = X[tl];
                const uint32_t tabs = tabs0 + (uint32_t)tl;
                for (int j = 0; j < nw; ++j) {
                    const int w = sh.w[j];
                    if (tau + w > a.nout_left || (tabs & (uint32_t)(sh.dec[j] - 1))) continue;
                    const long long B = (long long)(uint32_t)(X[tl + w] - p0);
                    double S;
                    if (measured) {
                        const double sg = sh.den[j];
                        if (!(sg > 0.0)) continue;
                        S = __ddiv_rn(__dsub_rn((double)B, sh.wmu[j]), sg);
                    } else {
                        S = __ddiv_rn(__dsub_rn((double)B, __dmul_rn((double)w, mu)), sh.den[j]);
                    }
                    if (best_w == 0 || S > best) { best = S; best_w = w; }
                }
                has = (best_w != 0) && (best >= a.thr);
            }
            const unsigned mask = __ballot_sync(0xffffffffu, has);
            if (mask) {
                uint32_t base = 0;
                const int leader = __ffs(mask) - 1;
                if (lane == leader) base = atomicAdd(a.count, (uint32_t)__popc(mask));
                base = __shfl_sync(0xffffffffu, base, leader);
                if (has) {
                    const uint32_t slot = base + __popc(mask & ((1u << lane) - 1));
                    if (slot < a.cap) {
                        aa_candidate c;
                        c.dm_index = a.dm_base + (uint32_t)d;
                        c.t_start = (a.tau0 + (uint32_t)tau) * a.bin;
                        c.width = (uint32_t)best_w * a.bin;
                        c.snr = (float)best;
                        a.cands[slot] = c;
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Cluster kernel, second version (white-noise scaling A10, every width at every sample, boxcar sums below 2^31).
// Same layout as sps_cluster_kernel (segment + boxcar tail of one normalisation block per CTA, cluster of C CTAs
// per block, series read from HBM once), a third of the instructions and ONE cluster-wide wait instead of five:
//   pass A   thread t walks its own chunk of the segment once: exact sum and sum of squares (the block's pass 0,
//            A8) and the chunk total for the prefix sums;
//   pass B   walks it again: writes the exclusive prefix sums in place and marks (one bit per sample) the samples
//            outside the CTA's "core" interval mu' +- 2.75 sigma' (mu', sigma' = plain moments of the segment
//            alone: a guess that needs no other CTA);
//   list     the marked samples (0.6 % of white noise) are appended to a small list that every CTA of the
//            cluster receives (DSMEM stores), with the CTA's exact sums and its core interval; one cluster barrier;
//   stats    warp 0 of every CTA then holds everything the three clip passes need: a 3-sigma interval I that
//            contains every core selects all samples but the listed ones outside I, so
//            (m, S1, S2)(I) = totals - sums over {listed x not in I}: exact integers, the oracle's mu and sigma
//            bit for bit.  If an interval does not contain a core (strong interference: sigma collapses after the
//            first clip), a list is full, or a core is empty, the pass and those after it walk the whole segment
//            as sps_cluster_kernel does;
//   boxcars  that chain (three dependent rounds of interval, sums, 128-bit moments, double division and root) is
//            serial and takes one warp several microseconds, so warps 1-7 do not wait for it: they run the integer
//            pre-filter th_w + P[tau] - P[tau + w] < 0 with thresholds GUESSED from the unclipped moments
//            (mu0 - sigma0 / 20, 0.9 sigma0) and keep one bit per tau.  When the chain is done the guess is checked
//            against the true thresholds (guess <= truth for every width: the bits are then a superset of the hits;
//            otherwise the pre-filter is repeated with the truth), and the marked taus get the double-precision S/N
//            of every width, the arg-max and the threshold test with the final mu and sigma.
//            Pre-filter: two widths per 3-input OR, widths below 4 from the next 16-byte piece, eight taus per thread.
constexpr int kListTotal = 1536;      // list entries per CTA (all ranks' outliers): 6 KB

struct SharedC2 {
    SharedC c;                           // the fields the slow path and the candidate stage share with version 1
    uint64_t redA[2][NT2 / 32];          // pass A: sum, sum of squares per warp
    uint64_t part2[kMaxCluster][6];      // per rank: n_own, S1, S2, (lc | hc << 32), listed entries, flags
    uint64_t lbar[NT2 / 32];             // mbarriers of the warps' bulk loads
    uint32_t nlist;                      // entries this CTA found (may exceed its room)
    int slow_from;                       // 0: statistics done by warp 0; k: passes k..3 take the slow path
    uint32_t ths[4];                     // pre-filter thresholds of widths 1, 2, 3 (index w; "never" if the width is not searched)
    int slot[kMaxWidths];                // where width j's threshold lives: wl index, or -w for the widths below 4
    uint32_t thg[kMaxWidths];            // guessed thresholds (plain), for the check against thr_u
    int nsm, guess_ok;
};

constexpr int NTP = NT2 - 32;            // threads of the pre-filter (warps 1-7)
constexpr uint32_t kNever = 0x7FFFFFFFu;
// th - 1 as a signed number: B >= th  <=>  (th - 1) - B < 0; th above every possible B (< 2^31) -> never
__device__ __forceinline__ uint32_t enc_thr(uint32_t th) { return th == 0u ? 0xFFFFFFFFu : (th > 0x7FFFFFFFu ? kNever : th - 1u); }

// Integer pre-filter over the taus [0, 4 ngroups) of the segment by the NTP threads gid = 0 .. NTP - 1: thread gid takes
// the groups of four taus g = it * 2 NTP + gid and g + NTP of round it; bit 8 it + k of the result marks tau k of the pair.
__device__ __forceinline__ void prefilter(const uint32_t *X, const SharedC2 &s2, int gid, int ngroups, uint64_t &flo, uint32_t &fhi)
{
    const SharedC &sh = s2.c;
    const int na = sh.na, nu = sh.nu, nsm = s2.nsm;
    constexpr int GB = 4 * NTP;
    flo = 0ull;
    fhi = 0u;
    const uint32_t th1 = s2.ths[1], th2 = s2.ths[2], th3 = s2.ths[3];
    int it = 0;
    for (int g0 = 0; g0 < ngroups; g0 += 2 * NTP, ++it) {
        const int g = g0 + gid;
        if (g >= ngroups) break;
        const bool two = g + NTP < ngroups;               // else the second group repeats the first
        const uint32_t *xg = X + 4 * g;
        const int gb = two ? GB : 0;
        const uint4 pa = *reinterpret_cast<const uint4 *>(xg), pb = *reinterpret_cast<const uint4 *>(xg + gb);
        uint32_t f0 = 0, f1 = 0, f2 = 0, f3 = 0, f4 = 0, f5 = 0, f6 = 0, f7 = 0;   // sign bits collect the hits
        if (nsm) {
            // widths 1, 2, 3: P[tau + w] comes from the group itself and the next 16-byte piece
            const uint4 na4 = *reinterpret_cast<const uint4 *>(xg + 4), nb4 = *reinterpret_cast<const uint4 *>(xg + gb + 4);
            f0 |= (th1 + pa.x - pa.y) | (th2 + pa.x - pa.z); f0 |= th3 + pa.x - pa.w;
            f1 |= (th1 + pa.y - pa.z) | (th2 + pa.y - pa.w); f1 |= th3 + pa.y - na4.x;
            f2 |= (th1 + pa.z - pa.w) | (th2 + pa.z - na4.x); f2 |= th3 + pa.z - na4.y;
            f3 |= (th1 + pa.w - na4.x) | (th2 + pa.w - na4.y); f3 |= th3 + pa.w - na4.z;
            f4 |= (th1 + pb.x - pb.y) | (th2 + pb.x - pb.z); f4 |= th3 + pb.x - pb.w;
            f5 |= (th1 + pb.y - pb.z) | (th2 + pb.y - pb.w); f5 |= th3 + pb.y - nb4.x;
            f6 |= (th1 + pb.z - pb.w) | (th2 + pb.z - nb4.x); f6 |= th3 + pb.z - nb4.y;
            f7 |= (th1 + pb.w - nb4.x) | (th2 + pb.w - nb4.y); f7 |= th3 + pb.w - nb4.z;
        }
        // widths that are multiples of 4: aligned 16-byte loads, two widths per round (one 3-input OR takes both)
#pragma unroll 2
        for (int j = 0; j + 1 < na; j += 2) {
            const uint4 w0 = sh.wl[j], w1 = sh.wl[j + 1];
            const uint4 qa = *reinterpret_cast<const uint4 *>(xg + w0.x), qb = *reinterpret_cast<const uint4 *>(xg + w0.x + gb);
            const uint4 ra = *reinterpret_cast<const uint4 *>(xg + w1.x), rb = *reinterpret_cast<const uint4 *>(xg + w1.x + gb);
            const uint32_t t0 = w0.y, t1 = w1.y;
            f0 |= (t0 + pa.x - qa.x) | (t1 + pa.x - ra.x); f1 |= (t0 + pa.y - qa.y) | (t1 + pa.y - ra.y);
            f2 |= (t0 + pa.z - qa.z) | (t1 + pa.z - ra.z); f3 |= (t0 + pa.w - qa.w) | (t1 + pa.w - ra.w);
            f4 |= (t0 + pb.x - qb.x) | (t1 + pb.x - rb.x); f5 |= (t0 + pb.y - qb.y) | (t1 + pb.y - rb.y);
            f6 |= (t0 + pb.z - qb.z) | (t1 + pb.z - rb.z); f7 |= (t0 + pb.w - qb.w) | (t1 + pb.w - rb.w);
        }
        if (na & 1) {                                     // an odd count: the last one alone
            const uint4 w0 = sh.wl[na - 1];
            const uint4 qa = *reinterpret_cast<const uint4 *>(xg + w0.x), qb = *reinterpret_cast<const uint4 *>(xg + w0.x + gb);
            const uint32_t t0 = w0.y;
            f0 |= t0 + pa.x - qa.x; f1 |= t0 + pa.y - qa.y; f2 |= t0 + pa.z - qa.z; f3 |= t0 + pa.w - qa.w;
            f4 |= t0 + pb.x - qb.x; f5 |= t0 + pb.y - qb.y; f6 |= t0 + pb.z - qb.z; f7 |= t0 + pb.w - qb.w;
        }
        // the others: the aligned pieces around tau + w, shifted by w mod 4 (uniform)
#pragma unroll 1
        for (int j = na; j < na + nu; ++j) {
            const uint4 wt2 = sh.wl[j];
            const uint32_t th = wt2.y;
            const int r = (int)(wt2.x & 3u);
            const uint32_t *xq = xg + (wt2.x - (uint32_t)r);
            const uint4 q0 = *reinterpret_cast<const uint4 *>(xq), q1 = *reinterpret_cast<const uint4 *>(xq + 4),
                        q2 = *reinterpret_cast<const uint4 *>(xq + gb), q3 = *reinterpret_cast<const uint4 *>(xq + gb + 4);
            uint32_t v0, v1, v2, v3, v4, v5, v6, v7;
            if (r == 1) { v0 = q0.y; v1 = q0.z; v2 = q0.w; v3 = q1.x; v4 = q2.y; v5 = q2.z; v6 = q2.w; v7 = q3.x; }
            else if (r == 2) { v0 = q0.z; v1 = q0.w; v2 = q1.x; v3 = q1.y; v4 = q2.z; v5 = q2.w; v6 = q3.x; v7 = q3.y; }
            else { v0 = q0.w; v1 = q1.x; v2 = q1.y; v3 = q1.z; v4 = q2.w; v5 = q3.x; v6 = q3.y; v7 = q3.z; }
            f0 |= th + pa.x - v0; f1 |= th + pa.y - v1; f2 |= th + pa.z - v2; f3 |= th + pa.w - v3;
            f4 |= th + pb.x - v4; f5 |= th + pb.y - v5; f6 |= th + pb.z - v6; f7 |= th + pb.w - v7;
        }
        if ((int)((f0 | f1 | f2 | f3) | (f4 | f5 | f6 | f7)) < 0) {
            uint32_t any = (f0 >> 31) | (f1 >> 31) << 1 | (f2 >> 31) << 2 | (f3 >> 31) << 3 | (f4 >> 31) << 4 | (f5 >> 31) << 5 |
                           (f6 >> 31) << 6 | (f7 >> 31) << 7;
            if (!two) any &= 15u;                         // the repeated group is not evaluated twice
            if (it < 8) flo |= (uint64_t)any << (8 * it);
            else fhi |= any << (8 * (it - 8));
        }
    }
}
// thresholds of the pre-filter into their slots (plain threshold th of width j)
__device__ __forceinline__ void put_threshold(SharedC2 &s2, int j, uint32_t th)
{
    const int sl = s2.slot[j];
    const uint32_t e = enc_thr(th);
    if (sl < 0) {
        s2.ths[-sl] = e;
    } else {
        s2.c.wl[sl].y = e;
    }
}


__device__ __forceinline__ void st_cluster_u32(const void *local, uint32_t rank, uint32_t v)
{
    uint32_t a = (uint32_t)__cvta_generic_to_shared(local), r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(r), "r"(v) : "memory");
}
__device__ __forceinline__ uint64_t warp_sum_all(uint64_t v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ void moments_from_sums(uint64_t m, uint64_t S1, unsigned __int128 S2, double &mu, double &sigma)
{
    const unsigned __int128 N = (unsigned __int128)m * S2 - (unsigned __int128)S1 * S1;
    const double dm = __ull2double_rn(m);
    mu = __ddiv_rn(__ull2double_rn(S1), dm);
    sigma = __dsqrt_rn(__ddiv_rn(u128_to_double(N), __dmul_rn(dm, dm)));
}

__global__ void __launch_bounds__(NT2) sps_cluster2_kernel(const SpsArgs a, const __grid_constant__ WidthTable wt, const int C, const int seg)
{
    extern __shared__ __align__(16) uint8_t dyn[];
    uint32_t *X = reinterpret_cast<uint32_t *>(dyn);     // segment + tail; later its exclusive prefix sums
    const int total = seg + a.wmax - 1 + 8;              // slots the boxcar loop may read
    uint32_t *LST = X + total;                           // [C][lreg] listed samples of every rank
    const int lreg = kListTotal / C;
    __shared__ SharedC2 s2;
    SharedC &sh = s2.c;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d = blockIdx.y;
    const uint32_t rank = C > 1 ? cluster_rank() : 0u;
    const int64_t blk = blockIdx.x / C;
    if (tid < kMaxWidths) { sh.w[tid] = wt.w[tid]; sh.dec[tid] = 1; }
    const int64_t b0 = blk * a.block_len;
    int64_t b1 = b0 + a.block_len;
    if (b1 > a.nout_left) b1 = a.nout_left;
    if (b0 >= b1 || b0 >= a.nemit) return;               // uniform over the cluster
    const int64_t n_k = b1 - b0;
    const uint32_t *row = a.D + (size_t)d * a.pitch;
    const int64_t s0 = b0 + (int64_t)rank * seg;         // first column of this CTA's segment
    const int64_t navail = a.ncols < a.nout_left ? (int64_t)a.ncols : a.nout_left;
    const int halo = a.wmax - 1;
    int n_in = (int)((navail - s0 > seg + halo) ? seg + halo : (navail - s0 < 0 ? 0 : navail - s0));   // columns held
    int n_own = (int)((b1 - s0 > seg) ? seg : (b1 - s0 < 0 ? 0 : b1 - s0));                             // ... of the block
    if (n_own > n_in) n_own = n_in;

    // ---- load: one bulk copy per warp (the part its threads walk), each onto its own mbarrier, so that a warp starts
    //      as soon as its own part has landed -------------------------------------------------------------------------
    int chunk = (n_in + 1 + NT2 - 1) / NT2;               // slots 0 .. n_in over the threads
    chunk |= 1;                                           // odd stride: conflict-free
    const int i0 = tid * chunk;
    const int c_in = min(max(n_in - i0, 0), chunk);       // elements of the thread's chunk that hold data
    const int c_own = min(max(n_own - i0, 0), chunk);     // ... that belong to the block (the rest is the boxcar tail)
    if (tid == 0) {
#pragma unroll
        for (int w = 0; w < NT2 / 32; ++w)
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((uint32_t)__cvta_generic_to_shared(&s2.lbar[w])));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        s2.nlist = 0;
        s2.slow_from = 0;
    }
    if (tid == 32) {
        // width classes of the pre-filter: below 4 (from the neighbouring piece), multiples of 4 (aligned loads, taken two
        // at a time), the rest
        int n = 0, nsm = 0;
        s2.ths[0] = s2.ths[1] = s2.ths[2] = s2.ths[3] = kNever;
        for (int j = 0; j < a.nwidths; ++j)
            if (wt.w[j] < 4) { s2.slot[j] = -wt.w[j]; ++nsm; }
        s2.nsm = nsm;
        for (int j = 0; j < a.nwidths; ++j)
            if ((wt.w[j] & 3) == 0) { s2.slot[j] = n; sh.wl[n++] = make_uint4((uint32_t)wt.w[j], kNever, 1u, 0u); }
        sh.na = n;
        int q = n;
        for (int j = 0; j < a.nwidths; ++j)
            if (wt.w[j] > 4 && (wt.w[j] & 3) != 0) { s2.slot[j] = q; sh.wl[q++] = make_uint4((uint32_t)wt.w[j], kNever, 1u, 0u); }
        sh.nu = q - n;
    }
    __syncthreads();
    // every CTA of the cluster must be running before its shared memory is written: arrive now, wait before the first remote store
    if (C > 1) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    {
        const int n4 = (n_in + 3) / 4 * 4;                // whole 16-byte pieces; the row pitch leaves room
        const int e0 = warp * 32 * chunk, e1 = min(e0 + 32 * chunk, n4);
        if (e1 > e0) {
            const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&s2.lbar[warp]);
            if (lane == 0) {
                const uint32_t bytes = (uint32_t)(e1 - e0) * 4u;
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                                 (uint32_t)__cvta_generic_to_shared(X + e0)),
                             "l"(row + s0 + e0), "r"(bytes), "r"(bar)
                             : "memory");
            }
            uint32_t ok = 0;
            while (!ok)
                asm volatile(
                    "{\n\t.reg .pred p;\n\t"
                    "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\t"
                    "selp.u32 %0, 1, 0, p;\n\t}"
                    : "=r"(ok)
                    : "r"(bar)
                    : "memory");
        }
    }

    // ---- pass A: the thread's chunk [i0, i0 + chunk): exact sums over the block's part, total over all of it ----
    uint32_t *xp = X + i0;
    uint32_t run = 0;
    uint64_t S1 = 0, S2 = 0;
    {
        const bool fast32 = (uint64_t)a.maxval * (uint64_t)chunk < 0x100000000ull;   // the chunk's sum fits 32 bits
        if (fast32) {
#pragma unroll 8
            for (int k = 0; k < c_own; ++k) {
                const uint32_t x = xp[k];
                run += x;
                S2 += (uint64_t)x * x;
            }
            S1 = run;
        } else {
#pragma unroll 4
            for (int k = 0; k < c_own; ++k) {
                const uint32_t x = xp[k];
                S1 += x;
                S2 += (uint64_t)x * x;
            }
            run = (uint32_t)S1;
        }
#pragma unroll 4
        for (int k = c_own; k < c_in; ++k) run += xp[k];
    }
    uint32_t incl = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    S1 = warp_sum_all(S1);
    S2 = warp_sum_all(S2);
    if (lane == 31) sh.warp_tot[warp] = incl;
    if (lane == 0) { s2.redA[0][warp] = S1; s2.redA[1][warp] = S2; }
    __syncthreads();
    // every thread: the segment's sums, its own exclusive prefix, and the core interval from the segment's plain moments
    uint32_t pre = incl - run;
    S1 = 0; S2 = 0;
#pragma unroll
    for (int w = 0; w < NT2 / 32; ++w) {
        if (w < warp) pre += sh.warp_tot[w];
        S1 += s2.redA[0][w];
        S2 += s2.redA[1][w];
    }
    uint32_t lc = 1u, hc = 0u;                            // empty core: everything is listed (-> slow path)
    if (n_own > 0) {
        const double kcore = 2.75;                        // 0.6 % of white noise outside: about 100 listed samples per segment
        const double inv = 1.0 / (double)n_own, mean = (double)S1 * inv;
        double var = (double)S2 * inv - mean * mean;      // a guess: need not be exact
        if (!(var > 0.0)) var = 0.0;
        const double sd = (double)sqrtf((float)var);
        double l = ceil(mean - kcore * sd), h = floor(mean + kcore * sd);
        if (l < 0.0) l = 0.0;
        if (h > 4294967295.0) h = 4294967295.0;
        if (l <= h) { lc = (uint32_t)l; hc = (uint32_t)h; }
    }
    const uint32_t cspan = hc - lc;                       // empty core: 0xFFFFFFFF, no sample passes (x - lc) <= ... see below
    const bool core_empty = lc > hc;

    // ---- pass B: exclusive prefix sums in place; one bit per sample of the block outside the core ---------------
    uint32_t mk[3] = {0u, 0u, 0u};
#pragma unroll
    for (int wd = 0; wd < 3; ++wd) {
        const int k0 = 32 * wd;
        const int kend = min(c_own - k0, 32);
        uint32_t m = 0, bit = 1u;
#pragma unroll 8
        for (int k = 0; k < kend; ++k) {
            const uint32_t x = xp[k0 + k];
            xp[k0 + k] = pre;
            pre += x;
            if ((x - lc) > cspan) m |= bit;
            bit += bit;
        }
        mk[wd] = m;
    }
    if (core_empty) {                                     // (x - 1) > 0xFFFFFFFF never holds: mark everything instead
#pragma unroll
        for (int wd = 0; wd < 3; ++wd) {
            const int kend = min(c_own - 32 * wd, 32);
            mk[wd] = kend <= 0 ? 0u : (kend >= 32 ? 0xFFFFFFFFu : ((1u << kend) - 1u));
        }
    }
    for (int k = c_own; k < c_in; ++k) {                  // the boxcar tail
        const uint32_t x = xp[k];
        xp[k] = pre;
        pre += x;
    }
    if (c_in > 0 && i0 + c_in == n_in) xp[c_in] = pre;    // slot n_in: the total
    if (n_in == 0 && tid == 0) X[0] = 0u;
    if (C > 1) asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");   // all CTAs run: remote stores may begin
    __syncthreads();
    {
        const uint32_t last = X[n_in];
        for (int i = n_in + 1 + tid; i < total; i += NT2) X[i] = last;
    }
    // the marked samples (x = P[i + 1] - P[i]) go to every CTA's copy of this rank's list
#pragma unroll
    for (int wd = 0; wd < 3; ++wd) {
        uint32_t m = mk[wd];
        while (m) {
            const int k = __ffs(m) - 1;
            m &= m - 1u;
            const int i = i0 + 32 * wd + k;
            const uint32_t x = X[i + 1] - X[i];
            const uint32_t pos = atomicAdd(&s2.nlist, 1u);
            if (pos < (uint32_t)lreg) {
                uint32_t *slot = LST + rank * lreg + pos;
                if (C > 1) {
                    for (int r = 0; r < C; ++r) st_cluster_u32(slot, (uint32_t)r, x);
                } else {
                    *slot = x;
                }
            }
        }
    }
    __syncthreads();
    if (tid == 0) {
        const uint32_t found = s2.nlist;
        const uint64_t flags = (found > (uint32_t)lreg || (core_empty && n_own > 0)) ? 1ull : 0ull;
        const uint64_t v[6] = {(uint64_t)n_own, S1, S2, (uint64_t)lc | ((uint64_t)hc << 32),
                               (uint64_t)(found > (uint32_t)lreg ? (uint32_t)lreg : found), flags};
        for (int r = 0; r < C; ++r)
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                if (C > 1) st_cluster_u64(&s2.part2[rank][q], (uint32_t)r, v[q]);
                else s2.part2[0][q] = v[q];
            }
    }
    if (C > 1) cluster_sync_all(); else __syncthreads();

    // ---- warp 0: statistics (A8) from the totals and the lists, the same integers in every CTA;
    //      warps 1-7 meanwhile: pre-filter with guessed thresholds ------------------------------------------------------
    const int n_emit = n_own;                             // taus [0, n_emit) of this segment may emit (blocks tile the sub-chunk)
    const int ngroups = (n_emit + 3) / 4;
    uint64_t flo = 0ull;
    uint32_t fhi = 0u;
    if (warp == 0) {
        uint64_t n = 0, T1 = 0;
        unsigned __int128 T2 = 0;
        bool listed_ok = true;
        uint32_t lcmin = 0xFFFFFFFFu, hcmax = 0u;         // an interval contains every core iff it contains [lcmin, hcmax]
        for (int r = 0; r < C; ++r) {
            n += s2.part2[r][0]; T1 += s2.part2[r][1]; T2 += s2.part2[r][2];
            if (s2.part2[r][5]) listed_ok = false;
            if (s2.part2[r][0]) {
                const uint64_t ch = s2.part2[r][3];
                lcmin = min(lcmin, (uint32_t)ch);
                hcmax = max(hcmax, (uint32_t)(ch >> 32));
            }
        }
        // the lists: 32 / C lanes walk the list of each rank
        const int lpr = 32 / C, lr = lane / lpr, l0 = lane % lpr;
        const int cnt = (int)s2.part2[lr][4];
        const uint32_t *L = LST + lr * lreg;
        double mu = 0.0, sigma = 0.0;
        int slow = 0;
        if (n) {
            moments_from_sums(n, T1, T2, mu, sigma);      // pass 0: every sample
            for (int pass = 1; pass < 4; ++pass) {
                uint32_t lo = 0, hi = 0;
                if (!clip_interval(mu, __dmul_rn(3.0, sigma), lo, hi)) break;   // nothing selected: keep the last values
                if (!(listed_ok && lo <= lcmin && hi >= hcmax)) { slow = pass; break; }
                const uint32_t span = hi - lo;
                uint64_t mr = 0, R1 = 0, R2 = 0, carry = 0;   // the listed samples the interval rejects
#pragma unroll 1
                for (int e = l0; e < cnt; e += lpr) {
                    const uint32_t x = L[e];
                    const bool rej = (x - lo) > span;
                    const uint32_t xr = rej ? x : 0u;
                    mr += rej ? 1u : 0u;
                    R1 += xr;
                    const uint64_t sq = (uint64_t)xr * xr;
                    R2 += sq;
                    carry += R2 < sq;
                }
                // one butterfly for the small numbers (count and carries: below 2^16 each), one for each 64-bit sum
                uint64_t mc = warp_sum_all(mr | (carry << 32));
                R1 = warp_sum_all(R1);
                const uint64_t r2lo = warp_sum_all(R2 & 0xFFFFFFFFull), r2hi = warp_sum_all(R2 >> 32);
                mr = mc & 0xFFFFFFFFull;
                carry = mc >> 32;
                const unsigned __int128 R2w = (unsigned __int128)r2lo + ((unsigned __int128)r2hi << 32) + ((unsigned __int128)carry << 64);
                const uint64_t m = n - mr;
                if (!m) break;
                moments_from_sums(m, T1 - R1, T2 - R2w, mu, sigma);
            }
        }
        if (lane == 0) { sh.mu = mu; sh.sigma = sigma; sh.m = n; s2.slow_from = slow; }
    } else {
        const int gid = tid - 32;
        if (gid < a.nwidths) {
            // the unclipped moments, roughly (nothing exact depends on them)
            uint64_t n = 0, T1 = 0, T2 = 0;
            for (int r = 0; r < C; ++r) { n += s2.part2[r][0]; T1 += s2.part2[r][1]; T2 += s2.part2[r][2]; }
            const double nn = (double)n, mean = (double)T1 / nn;
            double var = (double)T2 / nn - mean * mean;
            if (!(var > 0.0)) var = 0.0;
            const double sd = sqrt(var), w = (double)sh.w[gid];
            const double bt = floor(w * (mean - 0.05 * sd) + a.thr * (0.9 * sd) * sqrt(w)) - 1.0;
            const uint32_t th = bt <= 0.0 ? 0u : (bt >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)bt);
            s2.thg[gid] = th;
            put_threshold(s2, gid, th);
        }
        asm volatile("bar.sync 1, %0;" ::"n"(NTP) : "memory");
        if (n_emit > 0) prefilter(X, s2, gid, ngroups, flo, fhi);
    }
    __syncthreads();
    double mu = sh.mu, sigma = sh.sigma;
    const int slow_from = s2.slow_from;
    __syncthreads();
    if (slow_from) {
        // rare: the remaining passes over the whole segment, x = P[i + 1] - P[i], as version 1 does them
        int turn = 0;
        for (int pass = slow_from; pass < 4; ++pass) {
            uint32_t lo = 0u, span = 0u;
            bool run2 = true;
            if (tid == 0) {
                uint32_t l = 0, h = 0;
                sh.empty = clip_interval(mu, __dmul_rn(3.0, sigma), l, h) ? 0 : 1;
                sh.lo = l;
                sh.hi = h;
            }
            __syncthreads();
            run2 = !sh.empty;
            lo = sh.lo;
            span = sh.hi - lo;
            uint64_t m = 0, Q1 = 0, Q2 = 0, carry = 0;
            if (run2) {
                for (int i = tid; i < n_own; i += NT2) {
                    const uint32_t x = X[i + 1] - X[i];
                    if ((x - lo) <= span) {
                        m += 1;
                        Q1 += x;
                        const uint64_t sq = (uint64_t)x * x;
                        Q2 += sq;
                        carry += Q2 < sq;
                    }
                }
            }
            if (!cluster_moments(sh, C, rank, turn, m, Q1, Q2, carry, mu, sigma)) break;
        }
    }
    if (!(sigma > 0.0) || n_k < 32) return;

    // ---- per-width constants with the final mu, sigma; was the guess below the truth for every width? ---------------
    if (tid < a.nwidths) {
        const double w = (double)sh.w[tid];
        const double den = __dmul_rn(sigma, __dsqrt_rn(w));
        sh.den[tid] = den;
        // B >= floor(w mu + thr sigma sqrt w) - 1 is necessary for S >= thr; clamped to the 32-bit sums
        const long long bt = __double2ll_rd(w * mu + a.thr * den) - 1;
        sh.thr_u[tid] = bt <= 0 ? 0u : (bt >= 0xFFFFFFFFll ? 0xFFFFFFFFu : (uint32_t)bt);
    }
    __syncthreads();
    if (tid == 0) {
        int ok = 1;
        for (int j = 0; j < a.nwidths; ++j) ok &= s2.thg[j] <= sh.thr_u[j];
        s2.guess_ok = ok;
        if (!ok)
            for (int j = 0; j < a.nwidths; ++j) put_threshold(s2, j, sh.thr_u[j]);
    }
    __syncthreads();
    if (n_emit <= 0) return;
    if (!s2.guess_ok && warp > 0) prefilter(X, s2, tid - 32, ngroups, flo, fhi);   // rare: sigma fell by more than a tenth

    // ---- the marked taus: S/N of every width in double, arg-max, threshold, warp-aggregated append ---------------------
    const int nw = a.nwidths, gid = tid - 32;
    const int niter = (ngroups + 2 * NTP - 1) / (2 * NTP);
    if (warp == 0) return;                                // holds no marks
    for (int it = 0; it < niter; ++it) {
        const uint32_t any = it < 8 ? (uint32_t)(flo >> (8 * it)) & 0xFFu : (fhi >> (8 * (it - 8))) & 0xFFu;
        if (!__any_sync(0xffffffffu, any != 0)) continue;
        const int g = it * 2 * NTP + gid;
#pragma unroll 1
        for (int k = 0; k < 8; ++k) {
            if (!__any_sync(0xffffffffu, (any >> k) & 1u)) continue;
            const int tl = 4 * (g + (k >> 2) * NTP) + (k & 3);
            const int64_t tau = s0 + tl;                  // column inside the sub-chunk
            bool has = false;
            int best_w = 0;
            double best = 0.0;
            if (((any >> k) & 1u) && tl < n_emit) {
                const uint32_t p0 = X[tl];
                for (int j = 0; j < nw; ++j) {
                    const int w = sh.w[j];
                    if (tau + w > a.nout_left) continue;
                    const long long B = (long long)(uint32_t)(X[tl + w] - p0);
                    const double S = __ddiv_rn(__dsub_rn((double)B, __dmul_rn((double)w, mu)), sh.den[j]);
                    if (best_w == 0 || S > best) { best = S; best_w = w; }
                }
                has = (best_w != 0) && (best >= a.thr);
            }
            const unsigned mask = __ballot_sync(0xffffffffu, has);
            if (mask) {
                uint32_t base = 0;
                const int leader = __ffs(mask) - 1;
                if (lane == leader) base = atomicAdd(a.count, (uint32_t)__popc(mask));
                base = __shfl_sync(0xffffffffu, base, leader);
                if (has) {
                    const uint32_t slot = base + __popc(mask & ((1u << lane) - 1));
                    if (slot < a.cap) {
                        aa_candidate c;
                        c.dm_index = a.dm_base + (uint32_t)d;
                        c.t_start = (a.tau0 + (uint32_t)tau) * a.bin;
                        c.width = (uint32_t)best_w * a.bin;
                        c.snr = (float)best;
                        a.cands[slot] = c;
                    }
                }
            }
        }
    }
}

// cluster size and segment length of the cluster variant; false: use the generic kernel
bool sps_cluster_shape(const SpsArgs &a, bool wide, int &C, int &seg)
{
    if (wide || a.block_len % 4 != 0 || a.pitch % 4 != 0 || (reinterpret_cast<uintptr_t>(a.D) & 15) != 0) return false;
    if (a.wmax > 4096) return false;
    for (C = 1; C <= kMaxCluster; C *= 2) {
        if (a.block_len % (4 * C)) return false;
        seg = a.block_len / C;
        if (seg <= kSegMax) return true;
    }
    return false;
}

size_t sps_cluster_smem(const SpsArgs &a, int seg)
{
    return (size_t)(seg + a.wmax - 1 + 8) * 4;
}

size_t sps_cluster2_smem(const SpsArgs &a, int seg)
{
    return sps_cluster_smem(a, seg) + (size_t)kListTotal * 4;
}

size_t sps_smem(const SpsArgs &a, bool wide)
{
    return (size_t)(TT + a.wmax + 8) * (wide ? 8 : 4);
}

}  // namespace

cudaError_t sps_configure()
{
    cudaError_t e = cudaFuncSetAttribute(sps_kernel<uint32_t>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         160 * 1024);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(sps_kernel<uint64_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(sps_kernel<uint64_t, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(sps_kernel<uint32_t, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(sps_cluster2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(sps_cluster_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(sps_cluster_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
}

cudaError_t launch_sps(const SpsArgs &a, const WidthTable &wt, bool wide, bool small31, bool big, bool force_v1, cudaStream_t st)
{
    if (a.nemit <= 0 || a.ndms <= 0) return cudaSuccess;
    const unsigned nblk = (unsigned)((a.nemit + a.block_len - 1) / a.block_len);
    int C = 1, seg = 0;
    if (!big && sps_cluster_shape(a, wide, C, seg)) {
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(nblk * (unsigned)C, (unsigned)a.ndms);
        cfg.blockDim = dim3(NT2);
        cfg.dynamicSmemBytes = sps_cluster_smem(a, seg);
        cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)C;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        // version 2 serves the search BASELINE.json states: white-noise scaling, every width at every sample
        bool plain = small31 && a.sigma_mode == 0 && !force_v1;
        for (int j = 0; j < a.nwidths; ++j) plain = plain && wt.dec[j] == 1;
        if (plain) {
            cfg.dynamicSmemBytes = sps_cluster2_smem(a, seg);
            return cudaLaunchKernelEx(&cfg, sps_cluster2_kernel, a, wt, C, seg);
        }
        return small31 ? cudaLaunchKernelEx(&cfg, sps_cluster_kernel<true>, a, wt, C, seg)
                       : cudaLaunchKernelEx(&cfg, sps_cluster_kernel<false>, a, wt, C, seg);
    }
    dim3 grid(nblk, (unsigned)a.ndms);
    if (wide && big)
        sps_kernel<uint64_t, true><<<grid, NT, sps_smem(a, true), st>>>(a, wt);
    else if (wide)
        sps_kernel<uint64_t><<<grid, NT, sps_smem(a, true), st>>>(a, wt);
    else if (big)
        sps_kernel<uint32_t, true><<<grid, NT, sps_smem(a, false), st>>>(a, wt);
    else
        sps_kernel<uint32_t><<<grid, NT, sps_smem(a, false), st>>>(a, wt);
    return cudaGetLastError();
}

}  // namespace aa
