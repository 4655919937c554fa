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
    uint64_t red[3][NT / 32];
    double mu, sigma;
    uint64_t m;
    long long bthr[kMaxWidths];
    double den[kMaxWidths];
    unsigned long long warp_tot[NT / 32];
    int w[kMaxWidths];        // widths (a dynamically indexed kernel parameter would go through the ADU pipe)
};

template <typename ACC>
__global__ void __launch_bounds__(NT) sps_kernel(const SpsArgs a, const WidthTable wt)
{
    extern __shared__ __align__(16) uint8_t dyn[];
    ACC *P = reinterpret_cast<ACC *>(dyn);          // exclusive prefix sums of the current tile
    __shared__ Shared sh;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d = blockIdx.y;
    if (tid < kMaxWidths) sh.w[tid] = wt.w[tid];
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
        uint64_t m = 0, S1 = 0, S2 = 0;
        for (int64_t i = b0 + tid; i < b1; i += NT) {
            const uint32_t x = row[i];
            const bool sel = (pass == 0) || (fabs(__dsub_rn((double)x, mu)) <= lim);
            if (sel) {
                m += 1;
                S1 += x;
                S2 += (uint64_t)x * x;
            }
        }
        m = warp_sum(m); S1 = warp_sum(S1); S2 = warp_sum(S2);
        if (lane == 0) { sh.red[0][warp] = m; sh.red[1][warp] = S1; sh.red[2][warp] = S2; }
        __syncthreads();
        if (tid == 0) {
            m = S1 = S2 = 0;
            for (int w = 0; w < NT / 32; ++w) { m += sh.red[0][w]; S1 += sh.red[1][w]; S2 += sh.red[2][w]; }
            sh.m = m;
            if (m) {
                const unsigned __int128 N = (unsigned __int128)m * S2 - (unsigned __int128)S1 * S1;
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

    // ---- 2. per-width constants ---------------------------------------------------------
    if (tid < a.nwidths) {
        const double w = (double)sh.w[tid];
        const double den = __dmul_rn(sigma, __dsqrt_rn(w));
        sh.den[tid] = den;
        sh.bthr[tid] = __double2ll_rd(w * mu + a.thr * den) - 1;
    }
    __syncthreads();

    const int64_t e = b1 < a.nemit ? b1 : (int64_t)a.nemit;     // taus [b0, e) may emit
    const int64_t navail = a.ncols < a.nout_left ? (int64_t)a.ncols : a.nout_left;
    const int halo = a.wmax - 1;
    const int ept = (TT + halo + 1 + NT - 1) / NT;              // scan slots per thread (covers P[0..TT+halo])

    for (int64_t ts = b0; ts < e; ts += TT) {
        int64_t n_in = navail - ts;
        if (n_in > TT + halo) n_in = TT + halo;
        // block-wide exclusive prefix sum of row[ts .. ts+n_in) into P[0 .. n_in]
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
                for (int j = 0; j < a.nwidths; ++j) {
                    const int w = sh.w[j];
                    if (tau + w <= a.nout_left) {
                        const long long B = (long long)(ACC)(P[tl + w] - p0);
                        any |= (B >= sh.bthr[j]);
                    }
                }
                if (any) {
                    for (int j = 0; j < a.nwidths; ++j) {
                        const int w = sh.w[j];
                        if (tau + w > a.nout_left) continue;
                        const long long B = (long long)(ACC)(P[tl + w] - p0);
                        const double num = __dsub_rn((double)B, __dmul_rn((double)w, mu));
                        const double S = __ddiv_rn(num, sh.den[j]);
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
    return cudaFuncSetAttribute(sps_kernel<uint64_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
}

cudaError_t launch_sps(const SpsArgs &a, const WidthTable &wt, bool wide, cudaStream_t st)
{
    if (a.nemit <= 0 || a.ndms <= 0) return cudaSuccess;
    const unsigned nblk = (unsigned)((a.nemit + a.block_len - 1) / a.block_len);
    dim3 grid(nblk, (unsigned)a.ndms);
    if (wide)
        sps_kernel<uint64_t><<<grid, NT, sps_smem(a, true), st>>>(a, wt);
    else
        sps_kernel<uint32_t><<<grid, NT, sps_smem(a, false), st>>>(a, wt);
    return cudaGetLastError();
}

}  // namespace aa
