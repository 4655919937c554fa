// Brute-force incoherent dedispersion with exact sharing of partial sums between DM trials
// (BASELINE.json north_star):  D[d][tau] = sum_c y[c][tau + delta(c,d)].
//
// The plain kernels (kernels_dedisp.cu) spend one shared-memory byte and one issue slot per
// (channel, trial, sample) add and sit on the shared-memory pipe.  Here the channels are taken in
// groups of kSpG = 4.  Inside a block of 64 consecutive trials the group's rounded delays,
// relative to its first channel, form only ~4 distinct vectors (sp_tables.cu); the CTA sums the
// 4 channels once per vector into a row of 16-bit sums ("pattern row") and each trial then adds
// one row sample per group: 2 B of LDS and one add per 4 channel samples.  Same integers, same sums.
//
// CTA = NT threads = 64 trials x TB samples.  Per stage (one group of 4 channels):
//   1. cp.async.bulk (TMA 1-D, mbarrier complete_tx) brings the 4 channel windows and a record
//      (two stages ahead of its use); three staging buffers, issued two stages ahead.
//   2. build: a thread owns 8 consecutive row samples (+1 for the odd-aligned copy) of one pattern
//      and sums the 4 channels with IDP.2A (dp2a: two byte adds into two 15-bit lanes of one
//      register, FMA pipe).  Rows are stored twice, as (s[2j], s[2j+1]) and (s[2j+1], s[2j+2])
//      16-bit pairs, so that any integer offset is one aligned 32-bit load.
//   3. accumulate: a warp owns 64/NW trials, a lane TB/64 words of 2 samples; acc16 += row word
//      (SWAR, two 16-bit sums per register).  There is no CTA-wide barrier in the loop: a warp
//      builds its share of rows(s+1), arrives on that buffer's mbarrier and accumulates rows(s) once
//      all warps have arrived for it; three pattern-row buffers let warps drift apart so that the
//      ALU-heavy build of some overlaps the LDS-bound accumulate of others.
//   4. every sp_flush groups (64 for uint8: 64*4*255 < 2^16) the 16-bit lanes are added into the
//      uint32 output tile in global memory (L2 resident, owned by this thread) and cleared.
// No tensor cores: a gather-add, not a dense contraction.
#include "aa_internal.h"

namespace aa {

namespace {

constexpr int G = kSpG;
constexpr int DB = kSpDB;
constexpr int REC = (int)sizeof(SpRecord);
constexpr int NBUF = 3;                // pattern-row and staging buffers
constexpr int NREC = 8;                // record ring: stage s uses s, s+1, s+3 while s+5 is being fetched

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "SP_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra SP_DONE;\n\t"
        "bra SP_WAIT;\n\t"
        "SP_DONE:\n\t}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// Adds nine consecutive samples of one channel into five words of two 15-bit lanes: dp2a multiplies
// byte 0/2 of the window word by 1 and byte 1/3 by 2^15 (IDP.2A, FMA pipe).  `base` points at this
// thread's chunk (8 * chunk bytes into the staging buffer); p is the record's window word: bits
// 0-15 the 8-byte-aligned load offset, bits 16-21 eight times the byte shift 0..7 (warp-uniform).
__device__ __forceinline__ void add_window(uint32_t (&acc)[5], const uint8_t *base, uint32_t p)
{
    const uint8_t *q = base + (p & 0xFFFFu);
    const uint2 v0 = *reinterpret_cast<const uint2 *>(q);
    const uint2 v1 = *reinterpret_cast<const uint2 *>(q + 8);
    const bool up = (p & 0x200000u) != 0;              // shift >= 4 bytes: start one word later
    const uint32_t w0 = up ? v0.y : v0.x, w1 = up ? v1.x : v0.y, w2 = up ? v1.y : v1.x;
    const uint32_t s = p >> 16;                        // funnel shifts take the amount modulo 32
    const uint32_t x0 = __funnelshift_r(w0, w1, s), x1 = __funnelshift_r(w1, w2, s), x2 = __funnelshift_r(w2, 0u, s);
    constexpr uint32_t M = 0x80000001u;
    asm("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[0]) : "r"(M), "r"(x0));
    asm("dp2a.hi.u32.u32 %0, %1, %2, %0;" : "+r"(acc[1]) : "r"(M), "r"(x0));
    asm("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[2]) : "r"(M), "r"(x1));
    asm("dp2a.hi.u32.u32 %0, %1, %2, %0;" : "+r"(acc[3]) : "r"(M), "r"(x1));
    // sample 8 goes to lane 0 of word 4; lane 1 (sample 9) is never used
    asm("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[4]) : "r"(M), "r"(x2));
}

template <int NT, int TB>
__global__ void __launch_bounds__(NT, NT == 512 ? 1 : 2) dedisp_sp_kernel(const DedispArgs a)
{
    constexpr int NW = NT / 32;
    constexpr int DPW = DB / NW;           // trials per warp
    constexpr int NP = TB / 64;            // 2-sample words per lane
    static_assert(DPW % 4 == 0, "trial offsets are fetched four at a time");

    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t ROWS = (uint32_t)a.sp_rows;
    const uint32_t raw_bytes = G * ROWS;
    const uint32_t pbytes = (uint32_t)a.sp_pbytes;
    uint8_t *P0 = smem;                                     // [NBUF] pattern rows: [row][E|O][rowwords] uint32
    uint8_t *raw0 = P0 + NBUF * pbytes;                     // [NBUF][G][ROWS] staged channel windows
    uint8_t *rec0 = raw0 + NBUF * raw_bytes;                // [NREC][REC]
    uint64_t *rawbar = reinterpret_cast<uint64_t *>(rec0 + NREC * REC);   // [NBUF] rows(q) + record(q+2) landed
    uint64_t *full = rawbar + NBUF;                         // [NBUF] every warp has built its part of rows(q)
    uint64_t *setup = full + NBUF;                          // records 0 and 1

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d0 = blockIdx.x * DB;
    const int64_t t0 = (int64_t)blockIdx.y * TB;
    const int nstages = (a.nchans + G - 1) / G;
    const uint8_t *in = static_cast<const uint8_t *>(a.in) + a.col0 + t0;
    const uint8_t *recs = static_cast<const uint8_t *>(a.sp_tab) + (size_t)blockIdx.x * nstages * REC;

    if (tid == 0) {
#pragma unroll
        for (int j = 0; j < NBUF; ++j) {
            mbar_init(&rawbar[j], 1);
            mbar_init(&full[j], NW);
        }
        mbar_init(setup, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto record = [&](int q) { return reinterpret_cast<const SpRecord *>(rec0 + (q % NREC) * REC); };

    // thread 0: load group q = the four channel windows of stage q + the record of stage q+2.
    // Record q must have landed; raw slot q % NBUF and record slot (q+2) % NREC must be free.
    auto issue = [&](int q) {
        const SpRecord *R = record(q);
        const bool rec = q + 2 < nstages;
        uint32_t bytes = rec ? REC : 0;
#pragma unroll
        for (int i = 0; i < G; ++i) bytes += R->rbytes[i];
        uint64_t *bar = &rawbar[q % NBUF];
        mbar_expect_tx(bar, bytes);
        if (rec) bulk_g2s(rec0 + ((q + 2) % NREC) * REC, recs + (size_t)(q + 2) * REC, REC, bar);
        uint8_t *dst = raw0 + (q % NBUF) * raw_bytes;
#pragma unroll
        for (int i = 0; i < G; ++i)
            bulk_g2s(dst + i * ROWS, in + (size_t)(q * G + i) * a.pitch_in + R->rbase[i], R->rbytes[i], bar);
    };

    // pattern rows of stage q: warp-sized items (pattern, batch of 32 chunks) dealt round-robin, the
    // first warp rotating with q so that no warp always gets the extra item
    auto build = [&](int q) {
        const SpRecord *R = record(q);
        const uint32_t nchunk = R->nchunk, nbatch = R->nbatch, inv = R->inv;
        const uint32_t nitems = R->npat * nbatch, rowwords = nchunk * 4u;
        const uint8_t *raw = raw0 + (q % NBUF) * raw_bytes + lane * 8;
        uint32_t *P = reinterpret_cast<uint32_t *>(P0 + (q % NBUF) * pbytes) + lane * 4;
        for (uint32_t wi = (uint32_t)(warp + 5 * q) % NW; wi < nitems; wi += NW) {
            const uint32_t k = nbatch == 1 ? wi : (wi * inv) >> 16;
            const uint32_t b32 = (wi - k * nbatch) * 32u;
            if (b32 + lane < nchunk) {
                const uint4 wv = *reinterpret_cast<const uint4 *>(R->win[k]);
                const uint8_t *rawc = raw + b32 * 8;
                uint32_t acc[5] = {0, 0, 0, 0, 0};
                add_window(acc, rawc, wv.x);
                add_window(acc, rawc, wv.y);
                add_window(acc, rawc, wv.z);
                add_window(acc, rawc, wv.w);
                // 15-bit lanes -> 16-bit lanes: w + (w & ~0x7FFF) moves lane 1 up by one bit
                uint32_t c[5];
#pragma unroll
                for (int j = 0; j < 5; ++j) c[j] = acc[j] + (acc[j] & 0xFFFF8000u);
                uint32_t *dst = P + (size_t)(k * 2) * rowwords + b32 * 4;
                *reinterpret_cast<uint4 *>(dst) = make_uint4(c[0], c[1], c[2], c[3]);
                *reinterpret_cast<uint4 *>(dst + rowwords) =
                    make_uint4(__byte_perm(c[0], c[1], 0x5432), __byte_perm(c[1], c[2], 0x5432),
                               __byte_perm(c[2], c[3], 0x5432), __byte_perm(c[3], c[4], 0x5432));
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&full[q % NBUF]);
    };

    uint32_t acc16[DPW][NP];
#pragma unroll
    for (int k = 0; k < DPW; ++k)
#pragma unroll
        for (int i = 0; i < NP; ++i) acc16[k][i] = 0;

    // adds the 16-bit lanes into the uint32 output tile (first time: plain store) and clears them
    auto flush = [&](bool first) {
#pragma unroll
        for (int k = 0; k < DPW; ++k) {
            const int d = d0 + warp * DPW + k;
            uint32_t *orow = a.out + (size_t)d * a.pitch_out;
#pragma unroll
            for (int i = 0; i < NP; ++i) {
                const int64_t t = t0 + 2 * (lane + 32 * i);
                const uint32_t lo = acc16[k][i] & 0xFFFFu, hi = acc16[k][i] >> 16;
                acc16[k][i] = 0;
                if (d >= a.ndms) continue;
                if (t + 1 < a.ncols) {
                    uint2 v = make_uint2(0, 0);
                    if (!first) v = __ldcg(reinterpret_cast<const uint2 *>(orow + t));
                    v.x += lo;
                    v.y += hi;
                    __stcg(reinterpret_cast<uint2 *>(orow + t), v);
                } else if (t < a.ncols) {
                    uint32_t v = first ? 0u : __ldcg(orow + t);
                    __stcg(orow + t, v + lo);
                }
            }
        }
    };

    // prologue: records 0 and 1, then load groups 0, 1 (and 2 once record 2 is in), rows of stage 0
    if (tid == 0) {
        const int n = nstages > 1 ? 2 : 1;
        mbar_expect_tx(setup, n * REC);
        bulk_g2s(rec0, recs, n * REC, setup);
    }
    mbar_wait(setup, 0);
    if (tid == 0) {
        issue(0);
        if (nstages > 1) issue(1);
    }
    mbar_wait(&rawbar[0], 0);
    if (tid == 0 && nstages > 2) issue(2);
    build(0);

    // all warps flush at the same stage: a warp that flushed alone would hold up the others, which
    // may run at most one phase ahead of it
    const int FL = a.sp_flush;
    int since = 0;
    bool first = true;

    for (int s = 0; s < nstages; ++s) {
        // every warp has built rows(s) and therefore finished accumulate(s-2): pattern buffer
        // (s+1) % NBUF, raw slot s % NBUF and record slot (s-3) % NREC are free
        mbar_wait(&full[s % NBUF], (uint32_t)((s / NBUF) & 1));
        if (s + 1 < nstages) {
            mbar_wait(&rawbar[(s + 1) % NBUF], (uint32_t)(((s + 1) / NBUF) & 1));   // rows(s+1), record(s+3)
            if (tid == 0 && s + 3 < nstages) issue(s + 3);
            build(s + 1);
        }

        // ---- accumulate: one row word per (trial, group, sample pair) ---------------------------
        {
            const SpRecord *R = record(s);
            const uint8_t *P = P0 + (s % NBUF) * pbytes + lane * 4;
#pragma unroll
            for (int k4 = 0; k4 < DPW; k4 += 4) {
                const uint4 po = *reinterpret_cast<const uint4 *>(&R->poff[warp * DPW + k4]);
                const uint32_t pof[4] = {po.x, po.y, po.z, po.w};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const uint32_t *p = reinterpret_cast<const uint32_t *>(P + pof[k]);
#pragma unroll
                    for (int i = 0; i < NP; ++i) acc16[k4 + k][i] += p[i * 32];
                }
            }
            if (++since == FL) {
                flush(first);
                first = false;
                since = 0;
            }
        }
    }
    if (since || first) flush(first);
}

template <int NT, int TB>
cudaError_t launch_t(const DedispArgs &a, cudaStream_t st)
{
    dim3 grid((unsigned)((a.ndms + DB - 1) / DB), (unsigned)((a.ncols + TB - 1) / TB));
    dedisp_sp_kernel<NT, TB><<<grid, NT, dedisp_sp_smem_bytes(a.sp_rows, a.sp_pbytes), st>>>(a);
    return cudaGetLastError();
}

}  // namespace

size_t dedisp_sp_smem_bytes(int rows, int pbytes)
{
    return (size_t)NBUF * pbytes + (size_t)NBUF * G * rows + NREC * REC + (2 * NBUF + 1) * 8;
}

cudaError_t dedisp_sp_configure()
{
    cudaError_t e = cudaFuncSetAttribute(dedisp_sp_kernel<512, 1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(dedisp_sp_kernel<256, 512>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
}

cudaError_t launch_dedisp_sp(const DedispArgs &a, int tb, cudaStream_t st)
{
    if (a.ncols <= 0 || a.ndms <= 0) return cudaSuccess;
    return tb == 1024 ? launch_t<512, 1024>(a, st) : launch_t<256, 512>(a, st);
}

}  // namespace aa
