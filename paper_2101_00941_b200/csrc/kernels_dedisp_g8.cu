// Brute-force incoherent dedispersion, 8-channel shared-pattern kernel for uint8 input
// (BASELINE.json north_star):  D[d][tau] = sum_c y[c][tau + delta(c,d)], exact.
//
// The successor of kernels_dedisp_ws.cu on the headline workloads.  That kernel moves one 32-bit row word through
// shared memory per (trial, 4-channel group, 2 samples) and sits at 86 % of the shared-memory pipe; the only way
// down is fewer bytes per unit.  Here a row sample is the sum of EIGHT adjacent channels, so the consumers load half
// as many words.  Wider groups have more distinct delay patterns (each delay is rounded on its own), which is paid
// for in two ways (g8_tables.cu):
//   * rows are built per HALF of the CTA's 64 trials (32 trials see 8.8 patterns of 8 channels on the 4096-channel
//     workloads; 64 trials would see 14 and their rows would not fit the shared-memory ring);
//   * a pattern is a pair (A, B) of a 3-vector for channels 1-3 and a 4-vector for channels 4-7; a producer lane sums
//     channels 0-3 once per distinct A, channels 4-7 once per distinct B, and forms each occurring pair with four
//     packed adds, so a row costs nA + nB four-channel sums plus npat pair sums instead of npat eight-channel sums.
//
// CTA = 16 consumer warps + 8 producer warps, tile = 64 trials x 1024 samples; stage s = 2 * group + half.
//   producers all eight warps build every stage together: its batches (31 row chunks of 8 samples each) are dealt
//             round the warps, continuing from stage to stage, so the load is even whatever the row length.  Channel
//             windows arrive by cp.async.bulk (TMA 1-D, mbarrier complete_tx) two groups ahead, one window set per
//             group serving both halves; every warp prefetches its own copy of the plan-time record (cp.async).
//             Rows are stored twice, as (s[2j], s[2j+1]) and (s[2j+1], s[2j+2]) pairs, so that any integer offset is
//             one aligned 32-bit load; they live in a shared-memory ring whose offsets are fixed at plan time.
//   consumers warps 0-7 own the trials of half 0 and consume the even stages, warps 8-15 the odd ones; a warp owns 4
//             trials, a lane 16 words of 2 samples: acc16 += row word (SWAR).  Every 32 own stages (256 channels:
//             255 * 256 < 2^16) the 16-bit lanes are added into the uint32 output tile in tensor memory (TMEM).
//   full[] / empty[] mbarrier rings order the two sides; nothing in the loop is CTA-wide.
// No tensor cores: a gather-add, not a dense contraction.
#include "aa_internal.h"
#include "ptx_util.cuh"

namespace aa {

namespace {

using namespace ptx;

constexpr int G = kG8;
constexpr int DB = kSpDB;
constexpr int H = kG8Half;
constexpr int TB = kG8TB;
constexpr int NCW = 16;                // consumer warps
constexpr int NPW = kG8Producers;      // producer warps
constexpr int DPW = DB / NCW;          // trials per consumer warp
constexpr int NRAW = kG8Ahead + 1;     // staged channel-window slots (one per group in flight)
constexpr int NSLOT = kG8Slots;        // full[] / empty[] barrier slots (stage modulo NSLOT)
constexpr int NRECBUF = 4;             // private record copies per producer warp (this stage, next three)
constexpr int REC = (int)sizeof(G8Record);
constexpr int NT = 32 * (NCW + NPW);
constexpr int NP = TB / 64;            // 2-sample words per consumer lane and trial
constexpr int REG_CONS = 88, REG_PROD = 64;
static_assert(DPW == 4, "trial offsets are fetched four at a time");
static_assert(NCW * REG_CONS + NPW * REG_PROD <= (NCW + NPW) * 80, "register budget");
static_assert(kG8Window % 2 == 0 && kG8Window < NSLOT, "the window keeps the stage parity");

// One channel's window of this lane: 20 bytes from the 8-byte boundary at or below its first sample, aligned to the
// channel's smallest shift.  xs0 / xs1 / xs2 = bytes 0-3 / 4-7 / 8-11 after alignment.
__device__ __forceinline__ void load_window(uint32_t cd, const uint8_t *q, uint32_t &xs0, uint32_t &xs1, uint32_t &xs2)
{
    const uint8_t *qi = q + (cd & 0xFFFFu);
    const uint2 v0 = *reinterpret_cast<const uint2 *>(qi);
    const uint2 v1 = *reinterpret_cast<const uint2 *>(qi + 8);
    const uint32_t w4 = *reinterpret_cast<const uint32_t *>(qi + 16);
    const bool up = (cd & 0x200000u) != 0;             // smallest shift >= 4 bytes: start one word later
    const uint32_t t0 = up ? v0.y : v0.x, t1 = up ? v1.x : v0.y, t2 = up ? v1.y : v1.x, t3 = up ? w4 : v1.y;
    const uint32_t sh = cd >> 16;                      // funnel shifts take the amount modulo 32
    xs0 = __funnelshift_r(t0, t1, sh);
    xs1 = __funnelshift_r(t1, t2, sh);
    xs2 = __funnelshift_r(t2, t3, sh);
}

// 8 samples of one channel, shifted by e8 / 8 more bytes, into four words of two 15-bit lanes (IDP.2A)
__device__ __forceinline__ void add_channel(uint32_t (&acc)[4], uint32_t xs0, uint32_t xs1, uint32_t xs2, uint32_t e8)
{
    const uint32_t x0 = __funnelshift_r(xs0, xs1, e8), x1 = __funnelshift_r(xs1, xs2, e8);
    dp2a_lo(acc[0], x0);
    dp2a_hi(acc[1], x0);
    dp2a_lo(acc[2], x1);
    dp2a_hi(acc[3], x1);
}

// One batch (31 row chunks of 8 samples; lane 31 only feeds lane 30 its first word) of the rows whose A pattern is
// ka0 .. ka0+NA-1.  q: this lane's first window byte of channel 0, chunk offset included; dst: shared address of this
// lane's four words of row 0's even copy; st: this lane stores; rowbytes: bytes per copy; row: first row to emit.
template <int NA>
__device__ __forceinline__ void build_batch(const G8Record *R, const uint8_t *q, uint32_t dst, uint32_t st, uint32_t rowbytes,
                                            int ka0, uint32_t row)
{
    uint32_t A[NA][4];
#pragma unroll
    for (int k = 0; k < NA; ++k)
#pragma unroll
        for (int j = 0; j < 4; ++j) A[k][j] = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        uint32_t xs0, xs1, xs2;
        load_window(R->chdesc[i], q, xs0, xs1, xs2);
        uint32_t es = 0;
        if (i > 0) es = *reinterpret_cast<const uint32_t *>(&R->eA[i - 1][ka0]);   // ka0 is 0 or 4
#pragma unroll
        for (int k = 0; k < NA; ++k) add_channel(A[k], xs0, xs1, xs2, i > 0 ? es >> (8 * k) : 0u);
    }
    uint32_t xb[4][3];
#pragma unroll
    for (int i = 0; i < 4; ++i) load_window(R->chdesc[4 + i], q, xb[i][0], xb[i][1], xb[i][2]);

    const int nB = R->nB;
#pragma unroll 1
    for (int kb = 0; kb < nB; ++kb) {
        const uint32_t pairs = ((uint32_t)R->comb[kb] >> ka0) & ((1u << NA) - 1u);     // warp-uniform
        if (!pairs) continue;
        uint32_t Bs[4] = {0, 0, 0, 0};
#pragma unroll
        for (int i = 0; i < 4; ++i) add_channel(Bs, xb[i][0], xb[i][1], xb[i][2], R->eB[i][kb]);
#pragma unroll
        for (int k = 0; k < NA; ++k) {
            if (!(pairs >> k & 1u)) continue;
            // eight-channel sums <= 2040 < 2^15: the 15-bit lanes add without carry; then 15-bit -> 16-bit lanes:
            // w + (w & ~0x7FFF) moves lane 1 up by one bit
            uint32_t c[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                c[j] = A[k][j] + Bs[j];
                c[j] += c[j] & 0xFFFF8000u;
            }
            const uint32_t nx = __shfl_down_sync(0xFFFFFFFFu, c[0], 1);
            const uint32_t d = dst + 2u * row * rowbytes;
            sts128_if(d, c[0], c[1], c[2], c[3], st);
            sts128_if(d + rowbytes, __byte_perm(c[0], c[1], 0x5432), __byte_perm(c[1], c[2], 0x5432),
                      __byte_perm(c[2], c[3], 0x5432), __byte_perm(c[3], nx, 0x5432), st);
            ++row;
        }
    }
}

template <int NA>
__device__ __forceinline__ void build_pass(const G8Record *R, const uint8_t *rawslot, uint32_t P, int first, int lane, int ka0,
                                           uint32_t row0)
{
    const uint32_t nchunk = R->nchunk, nbatch = R->nbatch, rowbytes = 16u * nchunk;
    for (uint32_t b = (uint32_t)first; b < nbatch; b += NPW) {
        const uint32_t chunk = b * 31u + (uint32_t)lane;
        // chunk nchunk is read for its first sample only; nothing beyond it is read
        const uint8_t *q = rawslot + 8u * (chunk < nchunk ? chunk : nchunk);
        build_batch<NA>(R, q, P + 16u * chunk, lane < 31 && chunk < nchunk, rowbytes, ka0, row0);
    }
}

__device__ __forceinline__ void build_stage(const G8Record *R, const uint8_t *rawslot, uint32_t P, int first, int lane)
{
    const int nA = R->nA;
    switch (nA < 4 ? nA : 4) {
        case 1: build_pass<1>(R, rawslot, P, first, lane, 0, 0); break;
        case 2: build_pass<2>(R, rawslot, P, first, lane, 0, 0); break;
        case 3: build_pass<3>(R, rawslot, P, first, lane, 0, 0); break;
        default: build_pass<4>(R, rawslot, P, first, lane, 0, 0); break;
    }
    if (nA > 4) {
        const uint32_t row0 = R->rows0;
        switch (nA - 4) {
            case 1: build_pass<1>(R, rawslot, P, first, lane, 4, row0); break;
            case 2: build_pass<2>(R, rawslot, P, first, lane, 4, row0); break;
            case 3: build_pass<3>(R, rawslot, P, first, lane, 4, row0); break;
            default: build_pass<4>(R, rawslot, P, first, lane, 4, row0); break;
        }
    }
}

__global__ void __launch_bounds__(NT, 1) dedisp_g8_kernel(const DedispArgs a)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t ROWS = (uint32_t)a.sp_rows;
    const uint32_t raw_bytes = G * ROWS;
    const uint32_t ring_bytes = (uint32_t)a.sp_pbytes;
    uint8_t *P0 = smem;                                     // pattern-row ring: per stage [row][E|O][4 * nchunk] uint32
    uint8_t *raw0 = P0 + ring_bytes;                        // [NRAW][G][ROWS] staged channel windows
    uint8_t *rec0 = raw0 + NRAW * raw_bytes;                // [NPW][NRECBUF][REC] private record copies
    const uint32_t sm_P = smem_u32(P0), sm_raw = smem_u32(raw0), sm_rec = smem_u32(rec0);
    uint8_t *pof0 = rec0 + NPW * NRECBUF * REC;             // [NSLOT][H] trial offsets of the stages in flight
    const uint32_t sm_pof = smem_u32(pof0);
    const uint32_t rawfull = sm_pof + NSLOT * H * 4;        // [NRAW] windows of a group landed
    const uint32_t full = rawfull + 8 * NRAW;               // [NSLOT] every producer warp has built its part of stage s
    const uint32_t empty = full + 8 * NSLOT;                // [NSLOT] every consumer warp of the half has used it

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d0 = blockIdx.x * DB;
    const int64_t t0 = (int64_t)blockIdx.y * TB;
    const int ngrp = (a.nchans + G - 1) / G, nstages = 2 * ngrp;
    const uint8_t *recs = static_cast<const uint8_t *>(a.sp_tab) + (size_t)blockIdx.x * nstages * REC;

    // TMEM columns of the tile: 2 per packed accumulator word, 4 column groups (warp / 4) x 4 lane quadrants (warp % 4)
    constexpr uint32_t TCOLS = (uint32_t)(8 * DPW * NP);
    const uint32_t tmem_slot = empty + 8 * NSLOT;           // the allocator writes the TMEM base address here
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "n"(TCOLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid == 0) {
#pragma unroll
        for (int j = 0; j < NRAW; ++j) mbar_init(rawfull + 8 * j, 1);
#pragma unroll
        for (int j = 0; j < NSLOT; ++j) {
            mbar_init(full + 8 * j, NPW);
            mbar_init(empty + 8 * j, NCW / 2);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    uint32_t tmem_base_s;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base_s) : "r"(tmem_slot) : "memory");

    if (warp >= NCW) {
        // ================================ producers ================================================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(REG_PROD));
        const int pw = warp - NCW;
        const uint8_t *in = static_cast<const uint8_t *>(a.in) + (a.col0 + t0);
        const uint32_t myrec = sm_rec + pw * (NRECBUF * REC);
        const uint8_t *myrecp = rec0 + pw * (NRECBUF * REC);

        // this warp's private copy of record q into copy slot q % NRECBUF (asynchronous; one commit group)
        auto prefetch_record = [&](int q) {
            if (q < nstages && lane < REC / 16)
                cp_async16(myrec + (q % NRECBUF) * REC + lane * 16, recs + (size_t)q * REC + lane * 16);
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        // one lane: the eight channel windows of group gq, described by the descriptor record R carries, into slot w
        auto issue = [&](int gq, const G8Record *R, int w) {
            uint32_t bytes = 0;
#pragma unroll
            for (int i = 0; i < G; ++i) bytes += R->nrbytes[i];
            const uint32_t bar = rawfull + 8 * w;
            mbar_expect_tx(bar, bytes);
            const uint32_t dst = sm_raw + w * raw_bytes;
#pragma unroll
            for (int i = 0; i < G; ++i)
                bulk_g2s(dst + i * ROWS, in + ((size_t)(gq * G + i) * a.pitch_in + R->nrbase[i]), R->nrbytes[i], bar);
        };

        prefetch_record(0);
        prefetch_record(1);
        prefetch_record(2);
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncwarp();
        if (pw == 0 && lane == 0) {
            // groups 0 .. kG8Ahead-1: their own descriptors sit in the records of their first stages
            issue(0, reinterpret_cast<const G8Record *>(myrecp), 0);
            if (ngrp > 1) issue(1, reinterpret_cast<const G8Record *>(myrecp + 2 * REC), 1);
        }
        __syncwarp();

        for (int s = 0; s < nstages; ++s) {
            const int g = s >> 1;
            // record of stage s + 3 (its copy slot was last read one stage ago); then the record of this stage has landed
            prefetch_record(s + 3);
            asm volatile("cp.async.wait_group 3;" ::: "memory");
            __syncwarp();
            const G8Record *R = reinterpret_cast<const G8Record *>(myrecp + (s % NRECBUF) * REC);
            if (pw == 0 && lane == 0 && (s & 1) && g + kG8Ahead < ngrp) {
                // the windows of group g + kG8Ahead go to the slot of group g - 1: every producer warp must be done
                // with that group's last stage
                const int f = s - 2;
                if (f >= 0) mbar_wait_lane(full + 8 * (f % NSLOT), (uint32_t)((f / NSLOT) & 1));
                issue(g + kG8Ahead, R, (g + kG8Ahead) % NRAW);
            }
            __syncwarp();
            // the rows may be written once the consumers are done with the stages that lie under them in the ring
            const int dep0 = R->dep[0], dep1 = R->dep[1];
            if (dep0 >= 0) mbar_wait(empty + 8 * (dep0 % NSLOT), (uint32_t)((dep0 / NSLOT) & 1));
            if (dep1 >= 0) mbar_wait(empty + 8 * (dep1 % NSLOT), (uint32_t)((dep1 / NSLOT) & 1));
            // the stage's trial offsets go to its barrier slot (last used by stage s - NSLOT, consumed long ago)
            if (pw == s % NPW && lane < H / 4)
                *reinterpret_cast<uint4 *>(pof0 + (s % NSLOT) * (H * 4) + lane * 16) =
                    *reinterpret_cast<const uint4 *>(reinterpret_cast<const uint8_t *>(R->poff) + lane * 16);
            const int w = g % NRAW;
            mbar_wait(rawfull + 8 * w, (uint32_t)((g / NRAW) & 1));

            // this warp's batches: batch b of the stage is global batch bstart + b, dealt round the warps
            const int first = (pw - (int)R->bstart + NPW) % NPW;
            build_stage(R, raw0 + w * raw_bytes, sm_P + R->pofs, first, lane);
            __syncwarp();
            if (lane == 0) mbar_arrive(full + 8 * (s % NSLOT));
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        return;
    }

    // ==================================== consumers ================================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REG_CONS));
    uint32_t acc16[DPW][NP];
#pragma unroll
    for (int k = 0; k < DPW; ++k)
#pragma unroll
        for (int i = 0; i < NP; ++i) acc16[k][i] = 0;

    const bool whole = d0 + DB <= a.ndms && t0 + TB <= (int64_t)a.ncols;   // CTA-uniform: no edge tests
    uint32_t *otile = a.out + (size_t)(d0 + warp * DPW) * a.pitch_out + t0 + 2 * lane;

    // this warp's part of the tile in TMEM: lane quadrant warp % 4, 2 * DPW * NP columns from (warp / 4) * that
    const uint32_t ttile = tmem_base_s + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * (2 * DPW * NP));

    // adds the 16-bit lanes into the uint32 tile in TMEM (first time: plain store) and clears them
    auto flush = [&](bool first) {
#pragma unroll
        for (int k = 0; k < DPW; ++k) {
#pragma unroll
            for (int h = 0; h < NP; h += 4) {
                const uint32_t col = ttile + (uint32_t)(2 * (k * NP + h));
                uint32_t v[8];
                if (first) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) v[i] = 0;
                } else {
                    tmem_ld8(v, col);
                }
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    v[2 * i] += acc16[k][h + i] & 0xFFFFu;
                    v[2 * i + 1] += acc16[k][h + i] >> 16;
                    acc16[k][h + i] = 0;
                }
                tmem_st8(col, v);
            }
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    };
    // the finished tile: TMEM (if anything was flushed) plus what is still in the 16-bit lanes, to global memory
    auto write_out = [&](bool first) {
#pragma unroll
        for (int k = 0; k < DPW; ++k) {
            const int d = d0 + warp * DPW + k;
            uint32_t *orow = otile + (size_t)k * a.pitch_out;
#pragma unroll
            for (int h = 0; h < NP; h += 4) {
                uint32_t v[8];
                if (first) {
#pragma unroll
                    for (int i = 0; i < 8; ++i) v[i] = 0;
                } else {
                    tmem_ld8(v, ttile + (uint32_t)(2 * (k * NP + h)));
                }
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const uint32_t lo = v[2 * i] + (acc16[k][h + i] & 0xFFFFu), hi = v[2 * i + 1] + (acc16[k][h + i] >> 16);
                    if (whole) {
                        __stcg(reinterpret_cast<uint2 *>(orow + 64 * (h + i)), make_uint2(lo, hi));
                    } else if (d < a.ndms) {
                        const int64_t t = t0 + 2 * (lane + 32 * (h + i));
                        if (t + 1 < a.ncols) __stcg(reinterpret_cast<uint2 *>(orow + 64 * (h + i)), make_uint2(lo, hi));
                        else if (t < a.ncols) __stcg(orow + 64 * (h + i), lo);
                    }
                }
            }
        }
    };

    const int FL = a.sp_flush;
    int since = 0;
    bool first = true;
    const uint8_t *Pl = P0 + lane * 4;
    // this warp's four trial offsets (absolute inside the ring) are published by the producers with the rows
    const uint8_t *mypof = pof0 + (warp & 7) * (DPW * 4);
    for (int s = warp >> 3; s < nstages; s += 2) {
        const uint32_t sl = (uint32_t)(s % NSLOT), slot = 8u * sl;
        mbar_wait(full + slot, (uint32_t)((s / NSLOT) & 1));
        const uint4 po = *reinterpret_cast<const uint4 *>(mypof + sl * (H * 4));

        // one row word per (trial, group, sample pair); eight loads in flight per batch
        const uint32_t pof[4] = {po.x, po.y, po.z, po.w};
#pragma unroll
        for (int k = 0; k < DPW; ++k) {
            const uint32_t *p = reinterpret_cast<const uint32_t *>(Pl + pof[k]);
#pragma unroll
            for (int h = 0; h < NP; h += 8) {
                uint32_t v[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) v[i] = p[(h + i) * 32];
#pragma unroll
                for (int i = 0; i < 8; ++i) acc16[k][h + i] += v[i];
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + slot);

        if (++since == FL) {
            flush(first);
            first = false;
            since = 0;
        }
    }
    write_out(first);
    // every consumer warp is done with TMEM before warp 0 gives it back
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    asm volatile("bar.sync 1, %0;" ::"n"(32 * NCW) : "memory");
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base_s), "n"(TCOLS) : "memory");
    }
}

}  // namespace

size_t dedisp_g8_fixed_smem_bytes(int rows)
{
    return (size_t)NRAW * G * rows + (size_t)NPW * NRECBUF * REC + (size_t)NSLOT * H * 4 + (NRAW + 2 * NSLOT) * 8 + 8;
}

size_t dedisp_g8_smem_bytes(int rows, int ring_bytes)
{
    return (size_t)ring_bytes + dedisp_g8_fixed_smem_bytes(rows);
}

cudaError_t dedisp_g8_configure()
{
    return cudaFuncSetAttribute(dedisp_g8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
}

cudaError_t launch_dedisp_g8(const DedispArgs &a, cudaStream_t st)
{
    if (a.ncols <= 0 || a.ndms <= 0) return cudaSuccess;
    dim3 grid((unsigned)((a.ndms + DB - 1) / DB), (unsigned)((a.ncols + TB - 1) / TB));
    dedisp_g8_kernel<<<grid, NT, dedisp_g8_smem_bytes(a.sp_rows, a.sp_pbytes), st>>>(a);
    return cudaGetLastError();
}

}  // namespace aa
