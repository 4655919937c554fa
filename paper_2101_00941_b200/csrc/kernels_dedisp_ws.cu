// Brute-force incoherent dedispersion, warp-specialised shared-pattern kernel
// (BASELINE.json north_star):  D[d][tau] = sum_c y[c][tau + delta(c,d)], exact.
//
// Channels are taken in groups of kSpG = 4.  Inside a block of 64 consecutive trials the group's
// rounded delays, relative to its first channel, form only a few distinct vectors ("patterns",
// ws_tables.cu); the CTA sums the 4 channels once per pattern into a row of 16-bit sums and each
// trial then adds ONE row sample per group.  Same integers, same sums, a quarter of the adds.
//
// CTA = 16 consumer warps + 8 producer warps, tile = 64 trials x TB samples, one stage per group:
//   producers work in teams of TEAM warps; a team owns every NTEAM-th stage.  Its leader requests
//             the stage's 4 channel windows one turn ahead with cp.async.bulk (TMA 1-D, mbarrier
//             complete_tx); every warp prefetches its own copy of the plan-time record (cp.async).
//             A lane owns 8 consecutive row samples of EVERY pattern: per channel it loads one
//             20-byte window, aligns it to the smallest shift with funnel shifts, and per pattern
//             adds it with IDP.2A (dp2a: two byte adds into two 15-bit lanes, FMA pipe).  Rows are
//             stored twice, as (s[2j], s[2j+1]) and (s[2j+1], s[2j+2]) pairs, so that any integer
//             offset is one aligned 32-bit load (the 9th sample comes from the next lane by SHFL).
//             Pattern rows live in a shared-memory ring whose offsets are fixed at plan time, so a
//             stage takes exactly the room it needs and about six stages are in flight.
//   consumers a warp owns 4 trials, a lane TB/64 words of 2 samples: acc16 += row word (SWAR).
//             Every sp_flush groups the 16-bit lanes are added into the uint32 output tile, which lives in
//             tensor memory (TMEM); only the finished tile goes to global memory.
//   full[] / empty[] mbarrier rings (one slot per stage, modulo 16) order the two sides; nothing in
//   the loop is CTA-wide.
// No tensor cores: a gather-add, not a dense contraction.
#include "aa_internal.h"
#include "ptx_util.cuh"

namespace aa {

namespace {

using namespace ptx;

constexpr int G = kSpG;
constexpr int DB = kSpDB;
constexpr int NCW = 16;                // consumer warps
constexpr int NPW = 8;                 // producer warps
constexpr int DPW = DB / NCW;          // trials per consumer warp
constexpr int TEAM = kWsTeam;          // producer warps per stage
constexpr int NTEAM = NPW / TEAM;      // stages being built at the same time
constexpr int NRAW = 2 * NTEAM;        // staged channel-window slots: two per team
constexpr int NSLOT = kWsSlots;        // full[] / empty[] barrier slots (stage modulo NSLOT)
constexpr int NRECBUF = 3;             // private record copies per producer warp (this turn, next two)
constexpr int REC = (int)sizeof(WsRecord);
constexpr int NT = 32 * (NCW + NPW);
// Registers: the CTA is launched with 80 per thread (768 * 80 = 61440); the consumer warpgroups
// then take 88 (64 accumulators + loads in flight) and the producer warpgroups drop to 64.
constexpr int REG_CONS = 88, REG_PROD = 64;
static_assert(DPW == 4, "trial offsets are fetched four at a time");
static_assert(NCW % 4 == 0 && NPW % 4 == 0, "setmaxnreg works on warpgroups");
static_assert(NCW * REG_CONS + NPW * REG_PROD <= (NCW + NPW) * 80, "register budget");

// Pattern rows K0 .. K0+NPAT-1 of one batch (31 row chunks of 8 samples; lane 31 only feeds lane 30
// its first word).  q: this lane's first window byte of channel 0, chunk offset included; dst: shared
// address of this lane's four words of pattern 0's even copy; st: this lane stores; rowbytes: bytes per copy.
template <int NPAT, int K0>
__device__ __forceinline__ void build_batch(const uint32_t (&cds)[G], const WsRecord *Rr, const uint8_t *q, uint32_t dst, uint32_t st, uint32_t rowbytes)
{
    uint32_t acc[NPAT][4];
#pragma unroll
    for (int k = 0; k < NPAT; ++k)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[k][j] = 0;

#pragma unroll
    for (int i = 0; i < G; ++i) {
        const uint32_t cd = cds[i];
        const uint8_t *qi = q + (cd & 0xFFFFu);
        const uint2 v0 = *reinterpret_cast<const uint2 *>(qi);
        const uint2 v1 = *reinterpret_cast<const uint2 *>(qi + 8);
        const uint32_t w4 = *reinterpret_cast<const uint32_t *>(qi + 16);
        const bool up = (cd & 0x200000u) != 0;             // smallest shift >= 4 bytes: start one word later
        const uint32_t t0 = up ? v0.y : v0.x, t1 = up ? v1.x : v0.y, t2 = up ? v1.y : v1.x, t3 = up ? w4 : v1.y;
        const uint32_t sh = cd >> 16;                      // funnel shifts take the amount modulo 32
        const uint32_t xs0 = __funnelshift_r(t0, t1, sh), xs1 = __funnelshift_r(t1, t2, sh),
                       xs2 = __funnelshift_r(t2, t3, sh);
        uint2 es = make_uint2(0, 0);
        if (i > 0) es = *reinterpret_cast<const uint2 *>(Rr->esh[i]);
#pragma unroll
        for (int k = 0; k < NPAT; ++k) {
            uint32_t x0 = xs0, x1 = xs1;
            if (i > 0) {                                   // channel 0 is the reference: no extra shift
                const int kk = K0 + k;
                const uint32_t e8 = (kk < 4 ? es.x : es.y) >> (8 * (kk & 3));   // 8 * extra shift of pattern kk
                x0 = __funnelshift_r(xs0, xs1, e8);
                x1 = __funnelshift_r(xs1, xs2, e8);
            }
            dp2a_lo(acc[k][0], x0);
            dp2a_hi(acc[k][1], x0);
            dp2a_lo(acc[k][2], x1);
            dp2a_hi(acc[k][3], x1);
        }
    }

#pragma unroll
    for (int k = 0; k < NPAT; ++k) {
        // 15-bit lanes -> 16-bit lanes: w + (w & ~0x7FFF) moves lane 1 up by one bit
        uint32_t c[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) c[j] = acc[k][j] + (acc[k][j] & 0xFFFF8000u);
        const uint32_t nx = __shfl_down_sync(0xFFFFFFFFu, c[0], 1);
        const uint32_t d = dst + (uint32_t)(2 * (K0 + k)) * rowbytes;
        sts128_if(d, c[0], c[1], c[2], c[3], st);
        sts128_if(d + rowbytes, __byte_perm(c[0], c[1], 0x5432), __byte_perm(c[1], c[2], 0x5432),
                  __byte_perm(c[2], c[3], 0x5432), __byte_perm(c[3], nx, 0x5432), st);
    }
}

// The same for 16-bit input (time-binned ranges: samples <= 255 * bin, four-channel sums < 2^16, so the two
// 16-bit lanes of a word are simply added).  q: this lane's first window byte of channel 0 (16 bytes per
// chunk); a lane reads 12 samples per channel from the 8-byte boundary at or below its first sample, aligns
// them to the channel's smallest shift (word select + 16-bit funnel shift) and per pattern shifts by the
// extra e_{k,i} <= 2 samples with one PRMT (selector 0x3210 + e * 0x2222: 0, 2 or 4 bytes into the word pair).
template <int NPAT, int K0>
__device__ __forceinline__ void build_batch16(const uint32_t (&cds)[G], const WsRecord *Rr, const uint8_t *q, uint32_t dst, uint32_t st, uint32_t rowbytes)
{
    uint32_t acc[NPAT][4];
#pragma unroll
    for (int k = 0; k < NPAT; ++k)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[k][j] = 0;

#pragma unroll
    for (int i = 0; i < G; ++i) {
        const uint32_t cd = cds[i];
        const uint8_t *qi = q + (cd & 0xFFFFu);
        const uint2 v0 = *reinterpret_cast<const uint2 *>(qi);
        const uint2 v1 = *reinterpret_cast<const uint2 *>(qi + 8);
        const uint2 v2 = *reinterpret_cast<const uint2 *>(qi + 16);
        const uint32_t w6 = *reinterpret_cast<const uint32_t *>(qi + 24);
        const uint32_t sh = (cd >> 16) & 3u;               // smallest shift modulo 4 samples
        const bool up = sh >= 2u;                          // start one word later
        const uint32_t a0 = up ? v0.y : v0.x, a1 = up ? v1.x : v0.y, a2 = up ? v1.y : v1.x, a3 = up ? v2.x : v1.y,
                       a4 = up ? v2.y : v2.x, a5 = up ? w6 : v2.y;
        const uint32_t f = (sh & 1u) * 16u;
        const uint32_t t0 = __funnelshift_r(a0, a1, f), t1 = __funnelshift_r(a1, a2, f), t2 = __funnelshift_r(a2, a3, f),
                       t3 = __funnelshift_r(a3, a4, f), t4 = __funnelshift_r(a4, a5, f);
        uint2 es = make_uint2(0, 0);
        if (i > 0) es = *reinterpret_cast<const uint2 *>(Rr->esh[i]);
#pragma unroll
        for (int k = 0; k < NPAT; ++k) {
            uint32_t x0 = t0, x1 = t1, x2 = t2, x3 = t3;
            if (i > 0) {                                   // channel 0 is the reference: no extra shift
                const int kk = K0 + k;
                const uint32_t e = ((kk < 4 ? es.x : es.y) >> (8 * (kk & 3))) & 0xFFu;   // extra shift of pattern kk
                const uint32_t sel = 0x3210u + e * 0x2222u;
                x0 = __byte_perm(t0, t1, sel);
                x1 = __byte_perm(t1, t2, sel);
                x2 = __byte_perm(t2, t3, sel);
                x3 = __byte_perm(t3, t4, sel);
            }
            acc[k][0] += x0;
            acc[k][1] += x1;
            acc[k][2] += x2;
            acc[k][3] += x3;
        }
    }

#pragma unroll
    for (int k = 0; k < NPAT; ++k) {
        const uint32_t *c = acc[k];
        const uint32_t nx = __shfl_down_sync(0xFFFFFFFFu, c[0], 1);
        const uint32_t d = dst + (uint32_t)(2 * (K0 + k)) * rowbytes;
        sts128_if(d, c[0], c[1], c[2], c[3], st);
        sts128_if(d + rowbytes, __byte_perm(c[0], c[1], 0x5432), __byte_perm(c[1], c[2], 0x5432),
                  __byte_perm(c[2], c[3], 0x5432), __byte_perm(c[3], nx, 0x5432), st);
    }
}

template <bool IN16, int NPAT_LO, int NPAT_HI>
__device__ __forceinline__ void build_stage(const WsRecord *R, const uint8_t *rawslot, uint32_t P, uint32_t nchunk,
                                            uint32_t nbatch, int member, int lane)
{
    const uint32_t rowbytes = 16u * nchunk;
    // the stage's channel descriptors stay in registers over the batches (one uniform load and its latency less per
    // channel and batch: 25.88 -> 25.36 ms per cfg3 launch); the extra shifts too would spill (measured: slower)
    // (16-bit input keeps more values alive per lane and would spill: it reads them in every batch)
    uint32_t cds[G];
    if (!IN16) {
#pragma unroll
        for (int i = 0; i < G; ++i) cds[i] = R->chdesc[i];
    }
    for (uint32_t b = (uint32_t)member; b < nbatch; b += TEAM) {
        if (IN16) {
#pragma unroll
            for (int i = 0; i < G; ++i) cds[i] = R->chdesc[i];
        }
        const uint32_t chunk = b * 31u + (uint32_t)lane;
        // chunk nchunk is read for its first sample only; nothing beyond it is read
        const uint8_t *q = rawslot + (IN16 ? 16u : 8u) * (chunk < nchunk ? chunk : nchunk);
        const uint32_t dst = P + 16u * chunk;
        const uint32_t st = lane < 31 && chunk < nchunk;
        if (IN16) {
            build_batch16<NPAT_LO, 0>(cds, R, q, dst, st, rowbytes);
            if (NPAT_HI > 0) build_batch16<(NPAT_HI > 0 ? NPAT_HI : 1), NPAT_LO>(cds, R, q, dst, st, rowbytes);
        } else {
            build_batch<NPAT_LO, 0>(cds, R, q, dst, st, rowbytes);
            if (NPAT_HI > 0) build_batch<(NPAT_HI > 0 ? NPAT_HI : 1), NPAT_LO>(cds, R, q, dst, st, rowbytes);
        }
    }
}

// WIDE: the consumers keep one 32-bit accumulator per sample (TB = 512) and never flush: for coarse time bins,
// whose four-channel sums would fill 16-bit lanes after two or four groups.
template <int TB, bool IN16, bool WIDE = false>
__global__ void __launch_bounds__(NT, 1) dedisp_ws_kernel(const DedispArgs a)
{
    static_assert(!WIDE || TB == 512, "32-bit accumulators: 4 trials x 16 samples per lane");
    constexpr int ES = IN16 ? 2 : 1;       // bytes per input sample
    constexpr int NP = TB / 64;            // 2-sample words per consumer lane

    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t ROWS = (uint32_t)a.sp_rows;
    const uint32_t raw_bytes = G * ROWS;
    const uint32_t ring_bytes = (uint32_t)a.sp_pbytes;
    uint8_t *P0 = smem;                                     // pattern-row ring: per stage [pattern][E|O][4 * nchunk] uint32
    uint8_t *raw0 = P0 + ring_bytes;                        // [NRAW][G][ROWS] staged channel windows
    uint8_t *rec0 = raw0 + NRAW * raw_bytes;                // [NPW][NRECBUF][REC] private record copies
    const uint32_t sm_P = smem_u32(P0), sm_raw = smem_u32(raw0), sm_rec = smem_u32(rec0);
    uint8_t *pof0 = rec0 + NPW * NRECBUF * REC;             // [NSLOT][DB] trial offsets of the stages in flight
    const uint32_t sm_pof = smem_u32(pof0);
    const uint32_t rawfull = sm_pof + NSLOT * DB * 4;       // [NRAW] windows of a stage landed
    const uint32_t full = rawfull + 8 * NRAW;               // [NSLOT] the team has built the rows of stage s
    const uint32_t empty = full + 8 * NSLOT;                // [NSLOT] every consumer warp has used them

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d0 = blockIdx.x * DB;
    const int64_t t0 = (int64_t)blockIdx.y * TB;
    const int nstages = (a.nchans + G - 1) / G;
    const uint8_t *recs = static_cast<const uint8_t *>(a.sp_tab) + (size_t)blockIdx.x * nstages * REC;

    // TMEM columns of the tile: 2 per packed accumulator word, 4 column groups (warp / 4) x 4 lane quadrants (warp % 4)
    constexpr uint32_t TCOLS = WIDE ? 32u : (uint32_t)(8 * DPW * NP);
    const uint32_t tmem_slot = empty + 8 * NSLOT;           // the allocator writes the TMEM base address here
    if (!WIDE && warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "n"(TCOLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid == 0) {
#pragma unroll
        for (int j = 0; j < NRAW; ++j) mbar_init(rawfull + 8 * j, 1);
#pragma unroll
        for (int j = 0; j < NSLOT; ++j) {
            mbar_init(full + 8 * j, TEAM);
            mbar_init(empty + 8 * j, NCW);
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
        const int pw = warp - NCW, team = pw / TEAM, member = pw % TEAM;
        const uint8_t *in = static_cast<const uint8_t *>(a.in) + (a.col0 + t0) * ES;
        const uint32_t myrec = sm_rec + pw * (NRECBUF * REC);
        const uint8_t *myrecp = rec0 + pw * (NRECBUF * REC);

        // this warp's private copy of record q into copy slot j (asynchronous; one commit group)
        auto prefetch_record = [&](int q, int j) {
            if (q < nstages && lane < REC / 16) cp_async16(myrec + j * REC + lane * 16, recs + (size_t)q * REC + lane * 16);
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        // leader lane: the four channel windows of the stage described by record copy R (channels 4 R->group ..), into window slot w
        auto issue = [&](const WsRecord *R, int w) {
            uint32_t bytes = 0;
#pragma unroll
            for (int i = 0; i < G; ++i) bytes += R->rbytes[i];
            const uint32_t bar = rawfull + 8 * w;
            mbar_expect_tx(bar, bytes);
            const uint32_t dst = sm_raw + w * raw_bytes;
#pragma unroll
            for (int i = 0; i < G; ++i)
                bulk_g2s(dst + i * ROWS, in + ((size_t)(R->group * G + i) * a.pitch_in + R->rbase[i]) * ES, R->rbytes[i], bar);
        };

        // turn it of this team is stage s = team + it * NTEAM; record copy slot it % 3, window slot 2 * team + (it & 1)
        prefetch_record(team, 0);
        prefetch_record(team + NTEAM, 1);
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        __syncwarp();
        if (member == 0 && lane == 0 && team < nstages) issue(reinterpret_cast<const WsRecord *>(myrecp), 2 * team);
        __syncwarp();

        int rj = 0;                              // it % NRECBUF
        for (int s = team, it = 0; s < nstages; s += NTEAM, ++it) {
            const int rj1 = rj + 1 == NRECBUF ? 0 : rj + 1, rj2 = rj1 + 1 == NRECBUF ? 0 : rj1 + 1;
            // record of the turn after next (its copy slot was last read two turns ago); then the records of
            // this turn and the next one have landed
            prefetch_record(s + 2 * NTEAM, rj2);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
            __syncwarp();
            const WsRecord *R = reinterpret_cast<const WsRecord *>(myrecp + rj * REC);
            if (member == 0 && lane == 0 && s + NTEAM < nstages) {
                // next turn's windows go to the slot read one turn ago: the whole team must be done with it
                const int f = s - NTEAM;
                if (f >= 0) mbar_wait_lane(full + 8 * (f % NSLOT), (uint32_t)((f / NSLOT) & 1));
                issue(reinterpret_cast<const WsRecord *>(myrecp + rj1 * REC), 2 * team + ((it + 1) & 1));
            }
            __syncwarp();
            const uint32_t nchunk = R->nchunk, nbatch = R->nbatch, npat = R->npat;
            const int dep = R->dep;              // last stage whose rows overlap this stage's room in the ring
            if (dep >= 0) mbar_wait(empty + 8 * (dep % NSLOT), (uint32_t)((dep / NSLOT) & 1));
            // the stage's trial offsets go to its barrier slot (last used by stage s - NSLOT, consumed long ago)
            if (member == 0 && lane < DB / 4)
                *reinterpret_cast<uint4 *>(pof0 + (s % NSLOT) * (DB * 4) + lane * 16) =
                    *reinterpret_cast<const uint4 *>(reinterpret_cast<const uint8_t *>(R->poff) + lane * 16);
            const int w = 2 * team + (it & 1);
            mbar_wait(rawfull + 8 * w, (uint32_t)((it >> 1) & 1));

            const uint8_t *rawslot = raw0 + w * raw_bytes;
            const uint32_t P = sm_P + R->pofs;
            switch (npat) {
                case 1: build_stage<IN16, 1, 0>(R, rawslot, P, nchunk, nbatch, member, lane); break;
                case 2: build_stage<IN16, 2, 0>(R, rawslot, P, nchunk, nbatch, member, lane); break;
                case 3: build_stage<IN16, 3, 0>(R, rawslot, P, nchunk, nbatch, member, lane); break;
                case 4: build_stage<IN16, 4, 0>(R, rawslot, P, nchunk, nbatch, member, lane); break;
                case 5: build_stage<IN16, 5, 0>(R, rawslot, P, nchunk, nbatch, member, lane); break;
                case 6: build_stage<IN16, 6, 0>(R, rawslot, P, nchunk, nbatch, member, lane); break;
                case 7: build_stage<IN16, 4, 3>(R, rawslot, P, nchunk, nbatch, member, lane); break;
                default: build_stage<IN16, 4, 4>(R, rawslot, P, nchunk, nbatch, member, lane); break;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(full + 8 * (s % NSLOT));
            rj = rj1;
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        return;
    }

    // ==================================== consumers ================================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(REG_CONS));
    if constexpr (WIDE) {
        uint32_t acc[DPW][2 * NP];
#pragma unroll
        for (int k = 0; k < DPW; ++k)
#pragma unroll
            for (int i = 0; i < 2 * NP; ++i) acc[k][i] = 0;
        const uint8_t *Pl = P0 + lane * 4;
        const uint8_t *mypof = pof0 + warp * (DPW * 4);
        for (int s = 0; s < nstages; ++s) {
            const uint32_t sl = (uint32_t)(s % NSLOT), slot = 8u * sl;
            mbar_wait(full + slot, (uint32_t)((s / NSLOT) & 1));
            const uint4 po = *reinterpret_cast<const uint4 *>(mypof + sl * (DB * 4));
            const uint32_t pof[4] = {po.x, po.y, po.z, po.w};
#pragma unroll
            for (int k = 0; k < DPW; ++k) {
                const uint32_t *p = reinterpret_cast<const uint32_t *>(Pl + pof[k]);
                uint32_t v[NP];
#pragma unroll
                for (int i = 0; i < NP; ++i) v[i] = p[i * 32];
#pragma unroll
                for (int i = 0; i < NP; ++i) {
                    // low / high 16-bit lane of the row word into its own 32-bit accumulator (IDP.2A)
                    asm("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[k][2 * i]) : "r"(v[i]), "r"(0x00000001u));
                    asm("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc[k][2 * i + 1]) : "r"(v[i]), "r"(0x00000100u));
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + slot);
        }
#pragma unroll
        for (int k = 0; k < DPW; ++k) {
            const int d = d0 + warp * DPW + k;
            if (d >= a.ndms) continue;
            uint32_t *orow = a.out + (size_t)d * a.pitch_out + t0 + 2 * lane;
#pragma unroll
            for (int i = 0; i < NP; ++i) {
                const int64_t t = t0 + 2 * (lane + 32 * i);
                if (t + 1 < a.ncols) __stcg(reinterpret_cast<uint2 *>(orow + 64 * i), make_uint2(acc[k][2 * i], acc[k][2 * i + 1]));
                else if (t < a.ncols) __stcg(orow + 64 * i, acc[k][2 * i]);
            }
        }
        return;
    }
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
    const uint8_t *mypof = pof0 + warp * (DPW * 4);
    for (int s = 0; s < nstages; ++s) {
        const uint32_t sl = (uint32_t)(s % NSLOT), slot = 8u * sl;
        mbar_wait(full + slot, (uint32_t)((s / NSLOT) & 1));
        const uint4 po = *reinterpret_cast<const uint4 *>(mypof + sl * (DB * 4));

        // one row word per (trial, group, sample pair); eight loads in flight per batch.  A trial that reads the very
        // same row words as the previous one (same pattern, same offset: common with fine DM steps, 15-36 % of the
        // trials of cfg4's ranges) reuses the registers instead of loading again; the test is warp-uniform.
        const uint32_t pof[4] = {po.x, po.y, po.z, po.w};
#pragma unroll
        for (int h = 0; h < NP; h += 8) {
            uint32_t v[8];
#pragma unroll
            for (int k = 0; k < DPW; ++k) {
                if (k == 0 || pof[k] != pof[k - 1]) {
                    const uint32_t *p = reinterpret_cast<const uint32_t *>(Pl + pof[k]);
#pragma unroll
                    for (int i = 0; i < 8; ++i) v[i] = p[(h + i) * 32];
                }
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

template <int TB, bool IN16, bool WIDE = false>
cudaError_t launch_t(const DedispArgs &a, cudaStream_t st)
{
    dim3 grid((unsigned)((a.ndms + DB - 1) / DB), (unsigned)((a.ncols + TB - 1) / TB));
    dedisp_ws_kernel<TB, IN16, WIDE><<<grid, NT, dedisp_ws_smem_bytes(a.sp_rows, a.sp_pbytes), st>>>(a);
    return cudaGetLastError();
}

}  // namespace

size_t dedisp_ws_fixed_smem_bytes(int rows)
{
    return (size_t)NRAW * G * rows + (size_t)NPW * NRECBUF * REC + (size_t)NSLOT * DB * 4 + (NRAW + 2 * NSLOT) * 8 + 8;
}

size_t dedisp_ws_smem_bytes(int rows, int ring_bytes)
{
    return (size_t)ring_bytes + dedisp_ws_fixed_smem_bytes(rows);
}

cudaError_t dedisp_ws_configure()
{
    cudaError_t e = cudaFuncSetAttribute(dedisp_ws_kernel<1024, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(dedisp_ws_kernel<512, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(dedisp_ws_kernel<1024, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(dedisp_ws_kernel<512, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(dedisp_ws_kernel<512, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
}

cudaError_t launch_dedisp_ws(const DedispArgs &a, int tb, bool in16, bool wide, cudaStream_t st)
{
    if (a.ncols <= 0 || a.ndms <= 0) return cudaSuccess;
    if (wide) return launch_t<512, true, true>(a, st);                 // 32-bit accumulators (coarse bins)
    if (in16) return tb == 1024 ? launch_t<1024, true>(a, st) : launch_t<512, true>(a, st);
    return tb == 1024 ? launch_t<1024, false>(a, st) : launch_t<512, false>(a, st);
}

}  // namespace aa
