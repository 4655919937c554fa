// Brute-force incoherent dedispersion (BASELINE.json north_star):
//     D[d][tau] = sum_c y[c][tau + delta(c,d)],   exact unsigned integer sums.
//
// One CTA produces a tile of DB DM trials x 512 output samples.  Channels are processed in stages
// of CS rows.  For each stage one warp issues 1-D bulk async copies (cp.async.bulk, mbarrier
// completion) of every row's window [t0 + delta(c,d0) & ~15, +ROW) into a double-buffered staging
// area; all threads then expand the staged samples into two 16-bit-lane copies per row
//     E[i] = (y[2i], y[2i+1])     O[i] = (y[2i+1], y[2i+2])
// so that for ANY integer delay a thread can fetch two consecutive output samples with one
// aligned 32-bit shared load, and add two channels' worth with one 3-input integer add (SWAR:
// two 16-bit sums per register).  16-bit lanes are flushed into 32-bit accumulators before they
// can overflow (every floor(65535/(255*bin)) channels).  No tensor cores: this is a gather-add,
// not a dense contraction.
//
// Roofline: shared-memory bandwidth (one 32-bit LDS per two sample-adds) and the integer ALU;
// HBM traffic is only the final 4 B per output sample, the input windows come from L2.
#include "aa_internal.h"

namespace aa {

namespace {

constexpr int TB = kDedispTB;          // output samples per CTA
constexpr int NT = kDedispThreads;     // threads per CTA
constexpr int NW = NT / 32;            // warps
constexpr int NP = TB / 2 / 32;        // 16-bit-pair words per lane (8)

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
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "DONE:\n\t}" ::"r"(smem_u32(bar)),
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

// acc += x on the FMA pipe: IMAD acc = x * one + acc with a run-time multiplier of 1.  The ALU pipe
// (64 lanes/clk/SM) is busy with the byte unpacking; integer multiply-add issues on the other pipe.
__device__ __forceinline__ void fma_add(uint32_t &acc, uint32_t x, uint32_t one)
{
    asm("mad.lo.u32 %0, %1, %2, %0;" : "+r"(acc) : "r"(x), "r"(one));
}

template <int N>
struct OffVec;
template <>
struct OffVec<4> { using type = uint4; };
template <>
struct OffVec<2> { using type = uint2; };
template <>
struct OffVec<1> { using type = uint32_t; };

template <int DPW>
__device__ __forceinline__ void load_offsets(const uint32_t *p, uint32_t (&o)[DPW])
{
    typename OffVec<DPW>::type v = *reinterpret_cast<const typename OffVec<DPW>::type *>(p);
    const uint32_t *q = reinterpret_cast<const uint32_t *>(&v);
#pragma unroll
    for (int k = 0; k < DPW; ++k) o[k] = q[k];
}

// Expand 8 staged samples (+ the one after) into 4 E words and 4 O words.
// O_k = (y[2k+1], y[2k+2]) = high half of E_k | low half of E_{k+1}: one funnel shift each.
__device__ __forceinline__ void odd_from_even(const uint4 &e, uint32_t next, uint4 &o)
{
    o.x = __funnelshift_r(e.x, e.y, 16);
    o.y = __funnelshift_r(e.y, e.z, 16);
    o.z = __funnelshift_r(e.z, e.w, 16);
    o.w = __funnelshift_r(e.w, next, 16);
}
__device__ __forceinline__ void expand8(const uint8_t *s, uint4 &e, uint4 &o)
{
    uint2 v = *reinterpret_cast<const uint2 *>(s);
    e.x = __byte_perm(v.x, 0, 0x4140);  // (b0, b1)
    e.y = __byte_perm(v.x, 0, 0x4342);  // (b2, b3)
    e.z = __byte_perm(v.y, 0, 0x4140);
    e.w = __byte_perm(v.y, 0, 0x4342);
    odd_from_even(e, (uint32_t)s[8], o);
}
__device__ __forceinline__ void expand8(const uint16_t *s, uint4 &e, uint4 &o)
{
    e = *reinterpret_cast<const uint4 *>(s);
    odd_from_even(e, (uint32_t)s[8], o);
}

template <typename IN_T, int DPW, int CS>
__global__ void __launch_bounds__(NT, 2) dedisp_kernel(const DedispArgs a)
{
    constexpr int DB = DPW * NW;
    extern __shared__ __align__(128) uint8_t smem[];
    const int ROW = a.row;            // staged samples per row
    const int ROWW = ROW / 2;         // words per parity copy
    uint32_t *eo = reinterpret_cast<uint32_t *>(smem);                                   // [CS][2][ROWW]
    uint8_t *stg0 = smem + (size_t)CS * ROW * 4;
    const size_t stg_bytes = (size_t)CS * ROW * sizeof(IN_T) + 16;
    uint32_t *soff = reinterpret_cast<uint32_t *>(stg0 + 2 * stg_bytes);                 // [CS][DB]
    uint64_t *bar = reinterpret_cast<uint64_t *>(soff + CS * DB);                        // [2]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d0 = blockIdx.x * DB;
    const int64_t t0 = (int64_t)blockIdx.y * TB;
    const int nchans = a.nchans;
    const int nstages = (nchans + CS - 1) / CS;
    const IN_T *in = static_cast<const IN_T *>(a.in);
    const int32_t *dly0 = a.delays + (size_t)d0 * nchans;   // delays of the block's first trial

    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto issue = [&](int s, int buf) {   // warp 0
        const int c = s * CS + lane;
        int nvalid = nchans - s * CS;
        if (nvalid > CS) nvalid = CS;
        if (lane == 0) mbar_expect_tx(&bar[buf], (uint32_t)(nvalid * ROW * sizeof(IN_T)));
        if (lane < CS && c < nchans) {
            const int base = dly0[c] & ~(kAlign - 1);
            const IN_T *src = in + (size_t)c * a.pitch_in + a.col0 + t0 + base;
            bulk_g2s(stg0 + buf * stg_bytes + (size_t)lane * ROW * sizeof(IN_T), src,
                     (uint32_t)(ROW * sizeof(IN_T)), &bar[buf]);
        }
    };

    uint32_t acc16[DPW][NP];
    uint32_t acc32[DPW][2 * NP];
#pragma unroll
    for (int k = 0; k < DPW; ++k) {
#pragma unroll
        for (int i = 0; i < NP; ++i) acc16[k][i] = 0;
#pragma unroll
        for (int i = 0; i < 2 * NP; ++i) acc32[k][i] = 0;
    }
    int since_flush = 0;

    auto flush = [&]() {
#pragma unroll
        for (int k = 0; k < DPW; ++k)
#pragma unroll
            for (int i = 0; i < NP; ++i) {
                acc32[k][2 * i] += acc16[k][i] & 0xFFFFu;
                acc32[k][2 * i + 1] += acc16[k][i] >> 16;
                acc16[k][i] = 0;
            }
    };

    if (warp == 0) issue(0, 0);

    for (int s = 0; s < nstages; ++s) {
        const int buf = s & 1;
        if (warp == 0 && s + 1 < nstages) issue(s + 1, buf ^ 1);

        // per-(channel, trial) shared-memory byte offsets of this stage
        for (int e = tid; e < CS * DB; e += NT) {
            const int cl = e % CS, dl = e / CS;
            const int c = s * CS + cl;
            uint32_t off = (uint32_t)(cl * 2 * ROWW) * 4u;
            if (c < nchans) {
                int d = d0 + dl;
                if (d > a.ndms - 1) d = a.ndms - 1;
                const int rel = a.delays[(size_t)d * nchans + c] - (dly0[c] & ~(kAlign - 1));
                off = (uint32_t)((cl * 2 + (rel & 1)) * ROWW + (rel >> 1)) * 4u;
            }
            soff[cl * DB + dl] = off;
        }

        mbar_wait(&bar[buf], (uint32_t)((s >> 1) & 1));

        // expand staged samples into the E / O copies
        {
            const IN_T *stg = reinterpret_cast<const IN_T *>(stg0 + buf * stg_bytes);
            const int tasks_per_row = ROW / 8;
            for (int task = tid; task < CS * tasks_per_row; task += NT) {
                const int cl = task / tasks_per_row, k = task - cl * tasks_per_row;
                uint4 e, o;
                if (s * CS + cl < nchans) {
                    expand8(stg + (size_t)cl * ROW + k * 8, e, o);
                } else {
                    e = make_uint4(0, 0, 0, 0);
                    o = e;
                }
                uint32_t *dst = eo + (size_t)cl * 2 * ROWW + k * 4;
                *reinterpret_cast<uint4 *>(dst) = e;
                *reinterpret_cast<uint4 *>(dst + ROWW) = o;
            }
        }
        __syncthreads();

        // accumulate: two channels per step so that one IADD3 adds both
        {
            const uint8_t *eob = reinterpret_cast<const uint8_t *>(eo) + lane * 4;
#pragma unroll 2
            for (int cp = 0; cp < CS; cp += 2) {
                uint32_t o0[DPW], o1[DPW];
                load_offsets<DPW>(soff + cp * DB + warp * DPW, o0);
                load_offsets<DPW>(soff + (cp + 1) * DB + warp * DPW, o1);
#pragma unroll
                for (int k = 0; k < DPW; ++k) {
                    const uint32_t *p0 = reinterpret_cast<const uint32_t *>(eob + o0[k]);
                    const uint32_t *p1 = reinterpret_cast<const uint32_t *>(eob + o1[k]);
#pragma unroll
                    for (int i = 0; i < NP; ++i) acc16[k][i] += p0[i * 32] + p1[i * 32];
                }
                since_flush += 2;
                if (since_flush >= a.flush_ch) {
                    flush();
                    since_flush = 0;
                }
            }
        }
        __syncthreads();
    }
    flush();

    // epilogue: 32-bit sums, two consecutive samples per 8-byte store
#pragma unroll
    for (int k = 0; k < DPW; ++k) {
        const int d = d0 + warp * DPW + k;
        if (d >= a.ndms) continue;
        uint32_t *orow = a.out + (size_t)d * a.pitch_out;
#pragma unroll
        for (int i = 0; i < NP; ++i) {
            const int64_t t = t0 + 2 * (lane + 32 * i);
            if (t + 1 < a.ncols) {
                *reinterpret_cast<uint2 *>(orow + t) = make_uint2(acc32[k][2 * i], acc32[k][2 * i + 1]);
            } else if (t < a.ncols) {
                orow[t] = acc32[k][2 * i];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// uint8 input, 8-bit staging ("U8" path).  The 16-bit-lane kernel above is bound by shared-memory
// bandwidth (2 B of LDS per sample-add, 86 % of the pipe in profiles/r1_dedisp_ncu.txt).  Here a
// row stays 1 B per sample in shared memory: the staged row itself is "copy 0" and the expand step
// writes three more copies shifted by 1, 2 and 3 bytes, so a word-aligned 32-bit LDS returns four
// consecutive samples for ANY delay (copy = delay & 3, word = delay >> 2).  A thread owns quads
// of output samples; each loaded word is split into its even bytes (LOP3) and odd bytes (PRMT),
// i.e. two registers of two 16-bit lanes, and added to the quad's two accumulators.  That is 1 B
// of LDS and 1.25 issue slots per sample-add instead of 2 B and 0.75: the bound moves from the
// shared-memory pipe to instruction issue, with the adds shared between the ALU and FMA pipes.
template <int DPW, int CS>
__global__ void __launch_bounds__(NT, 2) dedisp_u8_kernel(const DedispArgs a)
{
    constexpr int DB = DPW * NW;
    constexpr int NQ = TB / 4 / 32;               // quads per lane (4)
    static_assert(DB <= 32 && CS == 16, "one delay-tile row per lane of warp 0; two staged rows per warp");
    extern __shared__ __align__(128) uint8_t smem[];
    const int ROW = a.row;
    const size_t stg_bytes = (size_t)CS * ROW + 16;
    uint8_t *stg0 = smem;                                           // [2][CS][ROW] (+16): copy 0
    uint8_t *cpy = smem + 2 * stg_bytes;                            // [3][CS][ROW]: copies 1..3
    uint32_t *soff = reinterpret_cast<uint32_t *>(cpy + (size_t)3 * CS * ROW);   // [CS][DB]
    int32_t *dtile = reinterpret_cast<int32_t *>(soff + CS * DB);   // [3][DB][CS] delays of a stage
    uint64_t *bar = reinterpret_cast<uint64_t *>(dtile + 3 * DB * CS);           // [3]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d0 = blockIdx.x * DB;
    const int64_t t0 = (int64_t)blockIdx.y * TB;
    const int nchans = a.nchans;
    const int nstages = (nchans + CS - 1) / CS;
    const uint8_t *in = static_cast<const uint8_t *>(a.in);

    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_init(&bar[2], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // Delay tile of stage s: one contiguous [DB][CS] block of the tiled delay table (trials clamped,
    // channels past nchans zero): a single 2 KB bulk copy.
    const int32_t *tiles = a.dtiles + (size_t)blockIdx.x * nstages * (DB * CS);
    // Rows of stage s (window base from the tile's first trial): every warp issues its own CS/NW rows,
    // so no warp serialises 16 copies; thread 0 arms the barrier and adds the delay tile of stage s+1.
    auto issue_rows = [&](int s, int buf) {
        if (tid == 0) {
            int nvalid = nchans - s * CS;
            if (nvalid > CS) nvalid = CS;
            const bool next_tile = s + 1 < nstages;
            mbar_expect_tx(&bar[buf], (uint32_t)(nvalid * ROW) + (next_tile ? DB * CS * 4 : 0));
            if (next_tile) bulk_g2s(dtile + ((s + 1) % 3) * DB * CS, tiles + (size_t)(s + 1) * DB * CS, DB * CS * 4, &bar[buf]);
        }
        if (lane < CS / NW) {
            const int cl = warp * (CS / NW) + lane, c = s * CS + cl;
            if (c < nchans) {
                const int base = dtile[(s % 3) * DB * CS + cl] & ~(kAlign - 1);
                const uint8_t *src = in + (size_t)c * a.pitch_in + a.col0 + t0 + base;
                bulk_g2s(stg0 + buf * stg_bytes + (size_t)cl * ROW, src, (uint32_t)ROW, &bar[buf]);
            }
        }
    };

    // one exact 32-bit accumulator per output sample: no 16-bit lanes, no flush, any channel count
    uint32_t acc[DPW][4 * NQ];
#pragma unroll
    for (int k = 0; k < DPW; ++k)
#pragma unroll
        for (int i = 0; i < 4 * NQ; ++i) acc[k][i] = 0;

    // prologue: tile 0 (own barrier), then rows 0 + tile 1
    if (tid == 0) {
        mbar_expect_tx(&bar[2], DB * CS * 4);
        bulk_g2s(dtile, tiles, DB * CS * 4, &bar[2]);
    }
    mbar_wait(&bar[2], 0);
    issue_rows(0, 0);

    for (int s = 0; s < nstages; ++s) {
        const int buf = s & 1;
        uint8_t *stg = stg0 + buf * stg_bytes;

        mbar_wait(&bar[buf], (uint32_t)((s >> 1) & 1));              // rows(s) and tile(s+1) have landed
        if (s + 1 < nstages) issue_rows(s + 1, buf ^ 1);

        // shared-memory byte offset of (channel, trial): copy (delay & 3), word (delay >> 2)
        {
            const uint32_t stg_off = (uint32_t)(stg - smem), cpy_off = (uint32_t)(cpy - smem);
            const int32_t *dt = dtile + (s % 3) * DB * CS;
            for (int e = tid; e < CS * DB; e += NT) {
                const int cl = e % CS, dl = e / CS;
                uint32_t off = cpy_off + (uint32_t)(cl * ROW);      // rows past nchans: zero-filled copy 1
                if (s * CS + cl < nchans) {
                    const int rel = dt[dl * CS + cl] - (dt[cl] & ~(kAlign - 1));
                    const int sh = rel & 3;
                    off = (sh == 0 ? stg_off + (uint32_t)(cl * ROW)
                                   : cpy_off + (uint32_t)(((sh - 1) * CS + cl) * ROW)) + (uint32_t)(rel >> 2) * 4u;
                }
                soff[cl * DB + dl] = off;
            }
        }

        // expand: copies shifted by 1, 2, 3 bytes; warp w owns rows 2w and 2w+1, 16 samples per task
        {
            const int tasks_per_row = ROW / 16;
#pragma unroll
            for (int rr = 0; rr < CS / NW; ++rr) {
                const int cl = warp * (CS / NW) + rr;
                const bool live = s * CS + cl < nchans;
                for (int k = lane; k < tasks_per_row; k += 32) {
                    uint4 c1, c2, c3;
                    if (live) {
                        const uint8_t *src = stg + (size_t)cl * ROW + k * 16;
                        const uint4 v = *reinterpret_cast<const uint4 *>(src);
                        const uint32_t nx = *reinterpret_cast<const uint32_t *>(src + 16);
                        c1 = make_uint4(__funnelshift_r(v.x, v.y, 8), __funnelshift_r(v.y, v.z, 8),
                                        __funnelshift_r(v.z, v.w, 8), __funnelshift_r(v.w, nx, 8));
                        c2 = make_uint4(__funnelshift_r(v.x, v.y, 16), __funnelshift_r(v.y, v.z, 16),
                                        __funnelshift_r(v.z, v.w, 16), __funnelshift_r(v.w, nx, 16));
                        c3 = make_uint4(__funnelshift_r(v.x, v.y, 24), __funnelshift_r(v.y, v.z, 24),
                                        __funnelshift_r(v.z, v.w, 24), __funnelshift_r(v.w, nx, 24));
                    } else {
                        c1 = c2 = c3 = make_uint4(0, 0, 0, 0);
                    }
                    uint8_t *dst = cpy + (size_t)cl * ROW + k * 16;
                    *reinterpret_cast<uint4 *>(dst) = c1;
                    *reinterpret_cast<uint4 *>(dst + (size_t)CS * ROW) = c2;
                    *reinterpret_cast<uint4 *>(dst + (size_t)2 * CS * ROW) = c3;
                }
            }
        }
        __syncthreads();

        {
            const uint8_t *sb = smem + lane * 4;
#pragma unroll 2
            for (int cp = 0; cp < CS; cp += 2) {
                uint32_t o0[DPW], o1[DPW];
                load_offsets<DPW>(soff + cp * DB + warp * DPW, o0);
                load_offsets<DPW>(soff + (cp + 1) * DB + warp * DPW, o1);
#pragma unroll
                for (int k = 0; k < DPW; ++k) {
                    const uint32_t *p0 = reinterpret_cast<const uint32_t *>(sb + o0[k]);
                    const uint32_t *p1 = reinterpret_cast<const uint32_t *>(sb + o1[k]);
#pragma unroll
                    for (int i = 0; i < NQ; ++i) {
                        const uint32_t w0 = p0[i * 32], w1 = p1[i * 32];
                        // interleave the two channels' bytes (PRMT, ALU pipe), then one dp4a per output
                        // sample adds both channels into its 32-bit accumulator (IDP4A, FMA pipe):
                        // 2 LDS + 2 PRMT + 4 IDP4A per 8 sample-adds
                        const uint32_t lo = __byte_perm(w0, w1, 0x5140);   // (a0, b0, a1, b1)
                        const uint32_t hi = __byte_perm(w0, w1, 0x7362);   // (a2, b2, a3, b3)
                        acc[k][4 * i + 0] = __dp4a(lo, 0x00000101u, acc[k][4 * i + 0]);
                        acc[k][4 * i + 1] = __dp4a(lo, 0x01010000u, acc[k][4 * i + 1]);
                        acc[k][4 * i + 2] = __dp4a(hi, 0x00000101u, acc[k][4 * i + 2]);
                        acc[k][4 * i + 3] = __dp4a(hi, 0x01010000u, acc[k][4 * i + 3]);
                    }
                }
            }
        }
        __syncthreads();
    }

#pragma unroll
    for (int k = 0; k < DPW; ++k) {
        const int d = d0 + warp * DPW + k;
        if (d >= a.ndms) continue;
        uint32_t *orow = a.out + (size_t)d * a.pitch_out;
#pragma unroll
        for (int i = 0; i < NQ; ++i) {
            const int64_t t = t0 + 4 * (lane + 32 * i);
            if (t + 3 < a.ncols) {
                *reinterpret_cast<uint4 *>(orow + t) =
                    make_uint4(acc[k][4 * i], acc[k][4 * i + 1], acc[k][4 * i + 2], acc[k][4 * i + 3]);
            } else {
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (t + j < a.ncols) orow[t + j] = acc[k][4 * i + j];
            }
        }
    }
}

template <int DPW, int CS>
size_t smem_bytes_u8(int row)
{
    return 2 * ((size_t)CS * row + 16) + (size_t)3 * CS * row + (size_t)CS * DPW * NW * 4 * 4 + 32;
}

template <int DPW, int CS>
cudaError_t launch_u8(const DedispArgs &a, cudaStream_t st)
{
    constexpr int DB = DPW * NW;
    dim3 grid((unsigned)((a.ndms + DB - 1) / DB), (unsigned)((a.ncols + TB - 1) / TB));
    dedisp_u8_kernel<DPW, CS><<<grid, NT, smem_bytes_u8<DPW, CS>(a.row), st>>>(a);
    return cudaGetLastError();
}

template <typename IN_T, int DPW, int CS>
size_t smem_bytes_t(int row)
{
    return (size_t)CS * row * 4 + 2 * ((size_t)CS * row * sizeof(IN_T) + 16) + (size_t)CS * DPW * NW * 4 + 16;
}

template <typename IN_T, int DPW, int CS>
cudaError_t launch_t(const DedispArgs &a, cudaStream_t st)
{
    constexpr int DB = DPW * NW;
    dim3 grid((unsigned)((a.ndms + DB - 1) / DB), (unsigned)((a.ncols + TB - 1) / TB));
    dedisp_kernel<IN_T, DPW, CS><<<grid, NT, smem_bytes_t<IN_T, DPW, CS>(a.row), st>>>(a);
    return cudaGetLastError();
}

constexpr int CS8 = 16;    // channels per stage, uint8 input
constexpr int CS16 = 8;    // channels per stage, uint16 input

}  // namespace

int dedisp_stage_channels(bool in16) { return in16 ? CS16 : CS8; }

size_t dedisp_smem_bytes(bool in16, int dpw, int row)
{
    if (in16) {
        return dpw == 4 ? smem_bytes_t<uint16_t, 4, CS16>(row)
               : dpw == 2 ? smem_bytes_t<uint16_t, 2, CS16>(row)
                          : smem_bytes_t<uint16_t, 1, CS16>(row);
    }
    return dpw == 4 ? smem_bytes_u8<4, CS8>(row)
           : dpw == 2 ? smem_bytes_u8<2, CS8>(row)
                      : smem_bytes_u8<1, CS8>(row);
}

cudaError_t dedisp_configure()
{
    const int maxb = 227 * 1024;
    cudaError_t e;
#define AA_CFG(T, D, C)                                                                                    \
    e = cudaFuncSetAttribute(dedisp_kernel<T, D, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, maxb); \
    if (e != cudaSuccess) return e;
    AA_CFG(uint16_t, 4, CS16) AA_CFG(uint16_t, 2, CS16) AA_CFG(uint16_t, 1, CS16)
#undef AA_CFG
#define AA_CFG8(D, C)                                                                                    \
    e = cudaFuncSetAttribute(dedisp_u8_kernel<D, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, maxb); \
    if (e != cudaSuccess) return e;
    AA_CFG8(4, CS8) AA_CFG8(2, CS8) AA_CFG8(1, CS8)
#undef AA_CFG8
    return cudaSuccess;
}

cudaError_t launch_dedisp(const DedispArgs &a, bool in16, int dpw, cudaStream_t st)
{
    if (a.ncols <= 0 || a.ndms <= 0) return cudaSuccess;
    if (in16) {
        return dpw == 4 ? launch_t<uint16_t, 4, CS16>(a, st)
               : dpw == 2 ? launch_t<uint16_t, 2, CS16>(a, st)
                          : launch_t<uint16_t, 1, CS16>(a, st);
    }
    return dpw == 4 ? launch_u8<4, CS8>(a, st)
           : dpw == 2 ? launch_u8<2, CS8>(a, st)
                      : launch_u8<1, CS8>(a, st);
}

}  // namespace aa
