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
    return dpw == 4 ? smem_bytes_t<uint8_t, 4, CS8>(row)
           : dpw == 2 ? smem_bytes_t<uint8_t, 2, CS8>(row)
                      : smem_bytes_t<uint8_t, 1, CS8>(row);
}

cudaError_t dedisp_configure()
{
    const int maxb = 227 * 1024;
    cudaError_t e;
#define AA_CFG(T, D, C)                                                                                    \
    e = cudaFuncSetAttribute(dedisp_kernel<T, D, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, maxb); \
    if (e != cudaSuccess) return e;
    AA_CFG(uint8_t, 4, CS8) AA_CFG(uint8_t, 2, CS8) AA_CFG(uint8_t, 1, CS8)
    AA_CFG(uint16_t, 4, CS16) AA_CFG(uint16_t, 2, CS16) AA_CFG(uint16_t, 1, CS16)
#undef AA_CFG
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
    return dpw == 4 ? launch_t<uint8_t, 4, CS8>(a, st)
           : dpw == 2 ? launch_t<uint8_t, 2, CS8>(a, st)
                      : launch_t<uint8_t, 1, CS8>(a, st);
}

}  // namespace aa
