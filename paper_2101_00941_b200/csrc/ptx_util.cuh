// PTX wrappers shared by the warp-specialised dedispersion kernels (kernels_dedisp_ws.cu, kernels_dedisp_g8.cu):
// mbarrier, 1-D bulk copies (TMA), cp.async, tensor-memory loads/stores, dp2a.  One-line restatements of the ISA.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace aa {
namespace ptx {

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
constexpr uint32_t kSuspendNs = 20000;   // try_wait may park the thread this long; arrival wakes it earlier
// mbarriers are addressed by their 32-bit shared-window address
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity), "r"(kSuspendNs)
        : "memory");
    return ok != 0;
}
// Whole-warp wait: every lane observes the completed phase itself (acquire), and the lanes leave the
// loop together, so the warp stays converged (lanes leaving one by one would split it for good).
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!__all_sync(0xFFFFFFFFu, mbar_try(bar, parity))) {
    }
}
// single-lane wait (inside a lane-0 section)
__device__ __forceinline__ void mbar_wait_lane(uint32_t bar, uint32_t parity)
{
    while (!mbar_try(bar, parity)) {
    }
}
__device__ __forceinline__ void sts128_if(uint32_t addr, uint32_t x, uint32_t y, uint32_t z, uint32_t w, uint32_t pred)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.u32 p, %5, 0;\n\t"
        "@p st.shared.v4.u32 [%0], {%1, %2, %3, %4};\n\t}" ::"r"(addr),
        "r"(x), "r"(y), "r"(z), "r"(w), "r"(pred)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// byte 0 / 2 of x times 1 plus byte 1 / 3 times 2^15: two samples into two 15-bit lanes (IDP.2A)
__device__ __forceinline__ void dp2a_lo(uint32_t &acc, uint32_t x)
{
    asm("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(acc) : "r"(0x80000001u), "r"(x));
}
__device__ __forceinline__ void dp2a_hi(uint32_t &acc, uint32_t x)
{
    asm("dp2a.hi.u32.u32 %0, %1, %2, %0;" : "+r"(acc) : "r"(0x80000001u), "r"(x));
}

// ---- tensor memory (TMEM) as the second-level accumulator -------------------------------------------------
// The 256 KB of TMEM of the SM hold the CTA's uint32 output tile (64 trials x 1024 samples): the 16-bit lanes
// are flushed into it with tcgen05.ld / add / tcgen05.st (on-chip, ~12 cycles) instead of a read-modify-write
// of the tile in L2.  A warp reaches the 32 TMEM lanes of its quadrant (warp % 4), one lane per thread
// (shape 32x32b: register j of thread t <-> TMEM lane base + t, column + j).
__device__ __forceinline__ void tmem_ld8(uint32_t (&v)[8], uint32_t taddr)
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr)
                 : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&v)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(v[0]), "r"(v[1]),
                 "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
                 : "memory");
}

__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}

}  // namespace ptx
}  // namespace aa
