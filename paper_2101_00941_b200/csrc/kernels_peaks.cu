// Peak finding on the device (reading A17): thins a sub-chunk's candidate list before it
// crosses the host link.  Two candidates are neighbours if their DM indices differ by at most 1 and their boxcars
// overlap or touch in raw samples (t' <= t + w and t <= t' + w'); a candidate is a peak iff no neighbour has a larger
// S/N (the stored float), ties going to the smaller (dm_index, t_start).
//
// The list is unordered (warp-aggregated appends), so it is first threaded onto a grid of buckets (DM row, 2^shift raw
// samples): head[row][bucket] -> next[] chains, one atomicExch per candidate.  Each candidate then walks the buckets of
// rows dm-1 .. dm+1 that can hold a neighbour.  A candidate whose neighbourhood reaches into the previous or the next
// sub-chunk ("border") cannot be decided here: it goes to the host with its flags, beaten or not, because it may still
// beat a candidate of the other sub-chunk; the host settles the borders on the merged list (aa_host.cu).  Everything
// else that is beaten stays on the device.  The rule is the oracle's, candidate by candidate; no clustering.
#include "aa_internal.h"

namespace aa {

namespace {

__global__ void __launch_bounds__(256) peaks_link_kernel(const PeakArgs a)
{
    const uint32_t n = min(*a.count, a.cap);
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const aa_candidate c = a.cands[i];
        const uint32_t b = (c.t_start - a.t0) >> a.shift;
        a.next[i] = (uint32_t)atomicExch(&a.head[(size_t)c.dm_index * a.nbk + b], (int32_t)i);
    }
}

__device__ __forceinline__ bool beats(const aa_candidate &x, const aa_candidate &c)    // x beats c
{
    if (x.snr != c.snr) return x.snr > c.snr;
    if (x.dm_index != c.dm_index) return x.dm_index < c.dm_index;
    return x.t_start < c.t_start;
}

__global__ void __launch_bounds__(256) peaks_decide_kernel(const PeakArgs a)
{
    const uint32_t n = min(*a.count, a.cap);
    const uint32_t lane = threadIdx.x & 31;
    // whole warps iterate together so that the append can be warp-aggregated
    for (uint32_t i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31u; i0 < n; i0 += gridDim.x * blockDim.x) {
        const uint32_t i = i0 + lane;
        bool emit = false;
        aa_candidate c{};
        if (i < n) {
            c = a.cands[i];
            const uint32_t t = c.t_start, te = t + c.width;                    // neighbours start in [t - wmax, te]
            const uint32_t lo_t = t > a.t0 + a.wmax_raw ? t - a.wmax_raw : a.t0;
            const uint32_t hi_t = te < a.t1 ? te : a.t1 - 1;
            const uint32_t b_lo = (lo_t - a.t0) >> a.shift, b_hi = (hi_t - a.t0) >> a.shift;
            bool beaten = false;
            for (int dd = -1; dd <= 1 && !beaten; ++dd) {
                const int64_t row = (int64_t)c.dm_index + dd;
                if (row < 0 || row >= a.nrows) continue;
                const int32_t *h = a.head + (size_t)row * a.nbk;
                for (uint32_t b = b_lo; b <= b_hi && !beaten; ++b) {
                    for (int32_t k = h[b]; k >= 0; k = (int32_t)a.next[k]) {
                        if ((uint32_t)k == i) continue;
                        const aa_candidate x = a.cands[k];
                        if (x.t_start <= te && t <= x.t_start + x.width && beats(x, c)) { beaten = true; break; }
                    }
                }
            }
            // a neighbour may sit in the next sub-chunk (it starts at or before te) or in the previous one (its boxcar,
            // at most wmax_raw long, reaches t)
            const bool border = (a.has_right && te >= a.t1) || (a.has_left && t < a.t0 + a.wmax_raw);
            emit = !beaten || border;
            c.dm_index |= (beaten ? 0x80000000u : 0u) | (border ? 0x40000000u : 0u);
        }
        const unsigned mask = __ballot_sync(0xffffffffu, emit);
        if (mask) {
            uint32_t base = 0;
            const int leader = __ffs(mask) - 1;
            if ((int)lane == leader) base = atomicAdd(a.out_count, (uint32_t)__popc(mask));
            base = __shfl_sync(0xffffffffu, base, leader);
            if (emit) {
                const uint32_t slot = base + __popc(mask & ((1u << lane) - 1));
                if (slot < a.out_cap) a.out[slot] = c;
            }
        }
    }
}

}  // namespace

cudaError_t launch_peaks(const PeakArgs &a, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(a.head, 0xFF, (size_t)a.nrows * a.nbk * sizeof(int32_t), st);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(a.out_count, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    peaks_link_kernel<<<148 * 2, 256, 0, st>>>(a);
    peaks_decide_kernel<<<148 * 4, 256, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace aa
