// aa_find_peaks_device_noalloc: peak finding (reading A17) on a candidate list that is already in device memory, for
// callers that may not allocate device memory while they run.
//
// Who that is.  Two kinds of caller in practice.  (1) A real-time ingest loop in its streamed phase: cudaMalloc and
// cudaFree wait for the whole device, so one allocation made between two sub-chunks stalls every other stream's copy
// and kernel and the overlap the pipeline lives on is gone (the paper allocates everything before the loop for this
// reason, PAPER.md:41 steps 1-2, :71).  (2) A process that has handed all device memory to one owner (a framework's
// caching pool, a fixed arena carved at start-up): a raw cudaMalloc made behind that owner's back fails or
// fragments what is left.  Both can still pass buffers they already own, which is all this call asks for.
//
// The peak kernels of kernels_peaks.cu thread the list onto a grid of buckets (DM row x 2^shift raw samples) and walk
// the neighbouring buckets of every record.  That grid (`head`) and the chain (`next`) are scratch memory; aa_run takes
// them from the plan's arena.  Here they live in ONE file-scope __device__ array of fixed size, part of the library
// image: every GPU that loads libaa.so holds these 8 MiB until the process exits, whether this entry point is ever
// called or not.  Limits, stated in aa.h: at most AA_PEAKS_NOALLOC_MAX_CANDS records and AA_PEAKS_NOALLOC_MAX_CELLS
// bucket cells per call; larger requests are refused with AA_ERR_LIMIT, never served from a hidden allocation.
//
// Host code cannot use the array's name as a pointer (on the host the name is only a handle for the symbol, not a device
// address), so the device address is looked up with cudaGetSymbolAddress, once per device, by the first call made
// with that device current; the kernels receive that address as an ordinary argument.
//
// All calls on one device share the array and it keeps whatever the last call left in it.  Every call therefore
// resets the cells it is about to use (on the caller's stream, before its kernels) and relies on nothing else; two
// calls that may run on the GPU at the same time (different streams without an ordering between them, or different host
// threads) would overwrite each other's grid: the caller must order them.
//
// The kernels below are variants of peaks_link_kernel / peaks_decide_kernel written for a stand-alone list (count by
// value, no sub-chunk borders, records outside the declared ranges ignored); the existing path is not touched.
#include <algorithm>
#include <mutex>

#include "aa_internal.h"

namespace {

constexpr uint32_t kMaxCands = AA_PEAKS_NOALLOC_MAX_CANDS;
constexpr uint32_t kMaxCells = AA_PEAKS_NOALLOC_MAX_CELLS;
constexpr int kMaxDevices = 64;

// [0, kMaxCells): int32 head of each bucket's chain (-1 = empty); [kMaxCells, kMaxCells + kMaxCands): uint32 next
static __device__ __align__(256) uint32_t g_peaks_scratch[(size_t)kMaxCells + kMaxCands];

struct NoallocArgs {
    const aa_candidate *cands;
    uint32_t n;
    int32_t *head;                 // [nrows][nbk]
    uint32_t *next;                // [n]
    uint32_t nrows, nbk, shift;
    uint32_t t_end;                // candidates start in [0, t_end)
    uint32_t wmax;                 // longest boxcar, raw samples
    aa_candidate *out;
    uint32_t *out_count;
    uint32_t out_cap;
};

__device__ __forceinline__ bool in_range(const aa_candidate &c, const NoallocArgs &a)
{
    return c.dm_index < a.nrows && c.t_start < a.t_end;
}

__global__ void __launch_bounds__(256) peaks_noalloc_link_kernel(const NoallocArgs a)
{
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += gridDim.x * blockDim.x) {
        const aa_candidate c = a.cands[i];
        if (!in_range(c, a)) continue;                          // never linked: not a peak, not a neighbour
        a.next[i] = (uint32_t)atomicExch(&a.head[(size_t)c.dm_index * a.nbk + (c.t_start >> a.shift)], (int32_t)i);
    }
}

__device__ __forceinline__ bool beats(const aa_candidate &x, const aa_candidate &c)    // x beats c
{
    if (x.snr != c.snr) return x.snr > c.snr;
    if (x.dm_index != c.dm_index) return x.dm_index < c.dm_index;
    return x.t_start < c.t_start;
}

__global__ void __launch_bounds__(256) peaks_noalloc_decide_kernel(const NoallocArgs a)
{
    const uint32_t lane = threadIdx.x & 31;
    // whole warps iterate together: the append below is one atomicAdd per warp
    for (uint32_t i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31u; i0 < a.n; i0 += gridDim.x * blockDim.x) {
        const uint32_t i = i0 + lane;
        bool emit = false;
        aa_candidate c{};
        if (i < a.n) {
            c = a.cands[i];
            if (in_range(c, a)) {
                // a neighbour x has x.t_start <= t + w and t <= x.t_start + x.width, so it starts in [t - wmax, t + w]
                const uint64_t te = (uint64_t)c.t_start + c.width;
                const uint32_t lo_t = c.t_start > a.wmax ? c.t_start - a.wmax : 0;
                const uint32_t hi_t = te < a.t_end ? (uint32_t)te : a.t_end - 1;
                const uint32_t b_lo = lo_t >> a.shift, b_hi = hi_t >> a.shift;
                bool beaten = false;
                for (int dd = -1; dd <= 1 && !beaten; ++dd) {
                    const int64_t row = (int64_t)c.dm_index + dd;
                    if (row < 0 || row >= (int64_t)a.nrows) continue;
                    const int32_t *h = a.head + (size_t)row * a.nbk;
                    for (uint32_t b = b_lo; b <= b_hi && !beaten; ++b) {
                        for (int32_t k = h[b]; k >= 0; k = (int32_t)a.next[k]) {
                            if ((uint32_t)k == i) continue;
                            const aa_candidate x = a.cands[k];
                            if ((uint64_t)x.t_start <= te && (uint64_t)c.t_start <= (uint64_t)x.t_start + x.width && beats(x, c)) {
                                beaten = true;
                                break;
                            }
                        }
                    }
                }
                emit = !beaten;
            }
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

// Device address of g_peaks_scratch on each device, looked up by the first call made with that device current.
std::mutex g_mu;
uint32_t *g_scratch_addr[kMaxDevices] = {};

cudaError_t scratch_of_current_device(uint32_t **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_addr[dev]) {
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_peaks_scratch);       // the symbol's address on the CURRENT device
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = static_cast<uint32_t *>(ptr);
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int aa_find_peaks_device_noalloc(const aa_candidate *cands, uint32_t n, uint32_t ndms, uint32_t t_end,
                                            uint32_t wmax, aa_candidate *out, uint32_t max_out, uint32_t *n_out,
                                            void *stream, int *cuda_error)
{
    if (cuda_error) *cuda_error = 0;
    if (!n_out || (!cands && n) || (!out && max_out) || ndms == 0 || t_end == 0) return AA_ERR_INVALID;
    if (n > kMaxCands || ndms > kMaxCells) return AA_ERR_LIMIT;
    // bucket grid: 2^shift raw samples per bucket, as fine as the fixed array allows (the plan's grid starts at 2^5 too)
    uint32_t shift = 5;
    while (shift < 32 && (uint64_t)ndms * ((((uint64_t)t_end - 1) >> shift) + 1) > kMaxCells) ++shift;
    if (shift >= 32) return AA_ERR_LIMIT;
    const uint32_t nbk = (uint32_t)((((uint64_t)t_end - 1) >> shift) + 1);

    auto fail = [&](cudaError_t e) { cudaGetLastError(); if (cuda_error) *cuda_error = (int)e; return (int)AA_ERR_CUDA; };
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    uint32_t *scratch = nullptr;
    cudaError_t e = scratch_of_current_device(&scratch);
    if (e != cudaSuccess) return fail(e);

    NoallocArgs a{};
    a.cands = cands; a.n = n;
    a.head = reinterpret_cast<int32_t *>(scratch);
    a.next = scratch + kMaxCells;
    a.nrows = ndms; a.nbk = nbk; a.shift = shift; a.t_end = t_end; a.wmax = wmax;
    a.out = out; a.out_count = n_out; a.out_cap = max_out;

    // the array still holds the previous call's chains: empty every cell this call can touch (next[] needs no reset,
    // the link kernel writes next[i] of every record it links before anything follows it)
    e = cudaMemsetAsync(a.head, 0xFF, (size_t)ndms * nbk * sizeof(int32_t), st);
    if (e != cudaSuccess) return fail(e);
    e = cudaMemsetAsync(n_out, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return fail(e);
    if (n == 0) return AA_OK;
    const unsigned blocks = (unsigned)std::min<uint64_t>(((uint64_t)n + 255) / 256, 148 * 4);
    peaks_noalloc_link_kernel<<<blocks, 256, 0, st>>>(a);
    peaks_noalloc_decide_kernel<<<blocks, 256, 0, st>>>(a);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(e);
    return AA_OK;
}
