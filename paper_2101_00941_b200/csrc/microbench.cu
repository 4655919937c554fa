// Micro-benchmarks behind the roofline denominators of DESIGN.md / bench.py ("measure the real
// IADD3 / DP4A rates", hard part H10: the INT32 lane count per SM is not in any guide).  One wave of CTAs, every
// thread runs independent chains of one instruction kind; each CTA records (SM id, first and last clock64), the host
// turns that into operations per clock per SM, which does not depend on the clock the GPU happened to run at.
// Nothing here is on the hot path; it measures the units the hot path is bound by.
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <vector>

#include "aa_internal.h"

namespace {

constexpr int kThreads = 512;
constexpr int kChains = 8;          // independent dependency chains per thread (latency 4-6, issue every 2)
constexpr int kUnroll = 32;         // instructions per chain per loop trip

struct Stamp { unsigned long long t0, t1; unsigned smid, pad; };

__device__ __forceinline__ unsigned smid()
{
    unsigned v;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(v));
    return v;
}

enum Kind : int {
    K_IADD3 = 0, K_LOP3, K_IMAD, K_IDP2A, K_IDP4A, K_PRMT, K_SHF, K_IADD3_IMAD,
    K_LDS32, K_LDS64, K_LDS128, K_STS128, K_LDS32_IADD, K_NKINDS
};

template <int KIND>
__device__ __forceinline__ void op(unsigned &a, unsigned b, unsigned c)
{
    if (KIND == K_IADD3) asm volatile("{.reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2;}" : "+r"(a) : "r"(b), "r"(c));
    if (KIND == K_LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a) : "r"(b), "r"(c));
    if (KIND == K_IMAD) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a) : "r"(b), "r"(c));
    if (KIND == K_IDP2A) asm volatile("dp2a.lo.u32.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(b), "r"(c));
    if (KIND == K_IDP4A) asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(b), "r"(c));
    if (KIND == K_PRMT) asm volatile("prmt.b32 %0, %0, %1, %2;" : "+r"(a) : "r"(b), "r"(c));
    if (KIND == K_SHF) asm volatile("shf.r.wrap.b32 %0, %0, %1, %2;" : "+r"(a) : "r"(b), "r"(c));
}

// arithmetic kinds: kChains chains x kUnroll instructions per trip
template <int KIND>
__global__ void __launch_bounds__(kThreads, 2) alu_kernel(int trips, unsigned seed, unsigned *sink, Stamp *stamps)
{
    unsigned a[kChains];
#pragma unroll
    for (int i = 0; i < kChains; ++i) a[i] = seed + threadIdx.x * 7u + i;
    const unsigned b = seed | 1u, c = (seed >> 3) | 5u;
    __syncthreads();
    const unsigned long long t0 = clock64();
    for (int t = 0; t < trips; ++t) {
#pragma unroll
        for (int u = 0; u < kUnroll; ++u)
#pragma unroll
            for (int i = 0; i < kChains; ++i) {
                if (KIND == K_IADD3_IMAD) {
                    if (i & 1) op<K_IMAD>(a[i], b, c);
                    else op<K_IADD3>(a[i], b, c);
                } else {
                    op<KIND>(a[i], b, c);
                }
            }
    }
    const unsigned long long t1 = clock64();
    unsigned s = 0;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s ^= a[i];
    if (s == 0x12345u) sink[0] = s;
    if (threadIdx.x == 0) stamps[blockIdx.x] = Stamp{t0, t1, smid(), 0};
}

// shared-memory kinds: conflict-free accesses of W words per lane from a 32 KB buffer; kChains loads in flight
template <int KIND>
__global__ void __launch_bounds__(kThreads, 2) smem_kernel(int trips, unsigned seed, unsigned *sink, Stamp *stamps)
{
    __shared__ __align__(16) unsigned buf[8192];
    for (int i = threadIdx.x; i < 8192; i += kThreads) buf[i] = seed + i;
    __syncthreads();
    constexpr int W = KIND == K_LDS64 ? 2 : (KIND == K_LDS128 || KIND == K_STS128) ? 4 : 1;   // words per lane
    const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // every warp reads its own 128*W-byte line; the line moves by an immediate offset per instruction
    const unsigned base = (unsigned)__cvta_generic_to_shared(buf) + ((warp * 32 * W + lane * W) * 4) % (4096 * 4);
    unsigned acc[kChains];
#pragma unroll
    for (int i = 0; i < kChains; ++i) acc[i] = lane + i;
    const unsigned long long t0 = clock64();
    for (int t = 0; t < trips; ++t) {
#pragma unroll (W == 1 ? 4 : W == 2 ? 2 : 1)
        for (int u = 0; u < kUnroll / (2 * W); ++u) {        // 128 / W accesses per trip, every address distinct
#pragma unroll
            for (int i = 0; i < kChains; ++i) {
                const unsigned addr = base + (unsigned)((u * kChains + i) * 128 * W);
                if (KIND == K_LDS32) {
                    unsigned v;
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
                    acc[i] ^= v;
                } else if (KIND == K_LDS32_IADD) {
                    unsigned v;
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
                    acc[i] += v;
                } else if (KIND == K_LDS64) {
                    unsigned v0, v1;
                    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v0), "=r"(v1) : "r"(addr));
                    acc[i] ^= v0 ^ v1;
                } else if (KIND == K_LDS128) {
                    unsigned v0, v1, v2, v3;
                    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v0), "=r"(v1), "=r"(v2), "=r"(v3) : "r"(addr));
                    acc[i] ^= v0 ^ v1 ^ v2 ^ v3;
                } else {
                    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(acc[i]), "r"(acc[i]), "r"(acc[i]), "r"(acc[i]) : "memory");
                }
            }
        }
    }
    const unsigned long long t1 = clock64();
    unsigned s = 0;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s ^= acc[i];
    __syncthreads();
    if (s == 0x12345u) sink[0] = s + buf[lane];
    if (threadIdx.x == 0) stamps[blockIdx.x] = Stamp{t0, t1, smid(), 0};
}

template <int KIND>
cudaError_t launch(int grid, int trips, unsigned *sink, Stamp *stamps, cudaStream_t st)
{
    if constexpr (KIND >= K_LDS32) smem_kernel<KIND><<<grid, kThreads, 0, st>>>(trips, 12345u, sink, stamps);
    else alu_kernel<KIND><<<grid, kThreads, 0, st>>>(trips, 12345u, sink, stamps);
    return cudaGetLastError();
}

const char *const kNames[K_NKINDS] = {"iadd3", "lop3", "imad", "idp2a", "idp4a", "prmt", "shf", "iadd3+imad",
                                      "lds32", "lds64", "lds128", "sts128", "lds32+iadd"};

}  // namespace

extern "C" {

int aa_microbench_count(void) { return K_NKINDS; }

const char *aa_microbench_name(int kind) { return kind >= 0 && kind < K_NKINDS ? kNames[kind] : nullptr; }

// Runs micro-benchmark `kind` on the current device: one wave of CTAs (ctas_per_sm per SM), `trips` loop trips of
// 256 instructions per thread.  Results (host pointers, any may be NULL):
//   per_clk_sm : arithmetic kinds: lane-operations per clock per SM (one IADD3 of a full warp = 32);
//                shared-memory kinds: BYTES per clock per SM (one conflict-free 128-byte wavefront per clock = 128)
//   ms         : kernel duration (CUDA events)
//   sm_mhz     : the SM clock the run saw (cycles of the slowest SM / duration)
int aa_microbench(int kind, int ctas_per_sm, int trips, double *per_clk_sm, double *ms, double *sm_mhz)
{
    if (kind < 0 || kind >= K_NKINDS || ctas_per_sm < 1 || ctas_per_sm > 2 || trips < 1) return AA_ERR_INVALID;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return AA_ERR_CUDA;
    const int grid = nsm * ctas_per_sm;
    unsigned *sink = nullptr;
    Stamp *stamps = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaStream_t st = nullptr;
    int rc = AA_OK;
    std::vector<Stamp> h(grid);
    float t = 0;
    auto run = [&](int tr) -> cudaError_t {
        switch (kind) {
            case K_IADD3: return launch<K_IADD3>(grid, tr, sink, stamps, st);
            case K_LOP3: return launch<K_LOP3>(grid, tr, sink, stamps, st);
            case K_IMAD: return launch<K_IMAD>(grid, tr, sink, stamps, st);
            case K_IDP2A: return launch<K_IDP2A>(grid, tr, sink, stamps, st);
            case K_IDP4A: return launch<K_IDP4A>(grid, tr, sink, stamps, st);
            case K_PRMT: return launch<K_PRMT>(grid, tr, sink, stamps, st);
            case K_SHF: return launch<K_SHF>(grid, tr, sink, stamps, st);
            case K_IADD3_IMAD: return launch<K_IADD3_IMAD>(grid, tr, sink, stamps, st);
            case K_LDS32: return launch<K_LDS32>(grid, tr, sink, stamps, st);
            case K_LDS64: return launch<K_LDS64>(grid, tr, sink, stamps, st);
            case K_LDS128: return launch<K_LDS128>(grid, tr, sink, stamps, st);
            case K_STS128: return launch<K_STS128>(grid, tr, sink, stamps, st);
            default: return launch<K_LDS32_IADD>(grid, tr, sink, stamps, st);
        }
    };
#define MB(call) do { if ((call) != cudaSuccess) { rc = AA_ERR_CUDA; goto out; } } while (0)
    MB(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
    MB(cudaMalloc(&sink, 256));
    MB(cudaMalloc(&stamps, sizeof(Stamp) * grid));
    MB(cudaEventCreate(&e0));
    MB(cudaEventCreate(&e1));
    MB(run(std::max(1, trips / 8)));           // warm-up
    MB(cudaStreamSynchronize(st));
    MB(cudaEventRecord(e0, st));
    MB(run(trips));
    MB(cudaEventRecord(e1, st));
    MB(cudaStreamSynchronize(st));
    MB(cudaEventElapsedTime(&t, e0, e1));
    MB(cudaMemcpy(h.data(), stamps, sizeof(Stamp) * grid, cudaMemcpyDeviceToHost));
    {
        // per SM: everything its CTAs did / (last end - first start); the median over SMs is reported
        const bool smem = kind >= K_LDS32;
        // arithmetic: 256 instructions per trip; shared memory: 128 / W accesses of 4 W bytes = 512 bytes per trip
        const double per_thread = smem ? (double)trips * 512.0 : (double)trips * kUnroll * kChains;
        const double unit = 1.0;
        std::vector<unsigned long long> lo(nsm, ~0ull), hi(nsm, 0ull);
        std::vector<int> n(nsm, 0);
        for (auto &s : h)
            if ((int)s.smid < nsm) { lo[s.smid] = std::min(lo[s.smid], s.t0); hi[s.smid] = std::max(hi[s.smid], s.t1); n[s.smid]++; }
        std::vector<double> rate;
        unsigned long long longest = 0;
        for (int i = 0; i < nsm; ++i)
            if (n[i]) {
                rate.push_back(n[i] * (double)kThreads * per_thread * unit / (double)(hi[i] - lo[i]));
                longest = std::max(longest, hi[i] - lo[i]);
            }
        std::sort(rate.begin(), rate.end());
        if (per_clk_sm) *per_clk_sm = rate.empty() ? 0.0 : rate[rate.size() / 2];
        if (ms) *ms = t;
        if (sm_mhz) *sm_mhz = t > 0 ? (double)longest / (t * 1e3) : 0.0;
    }
out:
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (sink) cudaFree(sink);
    if (stamps) cudaFree(stamps);
    if (st) cudaStreamDestroy(st);
    if (rc == AA_ERR_CUDA) cudaGetLastError();
    return rc;
#undef MB
}

// Pinned host <-> device copy bandwidth: `bytes` per copy, best of `reps`, GB/s (1e9).  dir 0 = H2D, 1 = D2H.
int aa_microbench_link(uint64_t bytes, int reps, int dir, double *gbs)
{
    if (!bytes || reps < 1 || !gbs) return AA_ERR_INVALID;
    void *h = nullptr, *d = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaStream_t st = nullptr;
    int rc = AA_OK;
    double best = 0;
#define MB(call) do { if ((call) != cudaSuccess) { rc = AA_ERR_CUDA; goto out; } } while (0)
    MB(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
    MB(cudaHostAlloc(&h, bytes, cudaHostAllocDefault));
    MB(cudaMalloc(&d, bytes));
    memset(h, 1, bytes);
    MB(cudaEventCreate(&e0));
    MB(cudaEventCreate(&e1));
    for (int r = 0; r <= reps; ++r) {
        MB(cudaEventRecord(e0, st));
        MB(dir == 0 ? cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, st) : cudaMemcpyAsync(h, d, bytes, cudaMemcpyDeviceToHost, st));
        MB(cudaEventRecord(e1, st));
        MB(cudaStreamSynchronize(st));
        float t = 0;
        MB(cudaEventElapsedTime(&t, e0, e1));
        if (r > 0 && t > 0) best = std::max(best, (double)bytes / (t * 1e6));
    }
    *gbs = best;
out:
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (h) cudaFreeHost(h);
    if (d) cudaFree(d);
    if (st) cudaStreamDestroy(st);
    if (rc == AA_ERR_CUDA) cudaGetLastError();
    return rc;
#undef MB
}

}  // extern "C"
