/*
 * aa_bench.h -- measurement probes of libaa.so.  NOT part of the search interface (that is include/aa.h): nothing here
 * is on the hot path, nothing here is needed to run a search.  bench.py and the report generators use these calls for
 * the roofline denominators SURVEY.md section 8(d) asks to be measured ("measure the real IADD3 / DP4A rates and
 * sustained clock first") and for the shared-memory cost model of the dedispersion kernel.
 * Same conventions as aa.h: plain C, aa_status return values, host pointers unless stated.
 */
#ifndef AA_BENCH_H_
#define AA_BENCH_H_

#include "aa.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Host-side cost model of the shared-pattern dedispersion kernels for range `range` of the plan `d` would build, from
 * its real delay table (no CUDA call): shared-memory wavefronts (128 bytes) per CTA = per (64 trials x tile_samples)
 * output tile, as the kernel issues them, the number of distinct delay patterns per stage, and the shared-memory
 * room the pattern rows take.  group_channels must be 4 (dedisp_ws_kernel: 4 channels x 64 trials per
 * stage; the 8-channel variant of round 2 was measured slower and removed).  AA_ERR_INVALID if the range does not fit
 * that kernel family (tables too large, or binned input with 4 * 255 * bin > 65535, which runs on the plain kernel).
 * wf_consumer counts the loads the kernel issues: a trial whose row word is the previous trial's reuses it.
 * Backs profiles/r2_cost_model.md; the binding shared-memory roofline of bench.py uses wf_* of the kernel that runs. */
typedef struct {
    int32_t  group_channels, block_trials, tile_samples, stages_per_cta;
    double   wf_consumer;          /* row-word loads of the consumer warps */
    double   wf_producer_load;     /* channel-window loads of the producer warps */
    double   wf_producer_store;    /* pattern-row stores (both alignments) */
    double   wf_bulk;              /* bytes landed by cp.async.bulk / 128 */
    double   patterns_mean;
    int32_t  patterns_max;
    int32_t  pad;
    double   stage_bytes_mean;
    uint64_t stage_bytes_max;
    uint64_t ring_bytes;           /* shared memory left for the ring of pattern rows */
    double   shared_offset_fraction; /* consecutive trials of a consumer warp that read the very same row words */
} aa_dedisp_model;
int aa_plan_dedisp_model(const aa_plan_desc *d, int32_t range, int32_t group_channels, aa_dedisp_model *out);

/* Micro-benchmarks of the units the hot path is bound by ("measure the real IADD3 / DP4A rates and
 * sustained clock first"); they back the roofline denominators of bench.py and DESIGN.md, they are not on the path.
 * aa_microbench runs kind 0 <= kind < aa_microbench_count() (aa_microbench_name: "iadd3", "lop3", "imad", "idp2a",
 * "idp4a", "prmt", "shf", "iadd3+imad", "lds32", "lds64", "lds128", "sts128", "lds32+iadd") as one wave of
 * ctas_per_sm (1..2) CTAs of 512 threads per SM, `trips` x 256 instructions per thread, and writes to host
 * pointers (each may be NULL): per_clk_sm = lane-operations per clock per SM for the arithmetic kinds (a full-warp
 * instruction counts 32), BYTES per clock per SM for the shared-memory kinds (conflict-free accesses), measured with
 * the SMs' own cycle counters; ms = kernel time (CUDA events); sm_mhz = the clock the run saw.
 * aa_microbench_link: pinned host <-> device copy of `bytes`, best of `reps`, in GB/s (dir 0 = H2D, 1 = D2H). */
int aa_microbench_count(void);
const char *aa_microbench_name(int kind);
int aa_microbench(int kind, int ctas_per_sm, int trips, double *per_clk_sm, double *ms, double *sm_mhz);
int aa_microbench_link(uint64_t bytes, int reps, int dir, double *gbs);

/* Which dedispersion kernel the plan chose for range r (the choice depends only on the delay table):
 * 0 = plain tiled kernel, 1 / 2 = shared-pattern kernel with 512 / 1024-sample tiles, 3 / 4 =
 * warp-specialised shared-pattern kernel with 512 / 1024-sample tiles, 5 = the same with 32-bit accumulators
 * (coarse time bins); AA_ERR_INVALID if r is out of range.  Used by tests to make sure every kernel is covered. */
int aa_plan_dedisp_variant(const aa_plan *p, int32_t r);

#ifdef __cplusplus
}
#endif
#endif /* AA_BENCH_H_ */
