/*
 * aa.h -- C ABI of the B200-native streamed dedispersion + single-pulse search.
 *
 * The hot path of "Implementing CUDA Streams into AstroAccelerate - A Case Study"
 * (arXiv 2101.00941): time chunks split into per-stream sub-chunks (PAPER.md:33,
 * Fig. 2), pinned host memory and asynchronous copies (PAPER.md:41 steps 1-5,
 * :49-51), dedispersion then single-pulse search per sub-chunk (PAPER.md:19, :43,
 * :71), one host thread per stream for the host-side output copy.
 * The paper states no interface (AstroAccelerate is a program); the three calls
 * and their arguments follow BASELINE.json:north_star, the arithmetic follows
 * SURVEY.md section 8(c) as restated in DESIGN.md.
 *
 * Conventions
 *   - plain C, no exceptions, no global state; every function returns an aa_status
 *     (0 = AA_OK, negative = error) unless stated otherwise.
 *   - "host" pointers are ordinary process memory; "pinned" means page-locked
 *     (cudaHostAlloc / cudaHostRegister / aa_host_alloc); "device" means CUDA
 *     device memory of the current device.
 *   - the caller owns every buffer it passes; aa_plan_create copies the arrays in
 *     the descriptor; the library owns what it allocates and frees it in aa_destroy.
 *   - one aa_plan may be used by one thread at a time; different plans are independent.
 */
#ifndef AA_H_
#define AA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    AA_OK = 0,
    AA_ERR_INVALID = -1,     /* bad argument / inconsistent descriptor */
    AA_ERR_NOT_PINNED = -2,  /* aa_run input is pageable host memory (never staged silently) */
    AA_ERR_OOM = -3,         /* device or pinned allocation failed */
    AA_ERR_CUDA = -4,        /* a CUDA call failed; see aa_last_cuda_error() */
    AA_ERR_OVERFLOW = -5,    /* more candidates than the output / per-sub-chunk buffers hold;
                                the run is otherwise valid and *n_cands is the true total */
    AA_ERR_LIMIT = -6        /* request larger than the fixed capacity of aa_find_peaks_device_noalloc */
} aa_status;

typedef enum {
    AA_DEDISP_AUTO = 0,
    AA_DEDISP_PLAIN = 1,     /* plain tiled kernel */
    AA_DEDISP_SP512 = 2,     /* shared-pattern kernel, 512-sample tiles */
    AA_DEDISP_SP1024 = 3,    /* ... 1024-sample tiles */
    AA_DEDISP_WS512 = 4,     /* warp-specialised shared-pattern kernel, 512-sample tiles */
    AA_DEDISP_WS1024 = 5     /* ... 1024-sample tiles */
} aa_dedisp_choice;

/* One DM range of the plan: DM_i = dm_low + i*dm_step (double), i = 0..ndms-1, searched on
 * the input summed over `bin` consecutive raw samples (time decimation). */
typedef struct {
    double  dm_low;      /* pc cm^-3 */
    double  dm_step;     /* pc cm^-3, >= 0 */
    int32_t ndms;        /* > 0 */
    int32_t bin;         /* >= 1, divides norm_block */
} aa_dm_range;

/* One detection. 16 bytes. */
typedef struct {
    uint32_t dm_index;   /* global trial index: ranges concatenated in plan order */
    uint32_t t_start;    /* first raw input sample of the boxcar (= tau*bin) */
    uint32_t width;      /* boxcar width in raw samples (= w*bin) */
    float    snr;        /* (B_w - w*mu)/(sigma*sqrt(w)), computed in double, stored as float */
} aa_candidate;

typedef struct {
    /* filterbank: x[t][c], time-major, channel 0 centred on f_top, foff < 0 (A1, A2); uint8 unless nbits says otherwise */
    int32_t  nchans;
    uint64_t nsamp;
    double   tsamp;            /* seconds */
    double   f_top;            /* MHz */
    double   foff;             /* MHz, negative */
    /* search plan */
    int32_t  nranges;
    const aa_dm_range *ranges;
    int32_t  nwidths;
    const int32_t *widths;     /* boxcar widths in BINNED samples of each range, ascending, >= 1 */
    double   snr_threshold;    /* double, not the float of SURVEY.md 8(b): the threshold test S >= threshold is taken in double on
                                  both sides (deviations) */
    /* streaming: each time chunk of chunk_len raw samples is split into n_streams
     * sub-chunks; chunk_len/n_streams must be a multiple of norm_block and at least the halo
     * (DM sweep + longest boxcar) reported by aa_plan_query. */
    int32_t  n_streams;        /* 1..64 */
    uint64_t chunk_len;        /* raw samples */
    uint32_t norm_block;       /* raw samples per normalisation block; 0 -> 65536 (A9) */
    /* optional resources owned by the caller (e.g. a torch tensor and torch streams);
     * NULL/0 -> the library allocates with cudaMalloc and creates non-blocking streams. */
    void    *device_arena;       /* device */
    uint64_t device_arena_bytes; /* must be >= aa_plan_arena_bytes(desc) */
    void *const *streams;        /* cudaStream_t[n_streams] or NULL */
    /* dense dedispersed rows to hand back: global dm indices, ascending.  A few rows serve parity checks; all of
     * them give the whole DM x time plane (the paper's device-to-host path): runs of consecutive
     * trials leave the device in one strided copy into the stream's pinned staging and the stream's host thread
     * moves them into tap_out.  Staging: sum over ranges of ntap_r * subchunk_len / bin_r * 4 bytes per stream. */
    int32_t  ntap;
    const uint32_t *tap_dm_indices;
    /* capacity of each stream's device candidate list per sub-chunk; 0 -> 1<<21 */
    uint64_t max_cands_per_subchunk;
    /* 1: every stream also gets a small pinned input staging buffer ((subchunk_len + halo) * nchans
     * bytes) so that aa_run_staged can take an observation held in pageable memory */
    int32_t  stage_input;
    /* TEST HOOK, not part of the search: leave 0.  (An aa_dedisp_choice.)  AA_DEDISP_AUTO (0) lets the plan pick the dedispersion kernel of
     * every range from its delay table.  Any other value restricts the choice to that one kernel family; a range the
     * forced kernel cannot serve (tables do not fit) runs on the plain kernel.  Unknown values: AA_ERR_INVALID.  All
     * kernels compute the same exact sums; tests force each one against the oracle. */
    int32_t  dedisp_variant;
    /* Bits per input sample (reading A19): 0 or 8 = uint8 [nsamp][nchans]; 4 = two samples per byte, the
     * even channel in the low nibble, [nsamp][nchans / 2] bytes (nchans even); 16 = little-endian uint16,
     * [nsamp][2 nchans] bytes.  4-bit samples are unpacked on the device; 16-bit samples are split into a low-byte and
     * a high-byte plane, both dedispersed by the 8-bit kernels and joined as D = D(low) + 256 D(high) (exact). */
    int32_t  nbits;
    /* Reading A20 (decimated long boxcars): 0 = every width at every sample (BASELINE.json).  wdec > 0:
     * a width w > wdec is searched on a coarser time grid, as in a search that halves the time resolution each time it
     * doubles the width: only at tau (absolute binned sample) with tau mod dec(w) == 0, dec(w) = the smallest power
     * of two with w / dec(w) <= wdec.  The boxcar sums themselves stay exact. */
    int32_t  width_decimation;
    /* Reading A18 (per-width measured sigma): 0 = S_w = (B_w - w mu) / (sigma sqrt w), white-noise
     * scaling of the block's statistics (BASELINE.json).  1 = S_w = (B_w - mu_w) / sigma_w with (mu_w, sigma_w) the same
     * robust estimator applied to the boxcar series of width w itself over the normalisation block (on the width's grid);
     * a width with sigma_w = 0 or fewer than 32 boxcars in the block is skipped.  Accepted on every range: where the
     * block does not fit the cluster kernel (64-bit boxcar sums, block / bin not a multiple of 4 or above 131072
     * samples) the generic kernel sweeps the block once per pass of the estimator (slower, same results). */
    int32_t  sigma_mode;
    /* 0 = aa_run returns every candidate (one per (DM, time), reading A11; BASELINE.json).  1 = it returns the PEAKS of
     * that list (reading A17, the rule of aa_find_peaks): each sub-chunk's list is thinned on the device before it
     * crosses the host link (kernels_peaks.cu), candidates whose neighbourhood reaches into an adjacent sub-chunk are
     * settled by the host on the merged list; the result is exactly aa_find_peaks of the full list.  *n_cands and
     * aa_stats.n_peaks then count peaks, aa_stats.n_candidates still counts the candidates found on the device. */
    int32_t  output_mode;
    /* TEST HOOK, not part of the search: leave 0.  Single-pulse-search kernel: 0 = the plan's choice; 1 = keep the first cluster
     * kernel (sps_cluster_kernel: four passes over the segment for the statistics) where the second
     * (sps_cluster2_kernel: one pass + the listed outliers) would serve.  Same results.  Other values: AA_ERR_INVALID. */
    int32_t  sps_variant;
    int32_t  reserved0;        /* keeps the size a multiple of 8; must be 0 */
} aa_plan_desc;

typedef struct {
    uint64_t maxshift;          /* raw samples, multiple of every bin */
    uint64_t t_valid;           /* nsamp - maxshift */
    uint64_t halo;              /* raw samples a sub-chunk reads past its own span */
    uint64_t subchunk_len;      /* chunk_len / n_streams */
    uint64_t n_subchunks;
    uint64_t ndms_total;
    uint64_t dm_trial_samples;  /* sum_r ndms_r * nout_r : the work unit of the metric */
    uint64_t arena_bytes;       /* device memory the plan uses */
    uint64_t pinned_bytes;      /* pinned staging the plan owns */
    uint64_t tap_row_len;       /* uint32 elements per tapped row in aa_run's tap_out
                                   (= max over ranges of nout_r); 0 if ntap == 0 */
} aa_plan_info;

typedef struct {
    double   wall_ms;           /* aa_run call -> return */
    double   sort_ms;           /* final host sort, inside wall_ms */
    uint64_t h2d_bytes, d2h_bytes;
    double   h2d_ms, d2h_ms;    /* sum of copy durations (CUDA events on their streams) */
    double   prep_ms;           /* corner turn + binning kernels, summed */
    double   dedisp_ms;         /* dedispersion kernels, summed over launches */
    double   sps_ms;            /* statistics + boxcar/candidate kernels, summed */
    uint64_t dedisp_launches, sps_launches, prep_launches;
    uint64_t n_candidates;      /* true total found */
    uint64_t n_stored;          /* records written to `out` (< n_candidates only on overflow) */
    int32_t  overflow;          /* 1 if any list was truncated */
    int32_t  n_streams;
    uint64_t h2h_bytes;         /* aa_run_staged: bytes copied host -> pinned staging by the stream threads */
    double   h2h_ms;            /* ... and the time those copies took, summed over threads */
    uint64_t n_peaks;           /* output_mode 1: peaks returned (0 otherwise) */
} aa_stats;

/* Device timeline of one sub-chunk of the last run, in milliseconds after the start of the run (CUDA events
 * on the sub-chunk's stream): the replacement for the paper's visual inspection of the profiler timeline
 * (Fig. 3-4). */
typedef struct {
    uint32_t index;             /* sub-chunk j: raw samples [j*subchunk_len, (j+1)*subchunk_len) */
    uint32_t stream;            /* stream / host thread that ran it (j mod n_streams) */
    double   h2d_begin, h2d_end;        /* host-to-device copy of its new rows (equal if resident) */
    double   prep_end;          /* corner turn done */
    double   compute_begin;     /* halo of sub-chunk j-1 available: binning / dedispersion may start */
    double   compute_end;       /* last range's SPS kernel done */
    double   d2h_end;           /* candidate list in pinned staging */
    double   dedisp_ms, sps_ms; /* kernel durations summed over ranges */
} aa_subchunk_times;

typedef struct aa_plan aa_plan;

/* Device bytes a plan built from `d` needs (for callers that bring their own arena).
 * Returns 0 if the descriptor is invalid. */
uint64_t aa_plan_arena_bytes(const aa_plan_desc *d);

/* The geometry a plan built from `d` would have (maxshift, halo, sub-chunks, work units, memory), without
 * creating it: no CUDA call, usable on a host without a GPU (e.g. to split an observation over ranks). */
int aa_plan_geometry(const aa_plan_desc *d, aa_plan_info *out);

/* Allocation phase (PAPER.md:19 part 2, :41 steps 1-2, :71): validates the descriptor, builds
 * the delay tables in double (north_star formula), creates streams and events, allocates the
 * device ring, per-stream work buffers, candidate lists and pinned staging.  Nothing is
 * allocated later.  *out is NULL on error. */
int aa_plan_create(aa_plan **out, const aa_plan_desc *d);

int aa_plan_query(const aa_plan *p, aa_plan_info *out);

/* nout_r (valid output samples, binned) of range r, or 0 if r is out of range. */
uint64_t aa_plan_nout(const aa_plan *p, int32_t r);

/* Copies the integer delay table of range r ([ndms_r][nchans] int32, binned samples) to host
 * memory `out`; used by tests to compare with the oracle entry by entry. */
int aa_plan_delays(const aa_plan *p, int32_t r, int32_t *out);

/*
 * The hot path: for every sub-chunk, on its stream:
 * async H2D of the new input rows -> corner turn into the device ring -> per range: (binning,)
 * dedispersion, block statistics + boxcar S/N + candidate compaction -> D2H of the candidate
 * list into pinned staging; one host thread per stream copies staging into `out`.
 *   host_input : PINNED host, uint8 [nsamp][nchans] (nbits 8; [nsamp][nchans * nbits / 8] bytes in general)
 *                (AA_ERR_NOT_PINNED otherwise)
 *   out        : host (pageable ok), room for max_cands records; sorted by (dm_index, t_start)
 *   n_cands    : host, receives the true number found; if it exceeds max_cands or a sub-chunk's
 *                device list overflowed the call returns AA_ERR_OVERFLOW and aa_stats.n_stored
 *                says how many (sorted) records `out` holds
 *   tap_out    : host (pageable ok) uint32 [ntap][tap_row_len] or NULL; row k receives the
 *                dedispersed series of tap_dm_indices[k], nout_r values, rest untouched
 * No allocation, no pageable copy and no device-wide synchronisation happen inside.
 *
 * Precondition on the process, not checked here (the library reads no environment variable): the CUDA context must
 * have at least n_streams hardware work queues, i.e. the CALLER sets CUDA_DEVICE_MAX_CONNECTIONS >= n_streams (default 8,
 * maximum 32) in the environment BEFORE CUDA initialises.  With fewer, streams share a queue and one stream's small
 * D2H copy waits behind another stream's kernels (a false dependency): results are identical, the overlap is not
 * (measured: 16 streams on 8 queues lose about 5 %).  bench.py and the Python tools set 32.
 */
int aa_run(aa_plan *p, const uint8_t *host_input, aa_candidate *out, uint64_t max_cands,
           uint64_t *n_cands, uint32_t *tap_out);

/* The paper's own input arrangement: the observation sits in ordinary PAGEABLE host
 * memory, too big to pin; every stream's host thread copies the rows of its next sub-chunk into its small
 * pinned staging buffer (host -> host), from where they go to the device with cudaMemcpyAsync.  The
 * host copy of sub-chunk j + n_streams runs while the stream still computes sub-chunk j.  Needs a plan
 * created with stage_input = 1 (AA_ERR_INVALID otherwise); host_input may be pageable or pinned.
 * Everything else, results included, is identical to aa_run. */
int aa_run_staged(aa_plan *p, const uint8_t *host_input, aa_candidate *out, uint64_t max_cands,
                  uint64_t *n_cands, uint32_t *tap_out);

/* Same path with the observation already in device memory (uint8 [nsamp][nchans], device):
 * the H2D step is skipped, everything else is identical.  Used for kernel-only timing. */
int aa_run_resident(aa_plan *p, const uint8_t *device_input, aa_candidate *out, uint64_t max_cands,
                    uint64_t *n_cands, uint32_t *tap_out);

/* Timings and counters of the last aa_run / aa_run_resident on this plan. */
int aa_get_stats(const aa_plan *p, aa_stats *out);

/* Per-sub-chunk device timeline of the last run: writes min(max, n_subchunks) entries in sub-chunk order and
 * the number of sub-chunks to *n. */
int aa_get_timeline(const aa_plan *p, aa_subchunk_times *out, uint64_t max, uint64_t *n);

/* Optional post-step on the host (the paper only cites the step): peak finding.
 * Two candidates are neighbours if their dm_index differ by at most 1 and their boxcars overlap or touch in raw
 * samples (t' <= t + w and t <= t' + w'); a candidate is a peak iff no neighbour has a larger snr (the stored
 * float), ties going to the smaller (dm_index, t_start).
 *   cands    : host, n records sorted by (dm_index, t_start) as aa_run returns them (AA_ERR_INVALID otherwise)
 *   out      : host, room for max_out records; receives the peaks in the same order (may alias nothing in cands)
 *   n_out    : host, number of peaks found; AA_ERR_OVERFLOW if it exceeds max_out (the first max_out are stored)
 *   nthreads : host threads to use (rows of DM trials are spread over them); < 1 -> all hardware threads
 * Pure host code: needs no plan and no GPU. */
int aa_find_peaks(const aa_candidate *cands, uint64_t n, aa_candidate *out, uint64_t max_out, uint64_t *n_out,
                  int32_t nthreads);

/*
 * Peak finding (the rule of aa_find_peaks, reading A17) on a candidate list that is already in DEVICE memory, for
 * callers that may not allocate device memory while they run: a real-time ingest loop in its streamed phase (one
 * cudaMalloc / cudaFree waits for the whole device and stalls every other stream's copies and kernels
 * and :71 allocate everything beforehand for that reason), or a process whose device memory all belongs to one
 * owner (a framework's caching pool, an arena carved at start-up) behind whose back a raw cudaMalloc would fail or
 * fragment.  The call makes no cudaMalloc / cudaFree and calls no library routine that allocates: the bucket grid
 * and chains the kernels need sit in a fixed array inside the library image.  That array costs 8 MiB of device
 * memory on every GPU that loads libaa.so, from load until the process exits, whether or not this function is used.
 *   cands   : device, n records in ANY order, at most one per (dm_index, t_start); records with dm_index >= ndms or
 *             t_start >= t_end are ignored (neither peaks nor neighbours)
 *   n       : <= AA_PEAKS_NOALLOC_MAX_CANDS, else AA_ERR_LIMIT
 *   ndms    : number of DM rows, > 0; t_end: candidates start in [0, t_end) raw samples, > 0.  The grid has
 *             ndms * ceil(t_end / 2^shift) cells, shift >= 5 chosen so that they fit AA_PEAKS_NOALLOC_MAX_CELLS;
 *             AA_ERR_LIMIT if ndms alone exceeds it.  Coarser cells only cost time.
 *   wmax    : no record's width exceeds it (raw samples); a longer boxcar may be missed as a neighbour
 *   out     : device, room for max_out records; receives the peaks, UNORDERED (sort by (dm_index, t_start) to
 *             compare with aa_find_peaks: the same set of records, bit for bit)
 *   n_out   : device uint32; receives the number of peaks found, which may exceed max_out (only max_out are stored)
 *   stream  : cudaStream_t of the current device (NULL = the default stream); everything is enqueued on it and the
 *             call returns without waiting: read out / n_out after synchronising the stream
 *   cuda_error : host, may be NULL; the cudaError_t when the call returns AA_ERR_CUDA, else 0
 * First call on a device: it looks up the array's device address (cudaGetSymbolAddress, once per device, with
 * the device that is current at the call) and remembers it; make that first call during set-up, before any stream
 * capture is begun.  Sharing: every call on a device uses the same array, which keeps the previous call's contents;
 * each call empties the cells it will use on `stream` before its kernels, so calls that follow one another on one
 * stream are independent, but two calls that can be on the GPU at the same time (two streams with no event
 * between them, two host threads) race on the array and give wrong peaks: order them.  Errors: AA_ERR_INVALID
 * (NULL pointers, ndms or t_end 0), AA_ERR_LIMIT (sizes above), AA_ERR_CUDA.
 */
#define AA_PEAKS_NOALLOC_MAX_CANDS (1u << 20)   /* records per call */
#define AA_PEAKS_NOALLOC_MAX_CELLS (1u << 20)   /* bucket cells per call */
int aa_find_peaks_device_noalloc(const aa_candidate *cands, uint32_t n, uint32_t ndms, uint32_t t_end, uint32_t wmax,
                                 aa_candidate *out, uint32_t max_out, uint32_t *n_out, void *stream, int *cuda_error);

/* NULL-safe.  Frees everything the plan allocated (not a caller-owned arena or streams). */
void aa_destroy(aa_plan *p);

/* Pinned host allocation helpers (cudaHostAlloc / cudaFreeHost). */
int  aa_host_alloc(void **p, uint64_t bytes);
void aa_host_free(void *p);

const char *aa_strerror(int status);
/* cudaError_t of the last failing CUDA call in this thread's last aa_* call (0 if none). */
int aa_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* AA_H_ */
