// Host side of libaa: plan (allocation phase), stream/event scheduler, output stage.
//
// Paper mapping: all allocation happens in aa_plan_create (PAPER.md:19 part 2, :71 "moved memory
// allocations ... to the Preparation/Memory allocation phase"); aa_run only issues asynchronous
// copies and kernels on per-sub-chunk streams with event dependencies (PAPER.md:41 steps 3-5) and
// uses one host thread per stream for the host-side copies.  Every stream owns a
// private candidate list and counter (the paper's atomics / cudaStreamWaitEvent trouble,
// PAPER.md:73, came from state shared across streams; nothing is shared here).
#include <algorithm>
#include <atomic>
#include <chrono>
#include <condition_variable>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <memory>
#include <mutex>
#include <new>
#include <thread>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "aa_internal.h"

using namespace aa;

namespace {

thread_local int g_last_cuda_error = 0;

inline uint64_t round_up(uint64_t v, uint64_t m) { return (v + m - 1) / m * m; }
inline uint64_t gcd64(uint64_t a, uint64_t b) { while (b) { uint64_t t = a % b; a = b; b = t; } return a; }

struct Range {
    aa_dm_range r{};
    uint64_t nout = 0;          // valid output samples (binned)
    int32_t maxdelay = 0;       // binned samples
    uint32_t dm_base = 0;
    std::vector<int32_t> h_delays;   // [ndms][nchans]
    int32_t *d_delays = nullptr;
    std::vector<int32_t> h_dtiles;   // [nblk][nstages][DB][CS]: per (DM block, channel stage) delay tiles
    int32_t *d_dtiles = nullptr;
    int row = 0;                // staged row length (elements)
    int dpw = 4;                // DM trials per warp in the dedispersion kernel
    bool in16 = false;
    int flush_ch = 2;
    bool wide = false;          // 64-bit boxcar sums
    bool small31 = false;       // boxcar sums below 2^31 (signed pre-filter arithmetic in the SPS kernel)
    int bin_slot = -1;          // index into the per-stream binned buffers
    int sp_tb = 0;              // shared-pattern kernel: time tile (1024 or 512); 0 = plain kernel
    bool ws = false;            // warp-specialised variant of the shared-pattern kernel
    bool ws_wide = false;       // ... with 32-bit accumulators and no intermediate flush (coarse time bins)
    std::vector<SpRecord> h_sp;
    std::vector<WsRecord> h_ws;
    void *d_sp = nullptr;
    size_t sp_table_bytes() const
    {
        return ws ? h_ws.size() * sizeof(WsRecord) : h_sp.size() * sizeof(SpRecord);
    }
    const void *sp_table() const
    {
        return ws ? (const void *)h_ws.data() : (const void *)h_sp.data();
    }
    int32_t sp_rows = 0, sp_pbytes = 0, sp_flush = 1;
    std::vector<std::pair<int, int>> taps;   // (local dm, tap row)
};

constexpr int kEvFixed = 9;     // h2d0 h2d1 ct1 bin0 bin1 list0 list1 peaks0 peaks1

struct Stream {
    cudaStream_t st = nullptr;
    bool own = false;
    uint8_t *d_raw = nullptr;
    std::vector<uint16_t *> d_binned;
    uint32_t *d_D = nullptr;
    uint32_t *d_D2 = nullptr;         // 16-bit input: dedispersed high-byte plane of the current range
    aa_candidate *d_cands = nullptr;
    uint32_t *d_count = nullptr;      // [0] candidates found, [1] records of the thinned list (output_mode 1)
    int32_t *d_head = nullptr;        // output_mode 1: bucket grid, chain and thinned list of the peak kernels
    uint32_t *d_next = nullptr;
    aa_candidate *d_peaks = nullptr;
    uint32_t *h_count = nullptr;      // pinned
    aa_candidate *h_cands = nullptr;  // pinned
    uint32_t *h_tap = nullptr;        // pinned
    uint8_t *h_stage = nullptr;       // pinned input staging (aa_run_staged), (L + halo) * nchans bytes
    std::vector<cudaEvent_t> ev;      // timing events
    struct TapCopy { int row; uint64_t tau0, n, off; };
    std::vector<TapCopy> tapcopies;   // capacity = ntap, reserved at plan creation; refilled per sub-chunk
    std::vector<uint32_t> sort_cur;   // [ndms_total + 1] cursors of the per-sub-chunk counting sort (sized at plan creation)
    // per-run accumulators
    double h2d_ms = 0, d2h_ms = 0, prep_ms = 0, dedisp_ms = 0, sps_ms = 0, h2h_ms = 0;
    uint64_t h2d_bytes = 0, d2h_bytes = 0, dedisp_launches = 0, sps_launches = 0, prep_launches = 0, h2h_bytes = 0;
};

}  // namespace

struct aa_plan {
    aa_plan_desc desc{};
    std::vector<aa_dm_range> ranges_in;
    std::vector<int32_t> widths;
    std::vector<uint32_t> taps_in;
    std::vector<Range> ranges;
    std::vector<int> bins;            // distinct bins > 1
    WidthTable wt{};
    int wmax = 1;
    uint64_t maxshift = 0, t_valid = 0, halo = 0, L = 0, n_sub = 0, ring_len = 0, ring_pitch = 0;
    uint64_t pitchD = 0, d_rows = 0, cap = 0, tap_row_len = 0, tap_stage_elems = 0;
    std::vector<uint64_t> pitch_b;
    uint32_t norm_block = 65536;
    int nbits = 8, planes = 1;        // planes: 8-bit planes the input is processed as (2 for 16-bit samples)
    uint64_t row_bytes = 0;           // bytes of one input time sample (all channels)
    bool big = false;                 // a block's sum of squares may pass 2^63: 128-bit statistics
    bool peaks = false;               // output_mode 1: lists are thinned on the device (reading A17)
    int pk_shift = 5, pk_nbk = 1;     // bucket grid of the peak kernels: 2^shift raw samples per bucket, buckets per row
    uint32_t wmax_raw = 1;            // longest boxcar in raw samples
    std::atomic<uint64_t> total_raw{0};
    int n_streams = 1;
    uint64_t arena_bytes = 0, pinned_bytes = 0;
    void *arena = nullptr;
    bool own_arena = false;
    uint8_t *d_ring = nullptr;
    uint64_t ring_plane_bytes = 0;    // distance of the high-byte ring from the low-byte ring
    std::vector<Stream> streams;
    std::vector<cudaEvent_t> ev_loaded, ev_dedisp, ev_copied;
    std::unique_ptr<std::atomic<int>[]> loaded, done, dedisp_issued, copied;
    std::atomic<int> error{0};
    std::atomic<uint64_t> out_pos{0}, total{0};
    std::atomic<int> overflow{0};
    aa_stats stats{};
    cudaEvent_t ev_start = nullptr;           // recorded on stream 0 when a run begins: origin of the timeline
    std::vector<aa_subchunk_times> timeline;  // one entry per sub-chunk, written by its stream's thread

    // Host threads are created once, here, and parked between runs (one host thread per stream; SURVEY
    // 8(b): aa_run allocates nothing and creates nothing).  `workers[s]` serves stream s; `helpers` copy tapped rows.
    int device = 0;
    enum class Cmd { none, run, scatter, copyback, quit };
    struct Job {                              // what the current aa_run call asked for
        const uint8_t *input = nullptr;
        int mode = 0;
        aa_candidate *out = nullptr;
        uint64_t max_cands = 0;
        uint32_t *tap_out = nullptr;
        uint64_t stored = 0;
    } job;
    std::vector<std::thread> workers;
    std::mutex mu;
    std::condition_variable cv_go, cv_done;
    Cmd cmd = Cmd::none;
    uint64_t seq = 0;                         // bumped with every command
    int pending = 0, nactive = 0;
    // helper pool for the host-to-host copies of dense planes
    struct CopyJob { const Stream *S; uint32_t *tap_out; size_t a, b; std::atomic<int> *left; };
    std::vector<std::thread> helpers;
    std::mutex hmu;
    std::condition_variable hcv;
    std::vector<CopyJob> hq;                  // fixed capacity, reserved at plan creation
    bool hquit = false;
    // final ordering without a global sort: every sub-chunk's list is sorted by its stream's thread while the GPU
    // works on, `run_cnt[j][d]` counts its records per trial, and the runs are interleaved through `scratch`
    struct Run { uint64_t pos = 0, n = 0; };
    std::vector<Run> runs;                    // [n_sub]
    std::vector<uint32_t> run_cnt;            // [n_sub][ndms_total + 1] start offset of trial d inside run j
    std::vector<uint64_t> dm_dst;             // [ndms_total + 1] first output record of trial d
    aa_candidate *scratch = nullptr;
    uint64_t scratch_cap = 0;
    uint32_t ndms_total = 0;
};

namespace {

#define AA_CUDA(call)                                   \
    do {                                                \
        cudaError_t e_ = (call);                        \
        if (e_ != cudaSuccess) {                        \
            g_last_cuda_error = (int)e_;                \
            return AA_ERR_CUDA;                         \
        }                                               \
    } while (0)

// Builds everything that depends only on the descriptor: validation, delay tables, geometry,
// buffer sizes.  Fills `p` (no CUDA calls).  Returns aa_status.
int build_geometry(aa_plan &p, const aa_plan_desc *d)
{
    if (!d || d->nchans < 1 || d->nsamp < 1 || !(d->tsamp > 0) || !(d->f_top > 0) || !(d->foff < 0))
        return AA_ERR_INVALID;
    if (!(d->f_top + (d->nchans - 1) * d->foff > 0)) return AA_ERR_INVALID;
    if (d->nranges < 1 || !d->ranges || d->nwidths < 1 || d->nwidths > kMaxWidths || !d->widths)
        return AA_ERR_INVALID;
    if (d->n_streams < 1 || d->n_streams > 64 || d->chunk_len < 1) return AA_ERR_INVALID;
    if (d->ntap < 0 || (d->ntap > 0 && !d->tap_dm_indices)) return AA_ERR_INVALID;
    if (d->dedisp_variant < AA_DEDISP_AUTO || d->dedisp_variant > AA_DEDISP_WS1024) return AA_ERR_INVALID;
    if (d->nsamp > 0xFFFFFFFFull) return AA_ERR_INVALID;       // candidates carry 32-bit sample indices

    p.desc = *d;
    p.ranges_in.assign(d->ranges, d->ranges + d->nranges);
    p.widths.assign(d->widths, d->widths + d->nwidths);
    p.taps_in.assign(d->tap_dm_indices, d->tap_dm_indices + d->ntap);
    p.desc.ranges = p.ranges_in.data();
    p.desc.widths = p.widths.data();
    p.desc.tap_dm_indices = p.taps_in.data();
    p.n_streams = d->n_streams;
    p.norm_block = d->norm_block ? d->norm_block : 65536u;
    p.nbits = d->nbits ? d->nbits : 8;
    if (p.nbits != 4 && p.nbits != 8 && p.nbits != 16) return AA_ERR_INVALID;
    if (p.nbits == 4 && (d->nchans & 1)) return AA_ERR_INVALID;
    p.planes = p.nbits == 16 ? 2 : 1;
    p.row_bytes = (uint64_t)d->nchans * (uint64_t)p.nbits / 8;
    const uint64_t maxsample = (1ull << p.nbits) - 1;

    if (d->width_decimation < 0 || d->sigma_mode < 0 || d->sigma_mode > 1) return AA_ERR_INVALID;
    for (int j = 0; j < d->nwidths; ++j) {
        if (p.widths[j] < 1 || (j && p.widths[j] <= p.widths[j - 1])) return AA_ERR_INVALID;
        p.wt.w[j] = p.widths[j];
        int dec = 1;                                  // reading A20: the time grid of a width above wdec
        if (d->width_decimation > 0)
            while ((int64_t)p.widths[j] > (int64_t)d->width_decimation * dec) dec *= 2;
        p.wt.dec[j] = dec;
    }
    for (int j = d->nwidths; j < kMaxWidths; ++j) p.wt.dec[j] = 1;
    p.wmax = p.widths.back();
    if (p.wmax > 4096) return AA_ERR_INVALID;

    uint64_t lcm = 1;
    int bin_max = 1;
    for (auto &r : p.ranges_in) {
        if (r.ndms < 1 || r.ndms > 65535 || r.bin < 1 || r.bin > 128 || !(r.dm_step >= 0) || !(r.dm_low >= 0))
            return AA_ERR_INVALID;
        if (p.norm_block % r.bin) return AA_ERR_INVALID;
        if (maxsample * d->nchans * r.bin >= (1ull << 32)) return AA_ERR_INVALID;
        lcm = lcm / gcd64(lcm, r.bin) * r.bin;
        bin_max = std::max(bin_max, r.bin);
    }
    if (p.norm_block % kAlign || p.norm_block % lcm) return AA_ERR_INVALID;
    // exact 64-bit sum of squares per block: norm_block*bin*(255*nchans)^2 < 2^63
    {
        // beyond it (16-bit input on thousands of channels) the statistics take 128-bit sums, in the generic SPS kernel
        long double bound = (long double)p.norm_block * bin_max * (long double)maxsample * (long double)maxsample * d->nchans * d->nchans;
        p.big = bound >= 9.2e18L;
        if (p.big && p.nbits != 16) return AA_ERR_INVALID;
    }

    // delay tables: delta(c,i) = floor(((4.148808e3*DM_i)*(1/f_c^2 - 1/f_top^2))/(tsamp*bin) + 0.5)
    // in double, each operation rounded separately (north_star).
    p.ranges.resize(d->nranges);
    uint32_t base = 0;
    p.maxshift = 0;
    std::vector<double> g(d->nchans);
    for (int c = 0; c < d->nchans; ++c) {
        const double f = d->f_top + (double)c * d->foff;
        const double a = 1.0 / (f * f);
        const double b = 1.0 / (d->f_top * d->f_top);
        g[c] = a - b;
    }
    for (int ri = 0; ri < d->nranges; ++ri) {
        Range &R = p.ranges[ri];
        R.r = p.ranges_in[ri];
        R.dm_base = base;
        base += (uint32_t)R.r.ndms;
        R.h_delays.resize((size_t)R.r.ndms * d->nchans);
        const double ts = d->tsamp * (double)R.r.bin;
        int64_t mx = 0;
        for (int i = 0; i < R.r.ndms; ++i) {
            const double prod = (double)i * R.r.dm_step;
            const double dm = R.r.dm_low + prod;
            const double kdm = 4.148808e3 * dm;
            for (int c = 0; c < d->nchans; ++c) {
                const double num = kdm * g[c];
                const double v = num / ts;
                const double rounded = std::floor(v + 0.5);
                if (!(rounded >= 0) || rounded > 1.0e9) return AA_ERR_INVALID;
                R.h_delays[(size_t)i * d->nchans + c] = (int32_t)rounded;
                mx = std::max<int64_t>(mx, (int64_t)rounded);
            }
        }
        R.maxdelay = (int32_t)mx;
        p.maxshift = std::max<uint64_t>(p.maxshift, (uint64_t)mx * R.r.bin);
    }
    p.maxshift = round_up(p.maxshift, lcm);
    if (p.maxshift >= d->nsamp) return AA_ERR_INVALID;
    p.t_valid = d->nsamp - p.maxshift;

    p.halo = round_up(p.maxshift + (uint64_t)(p.wmax - 1) * bin_max, std::max<uint64_t>(lcm, kAlign));
    if (d->chunk_len % d->n_streams) return AA_ERR_INVALID;
    p.L = d->chunk_len / d->n_streams;
    if (p.L % p.norm_block || p.L < p.halo) return AA_ERR_INVALID;
    p.n_sub = (p.t_valid + p.L - 1) / p.L;
    const uint64_t n_slots = std::min<uint64_t>((uint64_t)p.n_streams + 1, p.n_sub + 1);
    p.ring_len = n_slots * p.L;

    // taps
    for (int k = 0; k < d->ntap; ++k) {
        const uint32_t gi = p.taps_in[k];
        if (k && gi <= p.taps_in[k - 1]) return AA_ERR_INVALID;
        bool found = false;
        for (auto &R : p.ranges)
            if (gi >= R.dm_base && gi < R.dm_base + (uint32_t)R.r.ndms) {
                R.taps.emplace_back((int)(gi - R.dm_base), k);
                found = true;
            }
        if (!found) return AA_ERR_INVALID;
    }

    // per-range kernel configuration
    p.bins.clear();
    int max_row_u8 = 0;
    p.d_rows = 0;
    uint64_t max_cols = 0;
    p.tap_row_len = 0;
    p.tap_stage_elems = 0;
    for (auto &R : p.ranges) {
        R.nout = p.t_valid / R.r.bin;
        R.in16 = R.r.bin > 1;
        R.flush_ch = (int)((65535 / (255 * R.r.bin)) & ~1);
        if (R.flush_ch < 2) return AA_ERR_INVALID;
        R.wide = (long double)maxsample * d->nchans * R.r.bin * p.wmax >= 4294967296.0L;
        R.small31 = (long double)maxsample * d->nchans * R.r.bin * p.wmax < 2147483648.0L;
        // sigma_mode 1 (reading A18) runs everywhere: in the cluster kernel where the block fits its shared memory
        // (32-bit boxcar sums, block a multiple of 4 C with segments of at most 16384 samples), else in the generic
        // kernel, which sweeps the block once per pass of the estimator (64-bit sums, odd or very long blocks).
        if (R.in16) {
            auto it = std::find(p.bins.begin(), p.bins.end(), R.r.bin);
            if (it == p.bins.end()) { p.bins.push_back(R.r.bin); R.bin_slot = (int)p.bins.size() - 1; }
            else R.bin_slot = (int)(it - p.bins.begin());
        }
        // largest delay spread inside a block of DB trials decides the staged row length
        bool ok = false;
        for (int dpw : {4, 2, 1}) {
            const int DB = dpw * (kDedispThreads / 32);
            int spread = 0;
            for (int d0 = 0; d0 < R.r.ndms; d0 += DB) {
                const int d1 = std::min(d0 + DB, R.r.ndms) - 1;
                const int32_t *a = &R.h_delays[(size_t)d0 * d->nchans];
                const int32_t *b = &R.h_delays[(size_t)d1 * d->nchans];
                for (int c = 0; c < d->nchans; ++c) spread = std::max(spread, b[c] - a[c]);
            }
            const int row = (int)round_up((uint64_t)kDedispTB + spread + kAlign + 1, 16);
            if (dedisp_smem_bytes(R.in16, dpw, row) <= 110 * 1024 || (dpw == 1 && dedisp_smem_bytes(R.in16, dpw, row) <= 227 * 1024)) {
                R.dpw = dpw; R.row = row; ok = true;
                break;
            }
        }
        if (!ok) return AA_ERR_INVALID;     // DM step too coarse for the staged window
        {
            // tiled copy of the delay table: one contiguous [DB][CS] tile per (DM block, channel stage),
            // trials clamped to the last one, channels past nchans zero -> one bulk copy per stage
            const int DB = R.dpw * (kDedispThreads / 32), CS = dedisp_stage_channels(R.in16);
            const int nblk = (R.r.ndms + DB - 1) / DB, nst = (d->nchans + CS - 1) / CS;
            R.h_dtiles.assign((size_t)nblk * nst * DB * CS, 0);
            for (int b = 0; b < nblk; ++b)
                for (int st = 0; st < nst; ++st)
                    for (int dl = 0; dl < DB; ++dl) {
                        const int dd = std::min(b * DB + dl, R.r.ndms - 1);
                        for (int cl = 0; cl < CS; ++cl) {
                            const int c = st * CS + cl;
                            if (c < d->nchans)
                                R.h_dtiles[(((size_t)b * nst + st) * DB + dl) * CS + cl] = R.h_delays[(size_t)dd * d->nchans + c];
                        }
                    }
        }
        // shared-pattern kernels: tables within limits, rows within shared memory.  desc.dedisp_variant restricts
        // the choice to one kernel family (A/B timing, tests).
        R.sp_tb = 0;
        R.ws = false;
        {
            const int force = d->dedisp_variant;
            auto allowed = [&](int v) { return force == AA_DEDISP_AUTO || force == v; };
            // 16-bit lanes take floor(65535 / (255 bin 4)) groups between flushes into the TMEM tile.  Only with fewer
            // than 4 (bin 32) the 32-bit-accumulator variant (512-sample tiles, no flush) is the faster one.  Measured
            // on cfg4, seconds per step: wide for bin >= 4: 2.17, >= 16: 2.08, 32 only: 2.07, never: 2.08 (with the
            // earlier L2 read-modify-write flushes: wide for bin >= 4 was best, and bins 16 / 32 on 16-bit lanes lost
            // to the plain kernel).
            // The producers add the four channels of a group in 16-bit lanes: binned samples need 4 * 255 * bin < 2^16,
            // i.e. bin <= 64; coarser bins run on the plain kernel.
            const bool ws_ok = !R.in16 || 4ull * 255 * R.r.bin <= 65535;
            R.ws_wide = R.in16 && ws_ok && 65535 / (255 * R.r.bin * kSpG) < 4;
            // time tile: 1024 samples unless the range is so short per sub-chunk that 512-sample tiles (about 0.65 of
            // the time per CTA) need fewer waves of CTAs over the 148 SMs
            const uint64_t cols = p.L / (uint64_t)R.r.bin + (uint64_t)p.wmax - 1, nblk = ((uint64_t)R.r.ndms + kSpDB - 1) / kSpDB;
            const double cost1024 = (double)(((cols + 1023) / 1024 * nblk + 147) / 148);
            const double cost512 = 0.65 * (double)(((cols + 511) / 512 * nblk + 147) / 148);
            const int order[2] = {cost512 < cost1024 ? 512 : 1024, cost512 < cost1024 ? 1024 : 512};
            for (int tb : order) {
                if (R.ws_wide ? (tb != 512 || !(allowed(AA_DEDISP_WS1024) || allowed(AA_DEDISP_WS512)))
                              : !allowed(tb == 1024 ? AA_DEDISP_WS1024 : AA_DEDISP_WS512))
                    continue;
                if (!ws_ok || R.sp_tb) continue;
                if (ws_build_tables(R.h_delays.data(), R.r.ndms, d->nchans, tb, R.in16 ? 2 : 1, 226 * 1024, R.h_ws, R.sp_rows,
                                    R.sp_pbytes)) {
                    R.sp_tb = tb;
                    R.ws = true;
                }
            }
            if (!R.ws) { R.h_ws.clear(); R.h_ws.shrink_to_fit(); }
            for (int tb : {1024, 512}) {
                if (R.in16 || R.sp_tb || !allowed(tb == 1024 ? AA_DEDISP_SP1024 : AA_DEDISP_SP512)) continue;
                const size_t limit = tb == 1024 ? 227 * 1024 : 113 * 1024;
                if (sp_build_tables(R.h_delays.data(), R.r.ndms, d->nchans, tb, R.h_sp, R.sp_rows, R.sp_pbytes) &&
                    dedisp_sp_smem_bytes(R.sp_rows, R.sp_pbytes) + 1024 <= limit)
                    R.sp_tb = tb;
            }
            if (!R.sp_tb || R.ws) { R.h_sp.clear(); R.h_sp.shrink_to_fit(); }
            if (R.sp_tb) R.sp_flush = std::max(1, 65535 / (255 * R.r.bin * kSpG));
            if (!R.ws) R.ws_wide = false;
        }
        if (!R.in16) max_row_u8 = std::max(max_row_u8, std::max(R.row, R.sp_tb ? R.sp_rows + R.sp_tb : 0));
        p.d_rows = std::max<uint64_t>(p.d_rows, (uint64_t)R.r.ndms);
        max_cols = std::max<uint64_t>(max_cols, p.L / R.r.bin + p.wmax - 1);
        if (!R.taps.empty()) {
            p.tap_row_len = std::max<uint64_t>(p.tap_row_len, R.nout);
            p.tap_stage_elems += (uint64_t)R.taps.size() * (p.L / R.r.bin);
        }
    }
    p.pitchD = round_up(max_cols + 8, 64);
    p.ring_pitch = round_up(p.ring_len + p.halo + (uint64_t)max_row_u8 + kDedispTB + 64, 256);
    p.pitch_b.resize(p.bins.size());
    for (size_t k = 0; k < p.bins.size(); ++k) {
        int max_row = 0;
        for (auto &R : p.ranges)
            if (R.bin_slot == (int)k) max_row = std::max(max_row, std::max(R.row, R.sp_tb ? R.sp_rows + R.sp_tb : 0));
        p.pitch_b[k] = round_up((p.L + p.halo) / p.bins[k] + max_row + kDedispTB + 64, 128);
    }
    p.cap = d->max_cands_per_subchunk ? d->max_cands_per_subchunk : (1ull << 21);
    if (p.cap > (1ull << 30)) return AA_ERR_INVALID;
    if (d->output_mode < 0 || d->output_mode > 1) return AA_ERR_INVALID;
    if (d->sps_variant < 0 || d->sps_variant > 1 || d->reserved0 != 0) return AA_ERR_INVALID;
    p.peaks = d->output_mode == 1;
    p.wmax_raw = (uint32_t)p.wmax * (uint32_t)bin_max;
    p.pk_shift = 5;
    while (((p.L - 1) >> p.pk_shift) + 1 > 4096) ++p.pk_shift;
    p.pk_nbk = (int)(((p.L - 1) >> p.pk_shift) + 1);
    uint64_t ndms_all = 0;
    for (auto &R : p.ranges) ndms_all += (uint64_t)R.r.ndms;
    if (ndms_all >= (1ull << 30)) return AA_ERR_INVALID;       // the two top bits of dm_index carry the peak flags

    // arena layout (256-byte aligned bump allocation, computed identically in carve())
    uint64_t off = 0;
    auto take = [&](uint64_t bytes) { off = round_up(off, 256) + bytes; };
    p.ring_plane_bytes = round_up(round_up((uint64_t)d->nchans, kRingChPad) * p.ring_pitch, 256);
    take(p.ring_plane_bytes * (uint64_t)p.planes);              // zero rows pad the channels to a multiple of 8
    for (auto &R : p.ranges) {
        take((uint64_t)R.r.ndms * d->nchans * 4);
        take((uint64_t)R.h_dtiles.size() * 4);
        take((uint64_t)R.sp_table_bytes());
    }
    for (int s = 0; s < p.n_streams; ++s) {
        take((p.L + p.halo) * p.row_bytes);
        for (int pl = 0; pl < p.planes; ++pl)
            for (size_t k = 0; k < p.bins.size(); ++k) take(round_up((uint64_t)d->nchans, kSpG) * p.pitch_b[k] * 2);
        take(p.d_rows * p.pitchD * 4);
        if (p.planes == 2) take(p.d_rows * p.pitchD * 4);
        take(p.cap * sizeof(aa_candidate));
        take(256);
        if (p.peaks) {
            take(ndms_all * (uint64_t)p.pk_nbk * 4);
            take(p.cap * 4);
            take(p.cap * sizeof(aa_candidate));
        }
    }
    p.arena_bytes = round_up(off, 256);
    p.pinned_bytes = (uint64_t)p.n_streams * (256 + p.cap * sizeof(aa_candidate) + p.tap_stage_elems * 4 +
                                              (d->stage_input ? (p.L + p.halo) * p.row_bytes : 0));
    return AA_OK;
}

void carve(aa_plan &p)
{
    uint8_t *base = static_cast<uint8_t *>(p.arena);
    uint64_t off = 0;
    auto take = [&](uint64_t bytes) { off = round_up(off, 256); uint8_t *q = base + off; off += bytes; return q; };
    const int nchans = p.desc.nchans;
    p.d_ring = take(p.ring_plane_bytes * (uint64_t)p.planes);
    for (auto &R : p.ranges) {
        R.d_delays = reinterpret_cast<int32_t *>(take((uint64_t)R.r.ndms * nchans * 4));
        R.d_dtiles = reinterpret_cast<int32_t *>(take((uint64_t)R.h_dtiles.size() * 4));
        R.d_sp = take((uint64_t)R.sp_table_bytes());
    }
    for (auto &S : p.streams) {
        S.d_raw = take((p.L + p.halo) * p.row_bytes);
        S.d_binned.resize(p.bins.size() * (size_t)p.planes);          // [plane][bin slot]
        for (int pl = 0; pl < p.planes; ++pl)
            for (size_t k = 0; k < p.bins.size(); ++k)
                S.d_binned[(size_t)pl * p.bins.size() + k] =
                    reinterpret_cast<uint16_t *>(take(round_up((uint64_t)nchans, kSpG) * p.pitch_b[k] * 2));
        S.d_D = reinterpret_cast<uint32_t *>(take(p.d_rows * p.pitchD * 4));
        if (p.planes == 2) S.d_D2 = reinterpret_cast<uint32_t *>(take(p.d_rows * p.pitchD * 4));
        S.d_cands = reinterpret_cast<aa_candidate *>(take(p.cap * sizeof(aa_candidate)));
        S.d_count = reinterpret_cast<uint32_t *>(take(256));
        if (p.peaks) {
            uint64_t ndms_all = 0;
            for (auto &R : p.ranges) ndms_all += (uint64_t)R.r.ndms;
            S.d_head = reinterpret_cast<int32_t *>(take(ndms_all * (uint64_t)p.pk_nbk * 4));
            S.d_next = reinterpret_cast<uint32_t *>(take(p.cap * 4));
            S.d_peaks = reinterpret_cast<aa_candidate *>(take(p.cap * sizeof(aa_candidate)));
        }
    }
}

void destroy_plan(aa_plan *p)
{
    if (!p) return;
    if (!p->workers.empty()) {
        {
            std::lock_guard<std::mutex> lk(p->mu);
            p->cmd = aa_plan::Cmd::quit;
            ++p->seq;
        }
        p->cv_go.notify_all();
        for (auto &t : p->workers) t.join();
    }
    if (!p->helpers.empty()) {
        {
            std::lock_guard<std::mutex> lk(p->hmu);
            p->hquit = true;
        }
        p->hcv.notify_all();
        for (auto &t : p->helpers) t.join();
    }
    std::free(p->scratch);
    for (auto &S : p->streams) {
        if (S.st) cudaStreamSynchronize(S.st);
        for (auto e : S.ev) if (e) cudaEventDestroy(e);
        if (S.h_count) cudaFreeHost(S.h_count);
        if (S.h_cands) cudaFreeHost(S.h_cands);
        if (S.h_tap) cudaFreeHost(S.h_tap);
        if (S.h_stage) cudaFreeHost(S.h_stage);
        if (S.own && S.st) cudaStreamDestroy(S.st);
    }
    for (auto e : p->ev_loaded) if (e) cudaEventDestroy(e);
    for (auto e : p->ev_dedisp) if (e) cudaEventDestroy(e);
    for (auto e : p->ev_copied) if (e) cudaEventDestroy(e);
    if (p->ev_start) cudaEventDestroy(p->ev_start);
    if (p->own_arena && p->arena) cudaFree(p->arena);
    delete p;
}

// NVTX ranges: a profiler's timeline shows the call and, per stream thread, every sub-chunk; without a
// profiler attached the calls return at once
struct NvtxRange {
    explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
    NvtxRange(const NvtxRange &) = delete;
    NvtxRange &operator=(const NvtxRange &) = delete;
};

// order of the returned list: (dm_index, t_start); the two top bits of dm_index may carry peak flags on the way
inline bool cand_less(const aa_candidate &a, const aa_candidate &b)
{
    const uint32_t da = a.dm_index & kPeakDmMask, db = b.dm_index & kPeakDmMask;
    return da != db ? da < db : a.t_start < b.t_start;
}

inline bool wait_flag(aa_plan *p, std::atomic<int> &f)
{
    int spins = 0;
    while (!f.load(std::memory_order_acquire)) {
        if (p->error.load(std::memory_order_relaxed)) return false;
        if (++spins < 200) std::this_thread::yield();
        else std::this_thread::sleep_for(std::chrono::microseconds(20));
    }
    return true;
}

#define AA_W(call)                                                       \
    do {                                                                 \
        cudaError_t e_ = (call);                                         \
        if (e_ != cudaSuccess) {                                         \
            int z_ = 0;                                                  \
            p->error.compare_exchange_strong(z_, (int)e_);               \
            return;                                                      \
        }                                                                \
    } while (0)

// One stream's host thread: issues every sub-chunk j = s, s+n_streams, ... and copies its results out.
enum class Input { pinned, resident, staged };

void worker(aa_plan *p, int s, const uint8_t *input, Input mode, aa_candidate *out, uint64_t max_cands,
            uint32_t *tap_out)
{
    const bool resident = mode == Input::resident, staged = mode == Input::staged;
    Stream &S = p->streams[s];
    cudaStream_t st = S.st;
    const uint64_t L = p->L, halo = p->halo, R = p->ring_len, nsamp = p->desc.nsamp;
    const int nchans = p->desc.nchans;
    const int nr = (int)p->ranges.size();

    // input rows [t_first, t_last) that sub-chunk j brings in (its own span shifted by the halo; j = 0 also the halo)
    auto new_rows = [&](uint64_t j, uint64_t &t_first, uint64_t &nt) {
        t_first = j == 0 ? 0 : j * L + halo;
        const uint64_t t_last = std::min<uint64_t>((j + 1) * L + halo, nsamp);
        nt = t_last > t_first ? t_last - t_first : 0;
    };
    // host -> pinned staging copy of sub-chunk j's rows by this stream's thread
    auto stage = [&](uint64_t j) {
        uint64_t t_first, nt;
        new_rows(j, t_first, nt);
        if (!nt) return;
        const auto c0 = std::chrono::steady_clock::now();
        std::memcpy(S.h_stage, input + t_first * p->row_bytes, nt * p->row_bytes);
        S.h2h_ms += std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - c0).count();
        S.h2h_bytes += nt * p->row_bytes;
    };
    if (staged && (uint64_t)s < p->n_sub) stage((uint64_t)s);

    for (uint64_t j = (uint64_t)s; j < p->n_sub; j += (uint64_t)p->n_streams) {
        NvtxRange nvtx_sub("aa: sub-chunk (H2D, corner turn, dedispersion, SPS, D2H, host stage)");
        // the new rows overwrite ring columns last read by sub-chunks j-n_streams-1 and j-n_streams
        if (j >= (uint64_t)p->n_streams + 1 && !wait_flag(p, p->done[j - p->n_streams - 1])) return;

        uint64_t t_first, nt;
        new_rows(j, t_first, nt);
        const uint8_t *src = staged ? S.h_stage : input + t_first * p->row_bytes;

        // First round only (every stream is idle and would start its copy at once): the copies take the link one
        // after the other in sub-chunk order, so that sub-chunk 0 is complete after 1/n_streams of the time.
        const bool first_round = !resident && j < (uint64_t)p->n_streams;
        if (first_round && j > 0) {
            if (!wait_flag(p, p->copied[j - 1])) return;
            AA_W(cudaStreamWaitEvent(st, p->ev_copied[j - 1], 0));
        }
        AA_W(cudaEventRecord(S.ev[0], st));
        if (!resident && nt) {
            AA_W(cudaMemcpyAsync(S.d_raw, src, nt * p->row_bytes, cudaMemcpyHostToDevice, st));
            S.h2d_bytes += nt * p->row_bytes;
            src = S.d_raw;
        }
        AA_W(cudaEventRecord(S.ev[1], st));
        if (first_round) {
            AA_W(cudaEventRecord(p->ev_copied[j], st));
            p->copied[j].store(1, std::memory_order_release);
        }
        AA_W(launch_corner_turn(src, (int64_t)nt, nchans, p->nbits, (int64_t)t_first, p->d_ring, p->d_ring + p->ring_plane_bytes,
                                (int64_t)p->ring_pitch, (int64_t)R, (int64_t)halo, st));
        S.prep_launches += nt ? 1 : 0;
        AA_W(cudaEventRecord(S.ev[2], st));
        AA_W(cudaEventRecord(p->ev_loaded[j], st));
        p->loaded[j].store(1, std::memory_order_release);

        // the window [jL, (j+1)L + halo) also needs the rows loaded by sub-chunk j-1's stream
        if (j > 0) {
            if (!wait_flag(p, p->loaded[j - 1])) return;
            AA_W(cudaStreamWaitEvent(st, p->ev_loaded[j - 1], 0));
        }
        // Dedispersion kernels fill the GPU: run them in sub-chunk order, each after the previous sub-chunk's
        // last one.  Left to themselves the streams' kernels share the SMs, finish together and then all
        // streams start their next copy at the same moment (a convoy: link and SMs idle in turn).
        if (j > 0) {
            if (!wait_flag(p, p->dedisp_issued[j - 1])) return;
            AA_W(cudaStreamWaitEvent(st, p->ev_dedisp[j - 1], 0));
        }
        const uint64_t col0 = (j * L) % R;
        const uint64_t in_len = std::min<uint64_t>(L + halo, nsamp - j * L);

        AA_W(cudaEventRecord(S.ev[3], st));
        for (int pl = 0; pl < p->planes; ++pl) {
            // power-of-two bins up to 32 share one pass over the ring; anything else is binned on its own
            const uint8_t *ring_pl = p->d_ring + (uint64_t)pl * p->ring_plane_bytes;
            uint16_t *const *binned = &S.d_binned[(size_t)pl * p->bins.size()];
            BinMultiArgs ba{};
            bool any = false;
            for (size_t k = 0; k < p->bins.size(); ++k) {
                const int b = p->bins[k];
                int l = -1;
                for (int q = 0; q < 5; ++q) if (b == (2 << q)) l = q;
                if (l >= 0 && col0 % 16 == 0 && p->pitch_b[k] % 16 == 0) {
                    ba.out[l] = binned[k];
                    ba.pitch[l] = (int64_t)p->pitch_b[k];
                    ba.nbinned[l] = (int64_t)(in_len / b);
                    any = true;
                } else {
                    AA_W(launch_bin(ring_pl, (int64_t)p->ring_pitch, (int64_t)col0, nchans, b, (int64_t)(in_len / b),
                                    binned[k], (int64_t)p->pitch_b[k], st));
                    S.prep_launches++;
                }
            }
            if (any) {
                ba.ring = ring_pl;
                ba.ring_pitch = (int64_t)p->ring_pitch;
                ba.col0 = (int64_t)col0;
                ba.ngroups = (int64_t)((in_len + 31) / 32);
                AA_W(launch_bin_multi(ba, nchans, st));
                S.prep_launches++;
            }
        }
        AA_W(cudaEventRecord(S.ev[4], st));
        AA_W(cudaMemsetAsync(S.d_count, 0, sizeof(uint32_t), st));

        uint64_t tap_off = 0;
        auto &tapcopies = S.tapcopies;
        tapcopies.clear();                         // capacity reserved at plan creation
        for (int ri = 0; ri < nr; ++ri) {
            Range &Rg = p->ranges[ri];
            const uint64_t b = (uint64_t)Rg.r.bin;
            const uint64_t tau0 = j * L / b;
            cudaEvent_t e0 = S.ev[kEvFixed + 3 * ri], e1 = S.ev[kEvFixed + 3 * ri + 1], e2 = S.ev[kEvFixed + 3 * ri + 2];
            AA_W(cudaEventRecord(e0, st));
            if (tau0 < Rg.nout) {
                const uint64_t left = Rg.nout - tau0;
                const uint64_t nemit = std::min<uint64_t>(L / b, left);
                const uint64_t ncols = std::min<uint64_t>(L / b + p->wmax - 1, left);
                for (int pl = 0; pl < p->planes; ++pl) {
                    DedispArgs da{};
                    da.in = Rg.in16 ? (const void *)S.d_binned[(size_t)pl * p->bins.size() + Rg.bin_slot]
                                    : (const void *)(p->d_ring + (uint64_t)pl * p->ring_plane_bytes);
                    da.pitch_in = Rg.in16 ? (int64_t)p->pitch_b[Rg.bin_slot] : (int64_t)p->ring_pitch;
                    da.col0 = Rg.in16 ? 0 : (int64_t)col0;
                    da.delays = Rg.d_delays;
                    da.dtiles = Rg.d_dtiles;
                    da.nchans = nchans;
                    da.ndms = Rg.r.ndms;
                    da.ncols = (int32_t)ncols;
                    da.out = pl ? S.d_D2 : S.d_D;
                    da.pitch_out = (int64_t)p->pitchD;
                    da.row = Rg.row;
                    da.flush_ch = Rg.flush_ch;
                    da.sp_tab = Rg.d_sp;
                    da.sp_rows = Rg.sp_rows;
                    da.sp_pbytes = Rg.sp_pbytes;
                    da.sp_flush = Rg.sp_flush;
                    if (Rg.ws) AA_W(launch_dedisp_ws(da, Rg.sp_tb, Rg.in16, Rg.ws_wide, st));
                    else if (Rg.sp_tb) AA_W(launch_dedisp_sp(da, Rg.sp_tb, st));
                    else AA_W(launch_dedisp(da, Rg.in16, Rg.dpw, st));
                    S.dedisp_launches++;
                }
                // 16-bit input: D = D(low bytes) + 256 D(high bytes)
                if (p->planes == 2) AA_W(launch_combine_planes(S.d_D, S.d_D2, (int64_t)p->pitchD, Rg.r.ndms, (int32_t)ncols, st));
                AA_W(cudaEventRecord(e1, st));
                if (ri == nr - 1) {
                    AA_W(cudaEventRecord(p->ev_dedisp[j], st));
                    p->dedisp_issued[j].store(1, std::memory_order_release);
                }
                SpsArgs sa{};
                sa.D = S.d_D;
                sa.pitch = (int64_t)p->pitchD;
                sa.ndms = Rg.r.ndms;
                sa.ncols = (int32_t)ncols;
                sa.nemit = (int32_t)nemit;
                sa.nout_left = (int64_t)left;
                sa.block_len = (int32_t)(p->norm_block / b);
                sa.nwidths = (int32_t)p->widths.size();
                sa.wmax = p->wmax;
                sa.thr = p->desc.snr_threshold;
                sa.dm_base = Rg.dm_base;
                sa.tau0 = (uint32_t)tau0;
                sa.bin = (uint32_t)b;
                sa.cands = S.d_cands;
                sa.count = S.d_count;
                sa.cap = (uint32_t)p->cap;
                sa.sigma_mode = p->desc.sigma_mode;
                sa.maxval = (uint32_t)(((1ull << p->nbits) - 1) * (uint64_t)nchans * b);
                AA_W(launch_sps(sa, p->wt, Rg.wide, Rg.small31, p->big, p->desc.sps_variant == 1, st));
                S.sps_launches++;
                AA_W(cudaEventRecord(e2, st));
                // tapped rows: runs of consecutive trials leave in one strided copy (all rows tapped = the dense
                // DM x time plane of the sub-chunk, the paper's device-to-host path)
                for (size_t a0 = 0; a0 < Rg.taps.size();) {
                    size_t a1 = a0 + 1;
                    while (a1 < Rg.taps.size() && Rg.taps[a1].first == Rg.taps[a1 - 1].first + 1) ++a1;
                    const uint64_t nrows = a1 - a0;
                    AA_W(cudaMemcpy2DAsync(S.h_tap + tap_off, nemit * 4, S.d_D + (uint64_t)Rg.taps[a0].first * p->pitchD,
                                           p->pitchD * 4, nemit * 4, nrows, cudaMemcpyDeviceToHost, st));
                    for (size_t q = a0; q < a1; ++q) {
                        tapcopies.push_back({Rg.taps[q].second, tau0, nemit, tap_off});
                        tap_off += nemit;
                    }
                    S.d2h_bytes += nrows * nemit * 4;
                    a0 = a1;
                }
            } else {
                AA_W(cudaEventRecord(e1, st));
                AA_W(cudaEventRecord(e2, st));
                if (ri == nr - 1) {
                    AA_W(cudaEventRecord(p->ev_dedisp[j], st));
                    p->dedisp_issued[j].store(1, std::memory_order_release);
                }
            }
        }
        AA_W(cudaEventRecord(S.ev[7], st));
        if (p->peaks) {
            // thin the sub-chunk's list on the device: only peaks and border records cross the link (reading A17)
            PeakArgs pa{};
            pa.cands = S.d_cands; pa.count = S.d_count; pa.cap = (uint32_t)p->cap;
            pa.head = S.d_head; pa.next = S.d_next;
            pa.nrows = (int32_t)p->ndms_total; pa.nbk = p->pk_nbk; pa.shift = p->pk_shift;
            pa.t0 = (uint32_t)(j * L);
            pa.t1 = (uint32_t)std::min<uint64_t>((j + 1) * L, p->t_valid);
            pa.wmax_raw = p->wmax_raw;
            pa.has_left = j > 0; pa.has_right = j + 1 < p->n_sub;
            pa.out = S.d_peaks; pa.out_count = S.d_count + 1; pa.out_cap = (uint32_t)p->cap;
            AA_W(launch_peaks(pa, st));
        }
        AA_W(cudaEventRecord(S.ev[8], st));
        AA_W(cudaMemcpyAsync(S.h_count, S.d_count, 2 * sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
        if (staged && j + (uint64_t)p->n_streams < p->n_sub) {
            // the staging buffer is free once this sub-chunk's H2D is done: fill it for the next one while
            // the stream computes
            AA_W(cudaEventSynchronize(S.ev[1]));
            stage(j + (uint64_t)p->n_streams);
        }
        AA_W(cudaStreamSynchronize(st));           // stream-scoped wait, never device-wide
        p->done[j].store(1, std::memory_order_release);

        const uint64_t found_raw = S.h_count[0];
        if (found_raw > p->cap) p->overflow.store(1);
        p->total_raw.fetch_add(found_raw);
        const uint64_t found = p->peaks ? (uint64_t)S.h_count[1] : found_raw;   // records that cross the link
        const uint64_t n = std::min<uint64_t>(found, p->cap);
        AA_W(cudaEventRecord(S.ev[5], st));
        if (n) AA_W(cudaMemcpyAsync(S.h_cands, p->peaks ? S.d_peaks : S.d_cands, n * sizeof(aa_candidate), cudaMemcpyDeviceToHost, st));
        AA_W(cudaEventRecord(S.ev[6], st));
        AA_W(cudaStreamSynchronize(st));
        S.d2h_bytes += 8 + n * sizeof(aa_candidate);

        // host-to-host output stage of this stream: the sub-chunk's list goes to the caller's buffer
        // and is put in (dm_index, t_start) order right here, while the GPU works on the next sub-chunks
        p->total.fetch_add(found);
        const uint64_t pos = p->out_pos.fetch_add(n);
        uint64_t m = 0;
        if (pos < max_cands) {
            m = std::min<uint64_t>(n, max_cands - pos);
        }
        {
            // The kernel appends in no particular order.  The key (trial, start inside the sub-chunk) has few bits, so the
            // run is put in order by a least-significant-digit radix sort that ping-pongs between the pinned staging and the
            // caller's buffer (11 bits per pass, no other memory), instead of one m log m comparison sort; the table of
            // where each trial starts inside this run, which the final interleave needs, comes from one more histogram.
            p->runs[j].pos = pos < max_cands ? pos : max_cands;
            p->runs[j].n = m;
            const uint32_t nd = p->ndms_total;
            uint32_t *cnt = &p->run_cnt[j * (uint64_t)(nd + 1)];
            uint32_t *cur = S.sort_cur.data();
            aa_candidate *dst = out + pos, *src = S.h_cands;
            int tbits = 1, dbits = 1;
            while ((1ull << tbits) < L) ++tbits;
            while ((1u << dbits) < nd) ++dbits;
            const uint64_t t_sub = j * L;
            auto key = [&](const aa_candidate &c) {
                return ((uint64_t)(c.dm_index & kPeakDmMask) << tbits) | (uint64_t)(c.t_start - (uint32_t)t_sub);
            };
            bool in_range = true;
            std::fill(cur, cur + nd + 1, 0u);
            for (uint64_t i = 0; i < m; ++i) {
                const aa_candidate &c = src[i];
                const uint32_t d = c.dm_index & kPeakDmMask;
                in_range = in_range && d < nd && (uint64_t)(c.t_start - (uint32_t)t_sub) < (1ull << tbits);
                cur[std::min<uint32_t>(d, nd - 1) + 1]++;
            }
            for (uint32_t d = 0; d < nd; ++d) cur[d + 1] += cur[d];      // cur[d] = first record of trial d
            std::memcpy(cnt, cur, (size_t)(nd + 1) * sizeof(uint32_t));
            if (m && !in_range) {                       // never expected: keep the plain sort for it
                std::memcpy(dst, src, m * sizeof(aa_candidate));
                std::sort(dst, dst + m, cand_less);
            } else if (m) {
                constexpr int kDigit = 11;
                uint32_t hist[1 << kDigit];
                aa_candidate *a = src, *b = dst;
                for (int shift = 0; shift < tbits + dbits; shift += kDigit) {
                    std::memset(hist, 0, sizeof(hist));
                    for (uint64_t i = 0; i < m; ++i) hist[(key(a[i]) >> shift) & ((1u << kDigit) - 1)]++;
                    uint32_t run = 0;
                    for (uint32_t &h : hist) { const uint32_t c = h; h = run; run += c; }
                    for (uint64_t i = 0; i < m; ++i) b[hist[(key(a[i]) >> shift) & ((1u << kDigit) - 1)]++] = a[i];
                    std::swap(a, b);
                }
                if (a != dst) std::memcpy(dst, a, m * sizeof(aa_candidate));
            }
        }
        if (tap_out && !tapcopies.empty()) {
            // host-to-host copy of the tapped rows; a dense plane is hundreds of MB per sub-chunk,
            // so the stream's thread shares it with the plan's helper threads (created at plan creation)
            auto copy_rows = [&](size_t a, size_t b) {
                for (size_t i = a; i < b; ++i) {
                    const Stream::TapCopy &tc = tapcopies[i];
                    std::memcpy(tap_out + (uint64_t)tc.row * p->tap_row_len + tc.tau0, S.h_tap + tc.off, tc.n * 4);
                }
            };
            const uint64_t bytes = tap_off * 4;
            const size_t K = bytes < (64ull << 20) || p->helpers.empty()
                                 ? 1 : std::min<size_t>(1 + p->helpers.size() / (size_t)p->nactive, 4);
            if (K == 1) {
                copy_rows(0, tapcopies.size());
            } else {
                const size_t per = (tapcopies.size() + K - 1) / K;
                std::atomic<int> left{0};
                size_t inline_from = tapcopies.size();      // parts the queue has no room for are copied here
                {
                    std::lock_guard<std::mutex> lk(p->hmu);
                    for (size_t k = 1; k < K; ++k) {
                        const size_t a = std::min(k * per, tapcopies.size()), b = std::min((k + 1) * per, tapcopies.size());
                        if (a >= b) break;
                        if (p->hq.size() == p->hq.capacity()) { inline_from = a; break; }
                        left.fetch_add(1);
                        p->hq.push_back({&S, tap_out, a, b, &left});
                    }
                }
                p->hcv.notify_all();
                copy_rows(0, std::min(per, tapcopies.size()));
                copy_rows(inline_from, tapcopies.size());
                while (left.load(std::memory_order_acquire) > 0) std::this_thread::yield();
            }
        }

        float ms = 0;
        if (!resident && nt) { cudaEventElapsedTime(&ms, S.ev[0], S.ev[1]); S.h2d_ms += ms; }
        cudaEventElapsedTime(&ms, S.ev[1], S.ev[2]); S.prep_ms += ms;
        cudaEventElapsedTime(&ms, S.ev[3], S.ev[4]); S.prep_ms += ms;
        for (int ri = 0; ri < nr; ++ri) {
            cudaEventElapsedTime(&ms, S.ev[kEvFixed + 3 * ri], S.ev[kEvFixed + 3 * ri + 1]); S.dedisp_ms += ms;
            cudaEventElapsedTime(&ms, S.ev[kEvFixed + 3 * ri + 1], S.ev[kEvFixed + 3 * ri + 2]); S.sps_ms += ms;
        }
        cudaEventElapsedTime(&ms, S.ev[5], S.ev[6]); S.d2h_ms += ms;
        if (p->peaks) { cudaEventElapsedTime(&ms, S.ev[7], S.ev[8]); S.sps_ms += ms; }

        aa_subchunk_times &T = p->timeline[j];
        T = aa_subchunk_times{};
        T.index = (uint32_t)j;
        T.stream = (uint32_t)s;
        auto at = [&](cudaEvent_t e) { float v = 0; cudaEventElapsedTime(&v, p->ev_start, e); return (double)v; };
        T.h2d_begin = at(S.ev[0]); T.h2d_end = at(S.ev[1]); T.prep_end = at(S.ev[2]); T.compute_begin = at(S.ev[3]);
        T.compute_end = at(S.ev[kEvFixed + 3 * (nr - 1) + 2]); T.d2h_end = at(S.ev[6]);
        for (int ri = 0; ri < nr; ++ri) {
            cudaEventElapsedTime(&ms, S.ev[kEvFixed + 3 * ri], S.ev[kEvFixed + 3 * ri + 1]); T.dedisp_ms += ms;
            cudaEventElapsedTime(&ms, S.ev[kEvFixed + 3 * ri + 1], S.ev[kEvFixed + 3 * ri + 2]); T.sps_ms += ms;
        }
    }
}

// Sends one command to every active worker thread and waits until all of them are done with it.
void command(aa_plan *p, aa_plan::Cmd c)
{
    std::unique_lock<std::mutex> lk(p->mu);
    p->cmd = c;
    p->pending = p->nactive;
    ++p->seq;
    p->cv_go.notify_all();
    p->cv_done.wait(lk, [&] { return p->pending == 0; });
}

// Pieces of the final interleave: worker s of nactive takes every nactive-th trial (scatter) / an equal slice (copy back)
void merge_scatter(aa_plan *p, int s)
{
    const uint64_t W = (uint64_t)p->ndms_total + 1;
    const aa_candidate *out = p->job.out;
    for (uint32_t d = (uint32_t)s; d < p->ndms_total; d += (uint32_t)p->nactive) {
        uint64_t dst = p->dm_dst[d];
        for (uint64_t j = 0; j < p->n_sub; ++j) {
            const uint32_t a = p->run_cnt[j * W + d], b = p->run_cnt[j * W + d + 1];
            if (b > a) {
                std::memcpy(p->scratch + dst, out + p->runs[j].pos + a, (uint64_t)(b - a) * sizeof(aa_candidate));
                dst += b - a;
            }
        }
    }
}

void merge_copyback(aa_plan *p, int s)
{
    const uint64_t n = p->job.stored, per = (n + (uint64_t)p->nactive - 1) / (uint64_t)p->nactive;
    const uint64_t a = std::min(n, per * (uint64_t)s), b = std::min(n, a + per);
    if (b > a) std::memcpy(p->job.out + a, p->scratch + a, (b - a) * sizeof(aa_candidate));
}

// Body of the persistent host thread of stream s: parked on the condition variable between commands.
void worker_main(aa_plan *p, int s)
{
    cudaSetDevice(p->device);
    uint64_t seen = 0;
    for (;;) {
        aa_plan::Cmd c;
        {
            std::unique_lock<std::mutex> lk(p->mu);
            p->cv_go.wait(lk, [&] { return p->seq != seen; });
            seen = p->seq;
            c = p->cmd;
        }
        if (c == aa_plan::Cmd::quit) return;
        if (c == aa_plan::Cmd::run)
            worker(p, s, p->job.input, (Input)p->job.mode, p->job.out, p->job.max_cands, p->job.tap_out);
        else if (c == aa_plan::Cmd::scatter)
            merge_scatter(p, s);
        else if (c == aa_plan::Cmd::copyback)
            merge_copyback(p, s);
        {
            std::lock_guard<std::mutex> lk(p->mu);
            if (--p->pending == 0) p->cv_done.notify_all();
        }
    }
}

// Body of a helper thread: host-to-host copies of tapped rows handed over by the stream threads.
void helper_main(aa_plan *p)
{
    for (;;) {
        aa_plan::CopyJob jb;
        {
            std::unique_lock<std::mutex> lk(p->hmu);
            p->hcv.wait(lk, [&] { return p->hquit || !p->hq.empty(); });
            if (p->hq.empty()) return;           // quit
            jb = p->hq.back();
            p->hq.pop_back();
        }
        for (size_t i = jb.a; i < jb.b; ++i) {
            const Stream::TapCopy &tc = jb.S->tapcopies[i];
            std::memcpy(jb.tap_out + (uint64_t)tc.row * p->tap_row_len + tc.tau0, jb.S->h_tap + tc.off, tc.n * 4);
        }
        jb.left->fetch_sub(1, std::memory_order_release);
    }
}

// output_mode 1: `out[0..n)` is the merged list of what the sub-chunks sent, sorted by (dm_index, t_start): decided
// peaks, and border records (flagged; beaten on their own sub-chunk or not).  A border record that is not yet beaten
// is a peak iff no border record of the rows dm-1 .. dm+1 beats it (its other neighbours were all seen on the device).
// Beaten records still beat others, so flags are only added while the list is scanned, and dropped at the end.
uint64_t settle_borders(aa_plan *p, aa_candidate *out, uint64_t n)
{
    // first record of every trial
    uint64_t i = 0;
    for (uint32_t d = 0; d <= p->ndms_total; ++d) {
        while (i < n && (out[i].dm_index & kPeakDmMask) < d) ++i;
        p->dm_dst[d] = i;
    }
    auto beats = [](const aa_candidate &x, const aa_candidate &c) {
        if (x.snr != c.snr) return x.snr > c.snr;
        const uint32_t dx = x.dm_index & kPeakDmMask, dc = c.dm_index & kPeakDmMask;
        if (dx != dc) return dx < dc;
        return x.t_start < c.t_start;
    };
    for (uint64_t k = 0; k < n; ++k) {
        aa_candidate &c = out[k];
        if (!(c.dm_index & kPeakBorder) || (c.dm_index & kPeakBeaten)) continue;
        const uint32_t dm = c.dm_index & kPeakDmMask;
        const uint64_t t = c.t_start, te = t + c.width, t_lo = t > p->wmax_raw ? t - p->wmax_raw : 0;
        bool beaten = false;
        for (int dd = -1; dd <= 1 && !beaten; ++dd) {
            const int64_t row = (int64_t)dm + dd;
            if (row < 0 || row >= (int64_t)p->ndms_total) continue;
            const aa_candidate *b = out + p->dm_dst[row], *e = out + p->dm_dst[row + 1];
            const aa_candidate *q = std::lower_bound(b, e, t_lo, [](const aa_candidate &x, uint64_t v) { return x.t_start < v; });
            for (; q < e && (uint64_t)q->t_start <= te; ++q) {
                if (q == &c || !(q->dm_index & kPeakBorder) || t > (uint64_t)q->t_start + q->width) continue;
                if (beats(*q, c)) { beaten = true; break; }
            }
        }
        if (beaten) c.dm_index |= kPeakBeaten;
    }
    uint64_t m = 0;
    for (uint64_t k = 0; k < n; ++k)
        if (!(out[k].dm_index & kPeakBeaten)) {
            out[m] = out[k];
            out[m].dm_index &= kPeakDmMask;
            ++m;
        }
    return m;
}

int run_impl(aa_plan *p, const uint8_t *input, Input mode, aa_candidate *out, uint64_t max_cands,
             uint64_t *n_cands, uint32_t *tap_out)
{
    const bool resident = mode == Input::resident;
    if (!p || !input || !n_cands || (!out && max_cands)) return AA_ERR_INVALID;
    if (tap_out && p->taps_in.empty()) return AA_ERR_INVALID;
    g_last_cuda_error = 0;
    NvtxRange nvtx_run(resident ? "aa_run_resident" : mode == Input::staged ? "aa_run_staged" : "aa_run");
    cudaPointerAttributes at{};
    cudaError_t pe = cudaPointerGetAttributes(&at, input);
    if (pe != cudaSuccess) { cudaGetLastError(); at.type = cudaMemoryTypeUnregistered; }
    if (resident) {
        if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) return AA_ERR_INVALID;
    } else if (mode == Input::staged) {
        if (!p->desc.stage_input || at.type == cudaMemoryTypeDevice) return AA_ERR_INVALID;
    } else if (at.type != cudaMemoryTypeHost) {
        return AA_ERR_NOT_PINNED;                   // never staged through pageable memory silently
    }

    const auto t0 = std::chrono::steady_clock::now();
    for (uint64_t j = 0; j < p->n_sub; ++j) { p->loaded[j].store(0); p->done[j].store(0); p->dedisp_issued[j].store(0); }
    for (int j = 0; j < p->n_streams; ++j) p->copied[j].store(0);
    p->error.store(0); p->out_pos.store(0); p->total.store(0); p->total_raw.store(0); p->overflow.store(0);
    for (auto &S : p->streams) {
        S.h2d_ms = S.d2h_ms = S.prep_ms = S.dedisp_ms = S.sps_ms = S.h2h_ms = 0;
        S.h2d_bytes = S.d2h_bytes = S.dedisp_launches = S.sps_launches = S.prep_launches = S.h2h_bytes = 0;
    }
    if (cudaEventRecord(p->ev_start, p->streams[0].st) != cudaSuccess) { g_last_cuda_error = (int)cudaGetLastError(); return AA_ERR_CUDA; }
    // wake the plan's worker threads (one per stream, created at plan creation) and wait for them
    p->job.input = input; p->job.mode = (int)mode; p->job.out = out; p->job.max_cands = max_cands; p->job.tap_out = tap_out;
    for (uint64_t j = 0; j < p->n_sub; ++j) p->runs[j] = aa_plan::Run{};
    command(p, aa_plan::Cmd::run);
    if (p->error.load()) {
        for (auto &S : p->streams) cudaStreamSynchronize(S.st);
        g_last_cuda_error = p->error.load();
        return AA_ERR_CUDA;
    }

    const uint64_t total = p->total.load();
    const uint64_t stored = std::min<uint64_t>(p->out_pos.load(), max_cands);
    const auto t1 = std::chrono::steady_clock::now();
    // Every sub-chunk's run is already sorted, and the runs of one trial follow each other in time, so the final
    // order is: for every trial, its piece of run 0, of run 1, ...  Two parallel passes through the scratch buffer.
    if (stored > 1) {
        if (stored <= p->scratch_cap) {
            const uint64_t W = (uint64_t)p->ndms_total + 1;
            uint64_t acc = 0;
            for (uint32_t d = 0; d < p->ndms_total; ++d) {
                p->dm_dst[d] = acc;
                for (uint64_t j = 0; j < p->n_sub; ++j) acc += p->run_cnt[j * W + d + 1] - p->run_cnt[j * W + d];
            }
            p->dm_dst[p->ndms_total] = acc;
            p->job.stored = stored;
            command(p, aa_plan::Cmd::scatter);
            command(p, aa_plan::Cmd::copyback);
        } else {
            std::sort(out, out + stored, cand_less);
        }
    }
    uint64_t n_peaks = 0;
    if (p->peaks) {
        n_peaks = settle_borders(p, out, stored);
    }
    const auto t2 = std::chrono::steady_clock::now();
    *n_cands = p->peaks ? n_peaks : total;

    aa_stats &st = p->stats;
    st = aa_stats{};
    st.wall_ms = std::chrono::duration<double, std::milli>(t2 - t0).count();
    st.sort_ms = std::chrono::duration<double, std::milli>(t2 - t1).count();
    for (auto &S : p->streams) {
        st.h2d_bytes += S.h2d_bytes; st.d2h_bytes += S.d2h_bytes;
        st.h2d_ms += S.h2d_ms; st.d2h_ms += S.d2h_ms; st.prep_ms += S.prep_ms;
        st.dedisp_ms += S.dedisp_ms; st.sps_ms += S.sps_ms;
        st.dedisp_launches += S.dedisp_launches; st.sps_launches += S.sps_launches;
        st.prep_launches += S.prep_launches;
        st.h2h_bytes += S.h2h_bytes; st.h2h_ms += S.h2h_ms;
    }
    st.n_candidates = p->total_raw.load();
    st.n_stored = p->peaks ? n_peaks : stored;
    st.n_peaks = n_peaks;
    st.overflow = (p->overflow.load() || total > max_cands) ? 1 : 0;
    st.n_streams = p->n_streams;
    return st.overflow ? AA_ERR_OVERFLOW : AA_OK;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
extern "C" {

uint64_t aa_plan_arena_bytes(const aa_plan_desc *d)
{
    aa_plan tmp;
    if (build_geometry(tmp, d) != AA_OK) return 0;
    return tmp.arena_bytes;
}

int aa_plan_create(aa_plan **out, const aa_plan_desc *d)
{
    if (!out) return AA_ERR_INVALID;
    *out = nullptr;
    g_last_cuda_error = 0;
    aa_plan *p = new (std::nothrow) aa_plan;
    if (!p) return AA_ERR_OOM;
    int rc = build_geometry(*p, d);
    if (rc != AA_OK) { delete p; return rc; }

    auto fail = [&](int code, cudaError_t e) { g_last_cuda_error = (int)e; destroy_plan(p); return code; };
    cudaError_t e;
    if ((e = dedisp_configure()) != cudaSuccess) return fail(AA_ERR_CUDA, e);
    if ((e = dedisp_sp_configure()) != cudaSuccess) return fail(AA_ERR_CUDA, e);
    if ((e = dedisp_ws_configure()) != cudaSuccess) return fail(AA_ERR_CUDA, e);
    if ((e = sps_configure()) != cudaSuccess) return fail(AA_ERR_CUDA, e);

    if (d->device_arena) {
        if (d->device_arena_bytes < p->arena_bytes || ((uintptr_t)d->device_arena & 255)) return fail(AA_ERR_INVALID, cudaSuccess);
        p->arena = d->device_arena;
    } else {
        if ((e = cudaMalloc(&p->arena, p->arena_bytes)) != cudaSuccess) { cudaGetLastError(); return fail(AA_ERR_OOM, e); }
        p->own_arena = true;
    }
    p->streams.resize(p->n_streams);
    for (int s = 0; s < p->n_streams; ++s) {
        Stream &S = p->streams[s];
        if (d->streams) S.st = static_cast<cudaStream_t>(d->streams[s]);
        else {
            if ((e = cudaStreamCreateWithFlags(&S.st, cudaStreamNonBlocking)) != cudaSuccess) return fail(AA_ERR_CUDA, e);
            S.own = true;
        }
        S.ev.assign(kEvFixed + 3 * p->ranges.size(), nullptr);
        for (auto &ev : S.ev) if ((e = cudaEventCreate(&ev)) != cudaSuccess) return fail(AA_ERR_CUDA, e);
        if ((e = cudaHostAlloc((void **)&S.h_count, 256, cudaHostAllocDefault)) != cudaSuccess) { cudaGetLastError(); return fail(AA_ERR_OOM, e); }
        if ((e = cudaHostAlloc((void **)&S.h_cands, p->cap * sizeof(aa_candidate), cudaHostAllocDefault)) != cudaSuccess) { cudaGetLastError(); return fail(AA_ERR_OOM, e); }
        if (p->tap_stage_elems)
            if ((e = cudaHostAlloc((void **)&S.h_tap, p->tap_stage_elems * 4, cudaHostAllocDefault)) != cudaSuccess) { cudaGetLastError(); return fail(AA_ERR_OOM, e); }
        if (d->stage_input)
            if ((e = cudaHostAlloc((void **)&S.h_stage, (p->L + p->halo) * p->row_bytes, cudaHostAllocDefault)) != cudaSuccess) { cudaGetLastError(); return fail(AA_ERR_OOM, e); }
    }
    carve(*p);
    {
        const uint64_t ring_pad = round_up((uint64_t)d->nchans, kRingChPad) - (uint64_t)d->nchans;
        const uint64_t pad_rows = round_up((uint64_t)d->nchans, kSpG) - (uint64_t)d->nchans;
        for (int pl = 0; ring_pad && pl < p->planes; ++pl)
            if ((e = cudaMemset(p->d_ring + (uint64_t)pl * p->ring_plane_bytes + (uint64_t)d->nchans * p->ring_pitch, 0,
                                ring_pad * p->ring_pitch)) != cudaSuccess)
                return fail(AA_ERR_CUDA, e);
        for (auto &S : p->streams)
            for (size_t k = 0; pad_rows && k < S.d_binned.size(); ++k) {
                const uint64_t pitch = p->pitch_b[k % p->bins.size()];
                if ((e = cudaMemset(S.d_binned[k] + (uint64_t)d->nchans * pitch, 0, pad_rows * pitch * 2)) != cudaSuccess)
                    return fail(AA_ERR_CUDA, e);
            }
    }
    p->ev_loaded.assign(p->n_sub, nullptr);
    for (auto &ev : p->ev_loaded)
        if ((e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming)) != cudaSuccess) return fail(AA_ERR_CUDA, e);
    if ((e = cudaEventCreate(&p->ev_start)) != cudaSuccess) return fail(AA_ERR_CUDA, e);
    p->timeline.assign(p->n_sub, aa_subchunk_times{});
    p->ev_dedisp.assign(p->n_sub, nullptr);
    for (auto &ev : p->ev_dedisp)
        if ((e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming)) != cudaSuccess) return fail(AA_ERR_CUDA, e);
    p->ev_copied.assign(p->n_streams, nullptr);
    for (auto &ev : p->ev_copied)
        if ((e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming)) != cudaSuccess) return fail(AA_ERR_CUDA, e);
    p->loaded.reset(new std::atomic<int>[p->n_sub]);
    p->done.reset(new std::atomic<int>[p->n_sub]);
    p->dedisp_issued.reset(new std::atomic<int>[p->n_sub]);
    p->copied.reset(new std::atomic<int>[p->n_streams]);
    // host side of the runs to come: threads, helper pool, tap lists, run tables, merge scratch -- all of it now
    if (cudaGetDevice(&p->device) != cudaSuccess) return fail(AA_ERR_CUDA, cudaGetLastError());
    p->ndms_total = 0;
    for (auto &R : p->ranges) p->ndms_total += (uint32_t)R.r.ndms;
    p->nactive = (int)std::min<uint64_t>((uint64_t)p->n_streams, p->n_sub);
    try {
        for (auto &S : p->streams) {
            S.tapcopies.reserve((size_t)std::max(1, d->ntap));
            S.sort_cur.assign((size_t)p->ndms_total + 1, 0u);
        }
        p->runs.assign(p->n_sub, aa_plan::Run{});
        p->run_cnt.assign(p->n_sub * (uint64_t)(p->ndms_total + 1), 0u);
        p->dm_dst.assign((size_t)p->ndms_total + 1, 0);
        p->hq.reserve((size_t)p->nactive * 3);
        p->scratch_cap = std::min<uint64_t>(p->n_sub * p->cap, 1ull << 24);
        p->scratch = static_cast<aa_candidate *>(std::malloc(p->scratch_cap * sizeof(aa_candidate)));   // touched only as far as a run needs
        if (!p->scratch) p->scratch_cap = 0;                   // the final order then comes from one std::sort
        for (int s = 0; s < p->nactive; ++s) p->workers.emplace_back(worker_main, p, s);
        if (p->tap_stage_elems * 4 >= (64ull << 20)) {
            const int hw = (int)std::max(1u, std::thread::hardware_concurrency());
            const int nh = std::max(0, std::min(hw - p->nactive, 3 * p->nactive));
            for (int k = 0; k < nh; ++k) p->helpers.emplace_back(helper_main, p);
        }
    } catch (...) {
        return fail(AA_ERR_OOM, cudaSuccess);
    }
    for (auto &R : p->ranges) {
        if ((e = cudaMemcpy(R.d_delays, R.h_delays.data(), R.h_delays.size() * 4, cudaMemcpyHostToDevice)) != cudaSuccess)
            return fail(AA_ERR_CUDA, e);
        if ((e = cudaMemcpy(R.d_dtiles, R.h_dtiles.data(), R.h_dtiles.size() * 4, cudaMemcpyHostToDevice)) != cudaSuccess)
            return fail(AA_ERR_CUDA, e);
        if (R.sp_tb && (e = cudaMemcpy(R.d_sp, R.sp_table(), R.sp_table_bytes(), cudaMemcpyHostToDevice)) != cudaSuccess)
            return fail(AA_ERR_CUDA, e);
    }
    *out = p;
    return AA_OK;
}

static void fill_info(const aa_plan *p, aa_plan_info *o);

int aa_plan_geometry(const aa_plan_desc *d, aa_plan_info *o)
{
    if (!o) return AA_ERR_INVALID;
    aa_plan tmp;
    const int rc = build_geometry(tmp, d);
    if (rc != AA_OK) return rc;
    fill_info(&tmp, o);
    return AA_OK;
}

int aa_plan_dedisp_model(const aa_plan_desc *d, int32_t range, int32_t group_channels, aa_dedisp_model *out)
{
    if (!out) return AA_ERR_INVALID;
    aa_plan tmp;
    const int rc = build_geometry(tmp, d);
    if (rc != AA_OK) return rc;
    if (range < 0 || range >= (int32_t)tmp.ranges.size()) return AA_ERR_INVALID;
    const Range &R = tmp.ranges[range];
    // only ranges the warp-specialised family can serve: binned input adds four channels in 16-bit lanes, 4 * 255 * bin
    // must stay below 2^16 (coarser bins run on the plain kernel, a model of the ws kernel there would describe nothing)
    if (group_channels != 4 || (R.in16 && 4ull * 255 * R.r.bin > 65535)) return AA_ERR_INVALID;
    const bool wide = R.in16 && 65535 / (255 * R.r.bin * kSpG) < 4;      // the plan's rule for the 32-bit-accumulator variant
    const int tb = R.ws ? R.sp_tb : (wide ? 512 : 1024);
    return dedisp_model(R.h_delays.data(), R.r.ndms, d->nchans, R.in16 ? 2 : 1, group_channels, tb, wide, out);
}

int aa_plan_query(const aa_plan *p, aa_plan_info *o)
{
    if (!p || !o) return AA_ERR_INVALID;
    fill_info(p, o);
    return AA_OK;
}

static void fill_info(const aa_plan *p, aa_plan_info *o)
{
    o->maxshift = p->maxshift; o->t_valid = p->t_valid; o->halo = p->halo; o->subchunk_len = p->L;
    o->n_subchunks = p->n_sub;
    o->ndms_total = 0; o->dm_trial_samples = 0;
    for (auto &R : p->ranges) { o->ndms_total += (uint64_t)R.r.ndms; o->dm_trial_samples += (uint64_t)R.r.ndms * R.nout; }
    o->arena_bytes = p->arena_bytes; o->pinned_bytes = p->pinned_bytes; o->tap_row_len = p->tap_row_len;
}

uint64_t aa_plan_nout(const aa_plan *p, int32_t r)
{
    if (!p || r < 0 || r >= (int32_t)p->ranges.size()) return 0;
    return p->ranges[r].nout;
}

int aa_plan_delays(const aa_plan *p, int32_t r, int32_t *out)
{
    if (!p || !out || r < 0 || r >= (int32_t)p->ranges.size()) return AA_ERR_INVALID;
    const Range &R = p->ranges[r];
    AA_CUDA(cudaMemcpy(out, R.d_delays, R.h_delays.size() * 4, cudaMemcpyDeviceToHost));
    return AA_OK;
}

int aa_plan_dedisp_variant(const aa_plan *p, int32_t r)
{
    if (!p || r < 0 || r >= (int32_t)p->ranges.size()) return AA_ERR_INVALID;
    const Range &R = p->ranges[r];
    if (!R.sp_tb) return 0;
    if (R.ws_wide) return 5;
    return (R.ws ? 3 : 1) + (R.sp_tb == 1024 ? 1 : 0);
}

int aa_run(aa_plan *p, const uint8_t *host_input, aa_candidate *out, uint64_t max_cands, uint64_t *n_cands,
           uint32_t *tap_out)
{
    return run_impl(p, host_input, Input::pinned, out, max_cands, n_cands, tap_out);
}

int aa_run_staged(aa_plan *p, const uint8_t *host_input, aa_candidate *out, uint64_t max_cands, uint64_t *n_cands,
                  uint32_t *tap_out)
{
    return run_impl(p, host_input, Input::staged, out, max_cands, n_cands, tap_out);
}

int aa_run_resident(aa_plan *p, const uint8_t *device_input, aa_candidate *out, uint64_t max_cands,
                    uint64_t *n_cands, uint32_t *tap_out)
{
    return run_impl(p, device_input, Input::resident, out, max_cands, n_cands, tap_out);
}

int aa_get_stats(const aa_plan *p, aa_stats *out)
{
    if (!p || !out) return AA_ERR_INVALID;
    *out = p->stats;
    return AA_OK;
}

int aa_get_timeline(const aa_plan *p, aa_subchunk_times *out, uint64_t max, uint64_t *n)
{
    if (!p || !n || (!out && max)) return AA_ERR_INVALID;
    *n = p->timeline.size();
    const uint64_t m = std::min<uint64_t>(max, p->timeline.size());
    for (uint64_t i = 0; i < m; ++i) out[i] = p->timeline[i];
    return AA_OK;
}

void aa_destroy(aa_plan *p) { destroy_plan(p); }

int aa_host_alloc(void **ptr, uint64_t bytes)
{
    if (!ptr) return AA_ERR_INVALID;
    *ptr = nullptr;
    cudaError_t e = cudaHostAlloc(ptr, bytes, cudaHostAllocDefault);
    if (e != cudaSuccess) { cudaGetLastError(); g_last_cuda_error = (int)e; return AA_ERR_OOM; }
    return AA_OK;
}

void aa_host_free(void *ptr) { if (ptr) cudaFreeHost(ptr); }

const char *aa_strerror(int s)
{
    switch (s) {
        case AA_OK: return "ok";
        case AA_ERR_INVALID: return "invalid argument or inconsistent plan descriptor";
        case AA_ERR_NOT_PINNED: return "input buffer is not pinned host memory";
        case AA_ERR_OOM: return "out of device or pinned memory";
        case AA_ERR_CUDA: return "CUDA call failed (see aa_last_cuda_error)";
        case AA_ERR_OVERFLOW: return "candidate buffer overflow (list truncated)";
        case AA_ERR_LIMIT: return "request exceeds the fixed capacity of the no-allocation entry point (AA_PEAKS_NOALLOC_MAX_*)";
        default: return "unknown status";
    }
}

int aa_last_cuda_error(void) { return g_last_cuda_error; }

}  // extern "C"
