// Internal declarations of libaa (CUDA path).  Not part of the ABI; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/aa.h"
#include "../../include/aa_bench.h"

namespace aa {

// ---- geometry shared by host scheduler and kernels ------------------------------------------
constexpr int kDedispThreads = 256;   // 8 warps
constexpr int kDedispTB = 512;        // output samples per CTA (time tile)
constexpr int kAlign = 16;            // element alignment of every staged row start

struct DedispArgs {
    const void *in;        // [nchans][pitch_in] uint8 (ring) or uint16 (binned work buffer)
    int64_t pitch_in;      // elements
    int64_t col0;          // element column of output sample 0 with zero delay
    const int32_t *delays; // [ndms][nchans] binned samples (device)
    const int32_t *dtiles; // [nblk][nstages][DB][CS] the same delays tiled per (DM block, channel stage)
    int32_t nchans, ndms;
    int32_t ncols;         // output columns to produce
    uint32_t *out;         // [ndms][pitch_out]
    int64_t pitch_out;     // elements (even)
    int32_t row;           // staged row length in elements (multiple of 16)
    int32_t flush_ch;      // channels between 16->32 bit flushes (even, >= 2)
    // shared-pattern kernel (kernels_dedisp_shared.cu) only:
    const void *sp_tab;    // SpRecord [nblk][ngroups] (device)
    int32_t sp_rows;       // shared-memory bytes reserved per staged channel row (multiple of 16)
    int32_t sp_pbytes;     // bytes of one pattern-row buffer (multiple of 16)
    int32_t sp_flush;      // channel groups between 16-bit -> 32-bit flushes
};

// ---- shared-pattern dedispersion: plan-time record per (DM block, channel group) ---------------
// Within a block of kSpDB consecutive trials the rounded delays of kSpG adjacent channels, taken
// relative to the group's first channel, form only a few distinct vectors ("patterns": each delay
// is rounded on its own, so the differences jitter between floor and ceil).  The kernel sums the
// group's channels once per pattern into a 16-bit row and every trial then adds ONE row sample per
// group instead of kSpG channel samples.  Exact: the same integers are added, in another order.
constexpr int kSpG = 4;             // channels per group
constexpr int kSpDB = 64;           // DM trials per CTA
constexpr int kSpMaxPat = 8;        // pattern rows per record
struct SpRecord {
    int32_t rbase[kSpG];            // first staged sample of each channel row relative to col0 + t0 (multiple of 16)
    uint16_t rbytes[kSpG];          // staged bytes of each channel row (multiple of 16)
    uint16_t npat;                  // pattern rows
    uint16_t nchunk;                // 8-sample chunks per pattern row
    uint16_t nbatch;                // warp-sized batches of chunks per pattern row
    uint16_t inv;                   // ceil(65536 / nbatch): item / nbatch == (item * inv) >> 16
    // pattern k, channel i: row sample u is byte u + sh of the staged channel row.  bits 0-15:
    // i * sp_rows + (sh & ~7), the 8-byte-aligned load offset inside the staging buffer; bits 16-21: (sh & 7) * 8
    uint32_t win[kSpMaxPat][kSpG];
    uint32_t poff[kSpDB];           // byte offset, inside the pattern-row buffer, of trial d's word (tau 0, tau 1)
};
static_assert(sizeof(SpRecord) % 16 == 0, "records are fetched with 16-byte bulk copies");

// Builds the records of one range for time tiles of `tb` samples (host, plan time).  Returns false
// if the range does not fit the scheme (too many patterns, delays not monotone); the caller then
// uses the plain kernels.  rows / pbytes: see DedispArgs.
bool sp_build_tables(const int32_t *delays, int32_t ndms, int32_t nchans, int32_t tb, std::vector<SpRecord> &out,
                     int32_t &rows, int32_t &pbytes);
// tb = 1024 (512 threads, one CTA per SM) or 512 (256 threads, two CTAs per SM)
cudaError_t launch_dedisp_sp(const DedispArgs &a, int tb, cudaStream_t st);

// ---- warp-specialised shared-pattern kernel (kernels_dedisp_ws.cu): record per (DM block, channel group) ----
// Pattern k, channel i: row sample u is byte u + m_i + e_{k,i} of the staged channel row, m_i the
// smallest shift of the channel over the block's patterns and 0 <= e_{k,i} <= 3.
struct WsRecord {
    int32_t rbase[kSpG];            // first staged sample of each channel row relative to col0 + t0 (multiple of 16)
    uint16_t rbytes[kSpG];          // staged bytes of each channel row (multiple of 16)
    uint16_t npat;                  // pattern rows (1..kSpMaxPat)
    uint16_t nchunk;                // 8-sample chunks per pattern row
    uint16_t nbatch;                // warp-sized batches of 31 chunks per pattern row
    uint16_t pad;
    // bits 0-15: i * sp_rows + (m_i & ~7), the 8-byte-aligned load offset of chunk 0 inside the staging
    // slot; bits 16-20: 8 * (m_i & 3); bit 21: (m_i & 4) != 0.  16-bit input: bits 0-15: i * sp_rows +
    // 2 * (m_i & ~3) (bytes), bits 16-17: m_i & 3
    uint32_t chdesc[kSpG];
    uint32_t esh[kSpG][2];          // byte k of the pair: 8 * e_{k,i} (16-bit input: e_{k,i} <= 2)
    uint32_t pofs;                  // byte offset of this stage's pattern rows inside the shared-memory ring
    int32_t dep;                    // the rows may be written once the consumers are done with stage dep (-1: at once)
    uint32_t group;                 // channel group this stage sums: channels group * kSpG .. (stages are not in channel order)
    uint32_t pad2;
    uint32_t poff[kSpDB];           // byte offset, inside the ring, of trial d's word (tau 0, tau 1)
};
static_assert(sizeof(WsRecord) % 16 == 0, "records are fetched with 16-byte bulk copies");
constexpr int kWsTeam = 2;          // producer warps that build one stage together
constexpr int kWsSlots = 16;        // stages are ordered through barrier slots s % kWsSlots ...
constexpr int kWsWindow = 8;        // ... so a stage never starts before stage s - kWsWindow has been consumed
// smem_budget: dynamic shared memory the kernel may use; on success rows = bytes per staged channel row and
// ring_bytes = size of the pattern-row ring (DedispArgs::sp_rows / sp_pbytes)
// elem_bytes: 1 (uint8 input) or 2 (time-binned uint16 input)
bool ws_build_tables(const int32_t *delays, int32_t ndms, int32_t nchans, int32_t tb, int32_t elem_bytes,
                     size_t smem_budget, std::vector<WsRecord> &out, int32_t &rows, int32_t &ring_bytes);
// wide: the 32-bit-accumulator variant (512-sample tiles, 16-bit input only)
cudaError_t launch_dedisp_ws(const DedispArgs &a, int tb, bool in16, bool wide, cudaStream_t st);
size_t dedisp_ws_fixed_smem_bytes(int rows);            // everything but the ring
size_t dedisp_ws_smem_bytes(int rows, int ring_bytes);
cudaError_t dedisp_ws_configure();
size_t dedisp_sp_smem_bytes(int rows, int pbytes);
cudaError_t dedisp_sp_configure();

// The channel rows of the device ring are padded with zero rows to a multiple of this many channels (a whole number of
// kSpG groups; 8 since the rejected 8-channel kernel of round 2, kept so that the arena layout does not move).
constexpr int kRingChPad = 8;

// cost_model.cu: shared-memory wavefronts and room of one kernel family over a delay table (no GPU)
int dedisp_model(const int32_t *delays, int32_t ndms, int32_t nchans, int32_t elem_bytes, int family, int tb, bool wide, aa_dedisp_model *o);

struct SpsArgs {
    const uint32_t *D;     // [ndms][pitch] dedispersed sub-chunk
    int64_t pitch;
    int32_t ndms;
    int32_t ncols;         // columns available in D (own span + boxcar tail)
    int32_t nemit;         // taus [0, nemit) may emit candidates
    int64_t nout_left;     // nout_r - tau0: valid samples of the row from this sub-chunk's start
    int32_t block_len;     // norm block in binned samples
    int32_t nwidths;
    int32_t wmax;
    double thr;
    uint32_t dm_base;      // global index of this range's trial 0
    uint32_t tau0;         // absolute binned index of column 0
    uint32_t bin;
    aa_candidate *cands;
    uint32_t *count;
    uint32_t cap;
    int32_t sigma_mode;    // 1: S/N from the statistics of each width's own boxcar series (reading A18; cluster kernel only)
    uint32_t maxval;       // largest value a dedispersed sample can take (maxsample * nchans * bin)
};

// ---- peak finding on the device (kernels_peaks.cu, reading A17) ---------------------------------------------------
struct PeakArgs {
    const aa_candidate *cands;     // the sub-chunk's raw list
    const uint32_t *count;         // records found (may exceed cap)
    uint32_t cap;
    int32_t *head;                 // [nrows][nbk] first record of each bucket, -1 = empty
    uint32_t *next;                // [cap] chain
    int32_t nrows, nbk, shift;     // DM trials of the plan, buckets per row, log2 of the bucket length in raw samples
    uint32_t t0, t1;               // raw samples [t0, t1) in which this sub-chunk's candidates start
    uint32_t wmax_raw;             // longest boxcar in raw samples
    int32_t has_left, has_right;   // a previous / next sub-chunk exists
    aa_candidate *out;             // peaks and border records; dm_index bit 31 = beaten, bit 30 = border
    uint32_t *out_count;
    uint32_t out_cap;
};
cudaError_t launch_peaks(const PeakArgs &a, cudaStream_t st);
constexpr uint32_t kPeakBeaten = 0x80000000u, kPeakBorder = 0x40000000u, kPeakDmMask = 0x3FFFFFFFu;

constexpr int kMaxWidths = 32;
struct WidthTable { int32_t w[kMaxWidths]; int32_t dec[kMaxWidths]; };   // widths and the time grid of each (A20)

// ---- kernel launchers (each returns cudaGetLastError()) -------------------------------------
// nbits 8: uint8 rows; 4: two samples per byte (even channel low), unpacked into the ring; 16: little-endian words,
// low bytes into `ring`, high bytes into `ring_hi`
cudaError_t launch_corner_turn(const uint8_t *src, int64_t nt, int32_t nchans, int32_t nbits, int64_t t_abs0,
                               uint8_t *ring, uint8_t *ring_hi, int64_t ring_pitch, int64_t ring_len, int64_t mirror,
                               cudaStream_t st);
// 16-bit input: D += Dhi << 8 over [ndms][ncols]
cudaError_t launch_combine_planes(uint32_t *D, const uint32_t *Dhi, int64_t pitch, int32_t ndms, int32_t ncols, cudaStream_t st);
cudaError_t launch_bin(const uint8_t *ring, int64_t ring_pitch, int64_t col0, int32_t nchans,
                       int32_t bin, int64_t nbinned, uint16_t *out, int64_t out_pitch, cudaStream_t st);
// every power-of-two bin 2, 4, .., 32 the plan uses, in one pass (level l = bin 2^(l+1); out[l] == nullptr: not wanted)
struct BinMultiArgs {
    const uint8_t *ring;
    int64_t ring_pitch, col0;   // col0 and every out pitch: multiples of 16 elements
    int64_t ngroups;            // groups of 32 input samples to read (the last one may be partial)
    uint16_t *out[5];
    int64_t pitch[5];           // elements
    int64_t nbinned[5];         // valid outputs per row
};
cudaError_t launch_bin_multi(const BinMultiArgs &a, int32_t nchans, cudaStream_t st);
// dpw = DMs per warp (4, 2 or 1); in16 = input is uint16
cudaError_t launch_dedisp(const DedispArgs &a, bool in16, int dpw, cudaStream_t st);
size_t dedisp_smem_bytes(bool in16, int dpw, int row);
int dedisp_stage_channels(bool in16);
cudaError_t dedisp_configure();   // opt in to large dynamic shared memory (once per process)
// wide: boxcar sums need 64 bits (maxsample nchans bin wmax >= 2^32); small31: they stay below 2^31;
// big: a block's sum of squares may pass 2^63 (16-bit input on many channels): 128-bit sums in the generic kernel
// force_v1: keep sps_cluster_kernel where sps_cluster2_kernel would serve (A/B timing and tests)
cudaError_t launch_sps(const SpsArgs &a, const WidthTable &wt, bool wide, bool small31, bool big, bool force_v1, cudaStream_t st);
cudaError_t sps_configure();

}  // namespace aa
