// Internal declarations of libaa (CUDA path).  Not part of the ABI; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/aa.h"

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
};

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
};

constexpr int kMaxWidths = 32;
struct WidthTable { int32_t w[kMaxWidths]; };

// ---- kernel launchers (each returns cudaGetLastError()) -------------------------------------
cudaError_t launch_corner_turn(const uint8_t *src, int64_t nt, int32_t nchans, int64_t t_abs0,
                               uint8_t *ring, int64_t ring_pitch, int64_t ring_len, int64_t mirror,
                               cudaStream_t st);
cudaError_t launch_bin(const uint8_t *ring, int64_t ring_pitch, int64_t col0, int32_t nchans,
                       int32_t bin, int64_t nbinned, uint16_t *out, int64_t out_pitch, cudaStream_t st);
// dpw = DMs per warp (4, 2 or 1); in16 = input is uint16
cudaError_t launch_dedisp(const DedispArgs &a, bool in16, int dpw, cudaStream_t st);
size_t dedisp_smem_bytes(bool in16, int dpw, int row);
int dedisp_stage_channels(bool in16);
cudaError_t dedisp_configure();   // opt in to large dynamic shared memory (once per process)
cudaError_t launch_sps(const SpsArgs &a, const WidthTable &wt, bool wide, cudaStream_t st);
cudaError_t sps_configure();

}  // namespace aa
