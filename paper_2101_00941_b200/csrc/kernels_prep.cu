// Preparation kernels of a sub-chunk: corner turn of the freshly copied
// time-major rows into the channel-major device ring, and per-range time binning.
// Both are plain HBM-bound data movement (2 B and ~1+2/b B per input sample).
#include "aa_internal.h"

namespace aa {

// x[t][c] (nt rows of nchans bytes, absolute time of row 0 = t_abs0) -> ring[c][t mod ring_len];
// columns < mirror are also written at ring_len + col so that a window starting in the last
// slot of the ring is contiguous.
// Tile: 64 times x 64 channels through shared memory; global reads are coalesced along c,
// global writes along t.
__global__ void __launch_bounds__(256) corner_turn_kernel(const uint8_t *__restrict__ src, int64_t nt,
                                                          int32_t nchans, int64_t t_abs0,
                                                          uint8_t *__restrict__ ring, int64_t ring_pitch,
                                                          int64_t ring_len, int64_t mirror)
{
    __shared__ uint8_t tile[64][64 + 4];
    const int tx = threadIdx.x & 63, ty = threadIdx.x >> 6;   // 64 x 4
    const int64_t tb = (int64_t)blockIdx.x * 64;
    const int32_t cb = blockIdx.y * 64;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        int64_t t = tb + ty + 4 * k;
        int32_t c = cb + tx;
        tile[ty + 4 * k][tx] = (t < nt && c < nchans) ? src[t * nchans + c] : (uint8_t)0;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        int32_t c = cb + ty + 4 * k;
        int64_t t = tb + tx;
        if (t < nt && c < nchans) {
            uint8_t v = tile[tx][ty + 4 * k];
            int64_t col = (t_abs0 + t) % ring_len;
            ring[c * ring_pitch + col] = v;
            if (col < mirror) ring[c * ring_pitch + ring_len + col] = v;
        }
    }
}

cudaError_t launch_corner_turn(const uint8_t *src, int64_t nt, int32_t nchans, int64_t t_abs0,
                               uint8_t *ring, int64_t ring_pitch, int64_t ring_len, int64_t mirror,
                               cudaStream_t st)
{
    if (nt <= 0) return cudaSuccess;
    dim3 grid((unsigned)((nt + 63) / 64), (unsigned)((nchans + 63) / 64));
    corner_turn_kernel<<<grid, 256, 0, st>>>(src, nt, nchans, t_abs0, ring, ring_pitch, ring_len, mirror);
    return cudaGetLastError();
}

// y[c][k] = sum_{i<bin} ring[c][col0 + bin*k + i], k < nbinned  (integer sum before delaying, A6)
__global__ void __launch_bounds__(256) bin_kernel(const uint8_t *__restrict__ ring, int64_t ring_pitch,
                                                  int64_t col0, int32_t bin, int64_t nbinned,
                                                  uint16_t *__restrict__ out, int64_t out_pitch)
{
    const int32_t c = blockIdx.y;
    const uint8_t *row = ring + c * ring_pitch + col0;
    uint16_t *o = out + c * out_pitch;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < nbinned;
         k += (int64_t)gridDim.x * blockDim.x) {
        const uint8_t *p = row + k * bin;
        uint32_t s = 0;
        if ((bin & 3) == 0) {
            for (int i = 0; i < bin; i += 4) {
                uint32_t w = *reinterpret_cast<const uint32_t *>(p + i);   // col0, bin*k multiples of 4
                s += __dp4a(w, 0x01010101u, 0u);
            }
        } else {
            for (int i = 0; i < bin; ++i) s += p[i];
        }
        o[k] = (uint16_t)s;
    }
}

cudaError_t launch_bin(const uint8_t *ring, int64_t ring_pitch, int64_t col0, int32_t nchans,
                       int32_t bin, int64_t nbinned, uint16_t *out, int64_t out_pitch, cudaStream_t st)
{
    if (nbinned <= 0) return cudaSuccess;
    unsigned gx = (unsigned)((nbinned + 255) / 256);
    if (gx > 64) gx = 64;
    dim3 grid(gx, (unsigned)nchans);
    bin_kernel<<<grid, 256, 0, st>>>(ring, ring_pitch, col0, bin, nbinned, out, out_pitch);
    return cudaGetLastError();
}

}  // namespace aa
