// Preparation kernels of a sub-chunk: corner turn of the freshly copied
// time-major rows into the channel-major device ring, and per-range time binning.
// Both are plain HBM-bound data movement (2 B and ~1+2/b B per input sample).
#include <algorithm>

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

// Vector variant (nchans % 4 == 0; every time offset involved is a multiple of 16, see launch).
// CTA tile = 128 times x 128 channels.  Warp w takes times [16w, 16w+16): every lane loads the 4
// channels 4*lane..4*lane+3 of each of them (one 128-byte request per time row), transposes the 16 x 4
// byte block in registers (PRMT) and stores four 16-byte pieces "16 times of one channel" into the
// shared tile T[c][piece], pieces XOR-swizzled so that both the stores and the loads below are
// conflict-free.  Then every thread moves four pieces to the ring with 16-byte stores (8 lanes
// write 128 contiguous bytes of one channel row).
constexpr int kCtT = 128, kCtC = 128;

__device__ __forceinline__ void transpose4x4(uint32_t a, uint32_t b, uint32_t c, uint32_t d, uint32_t &o0,
                                             uint32_t &o1, uint32_t &o2, uint32_t &o3)
{
    const uint32_t ab01 = __byte_perm(a, b, 0x5140), cd01 = __byte_perm(c, d, 0x5140);   // a0 b0 a1 b1
    const uint32_t ab23 = __byte_perm(a, b, 0x7362), cd23 = __byte_perm(c, d, 0x7362);   // a2 b2 a3 b3
    o0 = __byte_perm(ab01, cd01, 0x5410);
    o1 = __byte_perm(ab01, cd01, 0x7632);
    o2 = __byte_perm(ab23, cd23, 0x5410);
    o3 = __byte_perm(ab23, cd23, 0x7632);
}

__global__ void __launch_bounds__(256) corner_turn_vec_kernel(const uint8_t *__restrict__ src, int64_t nt,
                                                              int32_t nchans, int64_t t_abs0,
                                                              uint8_t *__restrict__ ring, int64_t ring_pitch,
                                                              int64_t ring_len, int64_t mirror)
{
    __shared__ uint4 T[kCtC][kCtT / 16];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t tb = (int64_t)blockIdx.x * kCtT;
    const int32_t cb = blockIdx.y * kCtC;

    {
        const int32_t c = cb + 4 * lane;
        const int64_t t = tb + 16 * warp;
        uint32_t x[16];
#pragma unroll
        for (int i = 0; i < 16; ++i)
            x[i] = (c < nchans && t + i < nt) ? __ldcs(reinterpret_cast<const uint32_t *>(src + (t + i) * nchans + c)) : 0u;
        uint32_t o[4][4];            // [quarter of the 16 times][channel]
#pragma unroll
        for (int q = 0; q < 4; ++q)
            transpose4x4(x[4 * q], x[4 * q + 1], x[4 * q + 2], x[4 * q + 3], o[q][0], o[q][1], o[q][2], o[q][3]);
#pragma unroll
        for (int j = 0; j < 4; ++j)
            T[4 * lane + j][warp ^ (lane & 7)] = make_uint4(o[0][j], o[1][j], o[2][j], o[3][j]);
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const int item = threadIdx.x + 256 * k;          // 128 channels x 8 pieces
        const int cl = item >> 3, piece = item & 7;
        const int32_t c = cb + cl;
        const int64_t t = tb + 16 * piece;
        if (c < nchans && t < nt) {                      // nt is a multiple of 16
            const uint4 v = T[cl][piece ^ ((cl >> 2) & 7)];
            const int64_t col = (t_abs0 + t) % ring_len;
            uint8_t *dst = ring + c * ring_pitch + col;
            *reinterpret_cast<uint4 *>(dst) = v;
            if (col < mirror) *reinterpret_cast<uint4 *>(dst + ring_len) = v;
        }
    }
}

// Other input bit depths (reading A19), same tiling as corner_turn_kernel:
//   NBITS 4 : a row holds nchans / 2 bytes, even channel in the low nibble; the ring receives the nibbles as bytes;
//   NBITS 16: a row holds nchans little-endian words; the low bytes go to `ring`, the high bytes to `ring_hi` (two
//             8-bit planes: dedispersion is linear, D = D(low) + 256 D(high), so the 8-bit kernels serve both).
template <int NBITS>
__global__ void __launch_bounds__(256) corner_turn_packed_kernel(const uint8_t *__restrict__ src, int64_t nt, int32_t nchans,
                                                                 int64_t t_abs0, uint8_t *__restrict__ ring,
                                                                 uint8_t *__restrict__ ring_hi, int64_t ring_pitch,
                                                                 int64_t ring_len, int64_t mirror)
{
    __shared__ uint8_t tile[2][64][64 + 4];
    const int tx = threadIdx.x & 63, ty = threadIdx.x >> 6;   // 64 x 4
    const int64_t tb = (int64_t)blockIdx.x * 64;
    const int32_t cb = blockIdx.y * 64;
    const int64_t row_bytes = NBITS == 4 ? nchans / 2 : 2 * (int64_t)nchans;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const int64_t t = tb + ty + 4 * k;
        const int32_t c = cb + tx;
        uint8_t lo = 0, hi = 0;
        if (t < nt && c < nchans) {
            if (NBITS == 4) {
                const uint8_t b = src[t * row_bytes + (c >> 1)];
                lo = (c & 1) ? (uint8_t)(b >> 4) : (uint8_t)(b & 15);
            } else {
                const uint16_t v = *reinterpret_cast<const uint16_t *>(src + t * row_bytes + 2 * (int64_t)c);
                lo = (uint8_t)(v & 0xFF);
                hi = (uint8_t)(v >> 8);
            }
        }
        tile[0][ty + 4 * k][tx] = lo;
        if (NBITS == 16) tile[1][ty + 4 * k][tx] = hi;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const int32_t c = cb + ty + 4 * k;
        const int64_t t = tb + tx;
        if (t < nt && c < nchans) {
            const int64_t col = (t_abs0 + t) % ring_len;
            const uint8_t v = tile[0][tx][ty + 4 * k];
            ring[c * ring_pitch + col] = v;
            if (col < mirror) ring[c * ring_pitch + ring_len + col] = v;
            if (NBITS == 16) {
                const uint8_t h = tile[1][tx][ty + 4 * k];
                ring_hi[c * ring_pitch + col] = h;
                if (col < mirror) ring_hi[c * ring_pitch + ring_len + col] = h;
            }
        }
    }
}

// 16-bit input: D <- D(low bytes) + 256 * D(high bytes), element by element over the sub-chunk's output tile
__global__ void __launch_bounds__(256) combine_planes_kernel(uint32_t *__restrict__ D, const uint32_t *__restrict__ Dhi,
                                                             int64_t pitch, int32_t ncols)
{
    const int64_t row = (int64_t)blockIdx.y * pitch;
    for (int32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < ncols; i += gridDim.x * blockDim.x)
        D[row + i] += Dhi[row + i] << 8;
}

cudaError_t launch_combine_planes(uint32_t *D, const uint32_t *Dhi, int64_t pitch, int32_t ndms, int32_t ncols, cudaStream_t st)
{
    if (ndms <= 0 || ncols <= 0) return cudaSuccess;
    dim3 grid((unsigned)std::min<int64_t>((ncols + 255) / 256, 64), (unsigned)ndms);
    combine_planes_kernel<<<grid, 256, 0, st>>>(D, Dhi, pitch, ncols);
    return cudaGetLastError();
}

cudaError_t launch_corner_turn(const uint8_t *src, int64_t nt, int32_t nchans, int32_t nbits, int64_t t_abs0,
                               uint8_t *ring, uint8_t *ring_hi, int64_t ring_pitch, int64_t ring_len, int64_t mirror,
                               cudaStream_t st)
{
    if (nt <= 0) return cudaSuccess;
    if (nbits != 8) {
        dim3 grid((unsigned)((nt + 63) / 64), (unsigned)((nchans + 63) / 64));
        if (nbits == 4)
            corner_turn_packed_kernel<4><<<grid, 256, 0, st>>>(src, nt, nchans, t_abs0, ring, ring_hi, ring_pitch, ring_len, mirror);
        else
            corner_turn_packed_kernel<16><<<grid, 256, 0, st>>>(src, nt, nchans, t_abs0, ring, ring_hi, ring_pitch, ring_len, mirror);
        return cudaGetLastError();
    }
    // 16-sample pieces must not straddle the end of the ring, the mirror boundary or the end of the data
    const bool vec = nchans % 4 == 0 && nt % 16 == 0 && t_abs0 % 16 == 0 && ring_len % 16 == 0 && mirror % 16 == 0 &&
                     ring_pitch % 16 == 0 && (reinterpret_cast<uintptr_t>(src) & 3) == 0 &&
                     (reinterpret_cast<uintptr_t>(ring) & 15) == 0;
    if (vec) {
        dim3 grid((unsigned)((nt + kCtT - 1) / kCtT), (unsigned)((nchans + kCtC - 1) / kCtC));
        corner_turn_vec_kernel<<<grid, 256, 0, st>>>(src, nt, nchans, t_abs0, ring, ring_pitch, ring_len, mirror);
    } else {
        dim3 grid((unsigned)((nt + 63) / 64), (unsigned)((nchans + 63) / 64));
        corner_turn_kernel<<<grid, 256, 0, st>>>(src, nt, nchans, t_abs0, ring, ring_pitch, ring_len, mirror);
    }
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

// All power-of-two bins 2..32 of a sub-chunk in one pass over the ring: a thread takes 32 consecutive samples
// of one channel (two 16-byte loads) and forms the sums of 2, 4, 8, 16 and 32 by successive pairwise addition
// (16-bit lanes, SWAR), storing the levels the plan asks for.  The ring is read once instead of once per bin.
__global__ void __launch_bounds__(256) bin_multi_kernel(const BinMultiArgs a)
{
    const int32_t c = blockIdx.y;
    const uint8_t *row = a.ring + c * a.ring_pitch + a.col0;
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < a.ngroups; g += (int64_t)gridDim.x * blockDim.x) {
        const uint4 x0 = __ldg(reinterpret_cast<const uint4 *>(row + 32 * g));
        const uint4 x1 = __ldg(reinterpret_cast<const uint4 *>(row + 32 * g + 16));
        const uint32_t w[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
        uint32_t s2[8], s4[4], s8[2], s16, s32;
#pragma unroll
        for (int i = 0; i < 8; ++i) s2[i] = (w[i] & 0x00FF00FFu) + ((w[i] >> 8) & 0x00FF00FFu);     // two sums of 2
#pragma unroll
        for (int i = 0; i < 4; ++i) {                                                               // two sums of 4
            const uint32_t lo = (s2[2 * i] & 0xFFFFu) + (s2[2 * i] >> 16), hi = (s2[2 * i + 1] & 0xFFFFu) + (s2[2 * i + 1] >> 16);
            s4[i] = lo | hi << 16;
        }
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const uint32_t lo = (s4[2 * i] & 0xFFFFu) + (s4[2 * i] >> 16), hi = (s4[2 * i + 1] & 0xFFFFu) + (s4[2 * i + 1] >> 16);
            s8[i] = lo | hi << 16;
        }
        {
            const uint32_t lo = (s8[0] & 0xFFFFu) + (s8[0] >> 16), hi = (s8[1] & 0xFFFFu) + (s8[1] >> 16);
            s16 = lo | hi << 16;
            s32 = lo + hi;
        }
        // level l holds 32 >> (l + 1) sums of this group, packed two per word
        auto put = [&](int l, const uint32_t *v, int n) {
            uint16_t *o = a.out[l];
            if (!o) return;
            o += c * a.pitch[l];
            const int64_t first = g * n;
            if (first + n <= a.nbinned[l]) {
                if (n >= 8) {
#pragma unroll
                    for (int i = 0; i < n / 8; ++i)
                        reinterpret_cast<uint4 *>(o + first)[i] = make_uint4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
                } else if (n == 4) {
                    *reinterpret_cast<uint2 *>(o + first) = make_uint2(v[0], v[1]);
                } else if (n == 2) {
                    *reinterpret_cast<uint32_t *>(o + first) = v[0];
                } else {
                    o[first] = (uint16_t)v[0];
                }
            } else {
                for (int i = 0; i < n; ++i)
                    if (first + i < a.nbinned[l]) o[first + i] = (uint16_t)(v[i >> 1] >> (16 * (i & 1)));
            }
        };
        put(0, s2, 16);
        put(1, s4, 8);
        put(2, s8, 4);
        put(3, &s16, 2);
        put(4, &s32, 1);
    }
}

cudaError_t launch_bin_multi(const BinMultiArgs &a, int32_t nchans, cudaStream_t st)
{
    if (a.ngroups <= 0) return cudaSuccess;
    unsigned gx = (unsigned)((a.ngroups + 255) / 256);
    if (gx > 16) gx = 16;
    dim3 grid(gx, (unsigned)nchans);
    bin_multi_kernel<<<grid, 256, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace aa
