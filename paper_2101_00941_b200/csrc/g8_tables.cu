// Plan-time tables of the 8-channel shared-pattern dedispersion kernel (kernels_dedisp_g8.cu).  Host code.
//
// Same exact identity as ws_tables.cu, with wider groups and shorter trial blocks.  For a block of kG8Half
// consecutive DM trials d (one half of a CTA's 64 trials) and a group of 8 adjacent channels c0..c0+7 write
//     delta(c0+i, d) = ref(d) + rel_i(d),   ref(d) = delta(c0, d),   off(d) = ref(d) - ref(d_first).
// Every delay is rounded on its own, so rel(d) takes a handful of distinct vectors ("patterns").  For pattern k
//     P_k[u] = sum_{i<8} y[c0+i][t0 + ref(d_first) + u + rel_i^k]
// and   sum_i y[c0+i][t0 + tau + delta(c0+i, d)] = P_{k(d)}[tau + off(d)]   exactly (the same integers are added).
// A pattern is a pair (A, B): A = (rel_1, rel_2, rel_3), B = (rel_4 .. rel_7).  The kernel sums channels 0-3 once per
// distinct A and channels 4-7 once per distinct B, and forms every pair that occurs with four packed additions, so
// the cost of a row grows with nA + nB + npat rather than with 8 * npat.
#include <algorithm>
#include <array>
#include <map>

#include "aa_internal.h"

namespace aa {

bool g8_build_tables(const int32_t *delays, int32_t ndms, int32_t nchans, size_t smem_budget, G8Tables &T)
{
    constexpr int G = kG8, DB = kSpDB, H = kG8Half, TB = kG8TB;
    const int nblk = (ndms + DB - 1) / DB, ngrp = (nchans + G - 1) / G, nst = 2 * ngrp;
    T.nblk = nblk;
    T.nstages = nst;
    T.recs.assign((size_t)nblk * nst, G8Record{});
    T.wins.assign((size_t)nblk * ngrp, G8Window{});
    int64_t max_rows = 16, max_stage = 16;
    // m[h][i]: smallest shift of channel i inside its staged window, per stage (filled in once `rows` is known)
    std::vector<std::array<int, G>> mins((size_t)nblk * nst);

    for (int b = 0; b < nblk; ++b) {
        for (int g = 0; g < ngrp; ++g) {
            const int c0 = g * G;
            // trials past ndms repeat the last trial; channels past nchans repeat the last channel's delay and read
            // the zero rows that pad the input to a multiple of 8 channels
            auto dly = [&](int d, int i) {
                return delays[(size_t)std::min(d, ndms - 1) * nchans + std::min(c0 + i, nchans - 1)];
            };
            // absolute shifts S = ref + rel of every (half, trial, channel); the window of channel i starts at the
            // 16-aligned sample at or below the smallest one
            int smin[G], nchunk[2], ref0[2], mn[2][G];
            for (int i = 0; i < G; ++i) smin[i] = INT32_MAX;
            for (int h = 0; h < 2; ++h) {
                const int dfirst = b * DB + h * H;
                ref0[h] = dly(dfirst, 0);
                for (int i = 0; i < G; ++i) mn[h][i] = INT32_MAX;
                int prev = -1;
                for (int dl = 0; dl < H; ++dl) {
                    const int ref = dly(dfirst + dl, 0);
                    if (ref < ref0[h] || ref < prev) return false;           // delays must not decrease with the trial index
                    prev = ref;
                    for (int i = 0; i < G; ++i) {
                        const int rel = dly(dfirst + dl, i) - ref;
                        if (rel < 0) return false;                           // nor with the channel index
                        mn[h][i] = std::min(mn[h][i], rel);
                    }
                }
                const int offmax = prev - ref0[h];
                // trial d reads row words [off>>1, off>>1 + TB/2) of the (off&1) copy: samples 0 .. TB + offmax
                nchunk[h] = (TB + offmax + 1 + 7) / 8;
                if (nchunk[h] > 4000) return false;
                for (int i = 0; i < G; ++i) smin[i] = std::min(smin[i], ref0[h] + mn[h][i]);
            }
            G8Window &W = T.wins[(size_t)b * ngrp + g];
            int maxrb = 0;
            for (int i = 0; i < G; ++i) {
                W.rbase[i] = smin[i] & ~(kAlign - 1);
                int need = 0;
                for (int h = 0; h < 2; ++h) {
                    const int m = ref0[h] + mn[h][i] - W.rbase[i];          // smallest shift of the half inside the window
                    mins[((size_t)b * ngrp + g) * 2 + h][i] = m;
                    // a producer lane reads 20 bytes from the 8-byte boundary at or below 8*chunk + m, chunk <= nchunk
                    need = std::max(need, 8 * nchunk[h] + (m & ~7) + 20);
                }
                const int rb = (need + 15) / 16 * 16;
                if (rb > 16368) return false;
                W.rbytes[i] = (uint16_t)rb;
                maxrb = std::max(maxrb, rb);
            }
            max_rows = std::max<int64_t>(max_rows, maxrb);

            for (int h = 0; h < 2; ++h) {
                G8Record &R = T.recs[((size_t)b * ngrp + g) * 2 + h];
                const int dfirst = b * DB + h * H;
                std::vector<std::array<int, 3>> pa;        // distinct A = (rel_1, rel_2, rel_3)
                std::vector<std::array<int, 4>> pb;        // distinct B = (rel_4 .. rel_7)
                int ka[H], kb[H], off[H];
                for (int dl = 0; dl < H; ++dl) {
                    const int ref = dly(dfirst + dl, 0);
                    off[dl] = ref - ref0[h];
                    std::array<int, 3> a{};
                    std::array<int, 4> bb{};
                    for (int i = 1; i < 4; ++i) a[i - 1] = dly(dfirst + dl, i) - ref;
                    for (int i = 4; i < 8; ++i) bb[i - 4] = dly(dfirst + dl, i) - ref;
                    size_t x = std::find(pa.begin(), pa.end(), a) - pa.begin();
                    if (x == pa.size()) pa.push_back(a);
                    size_t y = std::find(pb.begin(), pb.end(), bb) - pb.begin();
                    if (y == pb.size()) pb.push_back(bb);
                    ka[dl] = (int)x;
                    kb[dl] = (int)y;
                }
                if ((int)pa.size() > kG8MaxA || (int)pb.size() > kG8MaxB) return false;
                // extra shifts over the smallest one: at most 3 bytes (one funnel shift inside a word pair)
                for (size_t k = 0; k < pa.size(); ++k)
                    for (int i = 1; i < 4; ++i) {
                        const int e = pa[k][i - 1] - mn[h][i];
                        if (e > 3) return false;
                        R.eA[i - 1][k] = (uint8_t)(8 * e);
                    }
                for (size_t k = 0; k < pb.size(); ++k)
                    for (int i = 4; i < 8; ++i) {
                        const int e = pb[k][i - 4] - mn[h][i];
                        if (e > 3) return false;
                        R.eB[i - 4][k] = (uint8_t)(8 * e);
                    }
                // the pairs that occur; rows are numbered in the order the kernel emits them: A patterns in passes of
                // four, inside a pass B patterns in order, inside a B pattern the A patterns of the pass in order
                for (int dl = 0; dl < H; ++dl) R.comb[kb[dl]] |= (uint8_t)(1u << ka[dl]);
                std::map<std::pair<int, int>, int> rowid;
                int nrow = 0;
                for (int p0 = 0; p0 < (int)pa.size(); p0 += 4) {
                    if (p0 == 4) R.rows0 = (uint8_t)nrow;
                    for (int y = 0; y < (int)pb.size(); ++y)
                        for (int x = p0; x < std::min(p0 + 4, (int)pa.size()); ++x)
                            if (R.comb[y] >> x & 1) rowid[{x, y}] = nrow++;
                }
                if ((int)pa.size() <= 4) R.rows0 = (uint8_t)nrow;
                R.nA = (uint8_t)pa.size();
                R.nB = (uint8_t)pb.size();
                R.npat = (uint8_t)nrow;
                R.nchunk = (uint16_t)nchunk[h];
                R.nbatch = (uint16_t)((nchunk[h] + 30) / 31);
                const int rowwords = nchunk[h] * 4;
                for (int dl = 0; dl < H; ++dl)       // relative to the stage's rows; the ring offset is added below
                    R.poff[dl] = (uint32_t)(((rowid[{ka[dl], kb[dl]}] * 2 + (off[dl] & 1)) * rowwords + (off[dl] >> 1)) * 4);
                max_stage = std::max<int64_t>(max_stage, (int64_t)nrow * 2 * rowwords * 4);
            }
        }
    }
    T.rows = (int32_t)max_rows;
    if ((int64_t)G * T.rows > 65535) return false;
    for (size_t r = 0; r < T.recs.size(); ++r)
        for (int i = 0; i < G; ++i) {
            const uint32_t m = (uint32_t)mins[r][i];
            // bits 0-15: byte offset of the lane-0 load inside the window slot; 16-20: 8 * (m & 3); 21: (m & 4) != 0
            T.recs[r].chdesc[i] = ((uint32_t)i * (uint32_t)T.rows + (m & ~7u)) | (8u * (m & 3u)) << 16 | ((m >> 2) & 1u) << 21;
        }

    // The pattern rows of successive stages go round a ring in shared memory whose offsets are fixed here, per DM
    // block.  The two halves consume their stages independently (each in order), so a stage may be written once the
    // latest overlapping earlier stage of EACH half has been consumed: dep[0] is that stage of the same half (never
    // older than s - kG8Window, because barrier slots are reused modulo kG8Slots), dep[1] the one of the other half.
    const size_t fixed = dedisp_g8_fixed_smem_bytes(T.rows);
    if (smem_budget < fixed + (size_t)max_stage + 128) return false;
    const int64_t C = (int64_t)((smem_budget - fixed) / 128 * 128);
    if (C > 0x7FFFFFFF) return false;
    for (int b = 0; b < nblk; ++b) {
        struct Live { int s; int64_t lo, hi; };
        std::vector<Live> live[2];
        int dep_run[2] = {-1, -1};        // a stage's wait also covers what earlier stages waited for only if it never decreases
        int64_t head = 0;
        uint32_t cum = 0;                 // batches before this stage (they are dealt round the producer warps)
        for (int s = 0; s < nst; ++s) {
            G8Record &R = T.recs[(size_t)b * nst + s];
            const int64_t size = ((int64_t)R.npat * 2 * R.nchunk * 16 + 127) / 128 * 128;
            if (head + size > C) head = 0;
            const int64_t lo = head, hi = head + size;
            head = hi;
            for (int q = 0; q < 2; ++q) {                 // q = 0: same half as s, 1: the other half
                const int hh = (s & 1) ^ q;
                int dep = -1;
                for (auto &L : live[hh])
                    if (L.lo < hi && lo < L.hi) dep = std::max(dep, L.s);
                dep = std::max(dep, dep_run[hh]);
                const int floor_s = q == 0 ? s - kG8Window : s - kG8Window - 1;
                if (floor_s >= 0) dep = std::max(dep, floor_s);
                dep_run[hh] = dep;
                auto &v = live[hh];
                v.erase(std::remove_if(v.begin(), v.end(), [&](const Live &L) { return L.s <= dep; }), v.end());
                R.dep[q] = dep;
            }
            live[s & 1].push_back({s, lo, hi});
            R.pofs = (uint32_t)lo;
            R.bstart = (uint16_t)(cum % kG8Producers);
            cum += R.nbatch;
            for (int dl = 0; dl < H; ++dl) R.poff[dl] += (uint32_t)lo;
        }
    }
    T.ring_bytes = (int32_t)C;
    // Window descriptors travel with the stage records: the record of stage 2g (first half of group g) holds group g's
    // own windows (the prologue requests groups 0 and 1 from them), the record of stage 2g+1 those of group
    // g + kG8Ahead, which the producers request while they build stage 2g+1.
    for (int b = 0; b < nblk; ++b)
        for (int g = 0; g < ngrp; ++g) {
            const G8Window &W = T.wins[(size_t)b * ngrp + g];
            G8Record &R0 = T.recs[((size_t)b * ngrp + g) * 2];
            for (int i = 0; i < G; ++i) { R0.nrbase[i] = W.rbase[i]; R0.nrbytes[i] = W.rbytes[i]; }
            if (g + kG8Ahead < ngrp) {
                const G8Window &N = T.wins[(size_t)b * ngrp + g + kG8Ahead];
                G8Record &R1 = T.recs[((size_t)b * ngrp + g) * 2 + 1];
                for (int i = 0; i < G; ++i) { R1.nrbase[i] = N.rbase[i]; R1.nrbytes[i] = N.rbytes[i]; }
            }
        }
    return true;
}

}  // namespace aa
