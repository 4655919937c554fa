// Plan-time tables of the warp-specialised shared-pattern dedispersion kernel
// (kernels_dedisp_ws.cu).  Host code.
//
// For a block of kSpDB consecutive DM trials d and a group of kSpG adjacent channels c0..c0+G-1
// write   delta(c0+i, d) = ref(d) + rel_i(d),   ref(d) = delta(c0, d).
// rel(d) is a vector of small integers; because every delay is rounded on its own it jitters
// between floor and ceil of the exact difference, so a block sees a handful of distinct vectors
// ("patterns": 4.7 per 64 trials on the 4096-channel workloads).  For pattern k
//     P_k[u] = sum_i y[c0+i][t0 + ref(d_first) + u + rel_i^k]
// and then  sum_i y[c0+i][t0 + tau + delta(c0+i,d)] = P_{k(d)}[tau + ref(d) - ref(d_first)]  exactly.
// The record lists, per (block, group): where each channel row's staged window starts and how long
// it is, the smallest shift m_i of each channel and every pattern's extra shift e_{k,i} = shift - m_i,
// and for every trial the position of its first word inside the pattern rows.
#include <algorithm>
#include <array>

#include "aa_internal.h"

namespace aa {

bool ws_build_tables(const int32_t *delays, int32_t ndms, int32_t nchans, int32_t tb, int32_t elem_bytes,
                     size_t smem_budget, std::vector<WsRecord> &out, int32_t &rows, int32_t &ring_bytes)
{
    // 8-bit input: extra shifts e <= 3 (bytes inside a word); 16-bit input: e <= 2 (one PRMT over a word pair)
    const int max_extra = elem_bytes == 1 ? 3 : 2;
    constexpr int G = kSpG, DB = kSpDB;
    const int nblk = (ndms + DB - 1) / DB, ngrp = (nchans + G - 1) / G;
    out.assign((size_t)nblk * ngrp, WsRecord{});
    int64_t max_rows = 16, max_pbytes = 16;      // largest staged channel row / largest stage of pattern rows
    std::vector<std::array<int, G>> mins((size_t)nblk * ngrp);

    for (int b = 0; b < nblk; ++b) {
        const int dfirst = b * DB;
        for (int g = 0; g < ngrp; ++g) {
            WsRecord &R = out[(size_t)b * ngrp + g];
            const int c0 = g * G;
            // trials past ndms repeat the last trial; channels past nchans repeat the last channel's delay
            // and read the zero rows that pad the input to a multiple of kSpG channels
            auto dly = [&](int d, int i) {
                return delays[(size_t)std::min(d, ndms - 1) * nchans + std::min(c0 + i, nchans - 1)];
            };
            const int ref0 = dly(dfirst, 0);

            // distinct patterns of the block
            std::array<int, G> pats[kSpMaxPat];
            int npat = 0, kd[DB], off[DB];
            for (int dl = 0; dl < DB; ++dl) {
                const int d = dfirst + dl, ref = dly(d, 0);
                std::array<int, G> rel{};
                for (int i = 0; i < G; ++i) {
                    rel[i] = dly(d, i) - ref;
                    if (rel[i] < 0) return false;        // delays must not decrease with channel index
                }
                off[dl] = ref - ref0;
                if (off[dl] < 0 || (dl && off[dl] < off[dl - 1])) return false;   // nor with the trial index
                int k = 0;
                while (k < npat && pats[k] != rel) ++k;
                if (k == npat) {
                    if (npat == kSpMaxPat) return false;
                    pats[npat++] = rel;
                }
                kd[dl] = k;
            }

            const int offmax = off[DB - 1];
            // trial d reads row words [off>>1, off>>1 + tb/2) of the (off&1) copy: samples 0 .. tb + offmax
            const int nchunk = (tb + offmax + 1 + 7) / 8;
            if (nchunk > 8000) return false;
            int maxrb = 0;
            for (int i = 0; i < G; ++i) {
                int mn = pats[0][i], mx = pats[0][i];
                for (int k = 1; k < npat; ++k) {
                    mn = std::min(mn, pats[k][i]);
                    mx = std::max(mx, pats[k][i]);
                }
                if (mx - mn > max_extra) return false;
                R.rbase[i] = (ref0 + mn) & ~(kAlign - 1);
                const int m = ref0 + mn - R.rbase[i];    // smallest shift inside the staged row, 0..15
                mins[(size_t)b * ngrp + g][i] = m;
                for (int k = 0; k < npat; ++k) {
                    // 8-bit input: funnel-shift bits; 16-bit input: the shift itself
                    const uint32_t e8 = (elem_bytes == 1 ? 8u : 1u) * (uint32_t)(pats[k][i] - mn);
                    R.esh[i][k >> 2] |= e8 << (8 * (k & 3));
                }
                // a producer lane reads 20 bytes from the 8-byte boundary at or below 8*chunk + m, chunk <= nchunk
                // (16-bit input: 14 samples from the 4-sample boundary at or below it)
                const int need = elem_bytes == 1 ? 8 * nchunk + (m & ~7) + 20 : 2 * (8 * nchunk + (m & ~3) + 14);
                const int rb = (need + 15) / 16 * 16;
                if (rb > 16368) return false;
                R.rbytes[i] = (uint16_t)rb;
                maxrb = std::max(maxrb, rb);
            }
            R.npat = (uint16_t)npat;
            R.nchunk = (uint16_t)nchunk;
            R.nbatch = (uint16_t)((nchunk + 30) / 31);
            const int rowwords = nchunk * 4;
            for (int dl = 0; dl < DB; ++dl)       // relative to the stage's rows; the ring offset is added below
                R.poff[dl] = (uint32_t)(((kd[dl] * 2 + (off[dl] & 1)) * rowwords + (off[dl] >> 1)) * 4);

            max_rows = std::max<int64_t>(max_rows, maxrb);
            max_pbytes = std::max<int64_t>(max_pbytes, (int64_t)npat * 2 * rowwords * 4);
        }
    }
    rows = (int32_t)max_rows;
    if ((int64_t)G * rows > 65535) return false;
    for (size_t r = 0; r < out.size(); ++r)
        for (int i = 0; i < G; ++i) {
            const uint32_t m = (uint32_t)mins[r][i];
            out[r].chdesc[i] = elem_bytes == 1
                                   ? ((uint32_t)i * (uint32_t)rows + (m & ~7u)) | (8u * (m & 3u)) << 16 | ((m >> 2) & 1u) << 21
                                   : ((uint32_t)i * (uint32_t)rows + 2u * (m & ~3u)) | (m & 3u) << 16;
        }
    // Stage order.  The producers' work per stage grows with the pattern count and the row length (3 patterns x 1100
    // samples at the top of a 300 MHz band, 7 x 1950 at the bottom) while the consumers' work is the same for every
    // stage, so in channel order the producers idle through the first half of a CTA and the consumers wait for them
    // through the second half.  The sum over channel groups may be taken in any order (exact integers): stages
    // alternate between the cheapest and the dearest groups left, and the ring of pattern rows evens out the pairs.
    // The kernel's producer teams take every fourth stage (8 producer warps in teams of kWsTeam = 2), so the alternation runs
    // cheap-dear-cheap-dear / dear-cheap-dear-cheap: every team gets both kinds.
    // One order for all DM blocks, so that the CTAs of a time tile still walk the channels together (L2).
    std::vector<double> cost((size_t)ngrp, 0.0);
    for (int b = 0; b < nblk; ++b)
        for (int g = 0; g < ngrp; ++g) {
            const WsRecord &R = out[(size_t)b * ngrp + g];
            cost[(size_t)g] += (double)R.nchunk * (40.0 + 34.0 * R.npat);
        }
    std::vector<int> rank((size_t)ngrp), order((size_t)ngrp);
    for (int g = 0; g < ngrp; ++g) rank[(size_t)g] = g;
    std::stable_sort(rank.begin(), rank.end(), [&](int x, int y) { return cost[(size_t)x] < cost[(size_t)y]; });
    for (int s = 0, lo = 0, hi = ngrp - 1; s < ngrp; ++s)
        order[(size_t)s] = ((s & 1) ^ ((s >> 2) & 1)) ? rank[(size_t)hi--] : rank[(size_t)lo++];
    {
        std::vector<WsRecord> staged(out.size());
        for (int b = 0; b < nblk; ++b)
            for (int s = 0; s < ngrp; ++s) {
                WsRecord &R = staged[(size_t)b * ngrp + s];
                R = out[(size_t)b * ngrp + order[(size_t)s]];
                R.group = (uint32_t)order[(size_t)s];
            }
        out.swap(staged);
    }
    // The pattern rows of successive stages go round a ring in shared memory.  Offsets are fixed here, per DM
    // block; dep = the latest earlier stage whose rows overlap the new ones (the producers wait until the
    // consumers are done with it), never older than s - kWsWindow (barrier slots are reused modulo kWsSlots).
    const size_t fixed = dedisp_ws_fixed_smem_bytes(rows);
    if (smem_budget < fixed + (size_t)max_pbytes + 128) return false;
    const int64_t C = (int64_t)((smem_budget - fixed) / 128 * 128);
    if (C > 0x7FFFFFFF) return false;
    for (int b = 0; b < nblk; ++b) {
        struct Live { int s; int64_t lo, hi; };
        std::vector<Live> live;
        size_t oldest = 0;
        int64_t head = 0;
        int dep_run = -1;     // stages dropped from `live` are covered by an earlier wait only if dep never decreases
        for (int s = 0; s < ngrp; ++s) {
            WsRecord &R = out[(size_t)b * ngrp + s];
            const int64_t size = ((int64_t)R.npat * 2 * R.nchunk * 16 + 127) / 128 * 128;
            if (head + size > C) head = 0;
            const int64_t lo = head, hi = head + size;
            head = hi;
            int dep = -1;
            // stages are consumed in order: everything up to the newest overlapping one must be gone
            for (size_t j = oldest; j < live.size(); ++j)
                if (live[j].lo < hi && lo < live[j].hi) dep = live[j].s;
            dep = std::max(dep, std::max(dep_run, s - kWsWindow));
            dep_run = dep;
            while (oldest < live.size() && live[oldest].s <= dep) ++oldest;
            live.push_back({s, lo, hi});
            R.pofs = (uint32_t)lo;
            R.dep = dep;
            for (int dl = 0; dl < DB; ++dl) R.poff[dl] += (uint32_t)lo;
        }
    }
    ring_bytes = (int32_t)C;
    return true;
}

}  // namespace aa
