// Peak finding on the sorted candidate list (host code; reading A17).
//
// Part of the host output stage: the list aa_run returns is small (only candidates cross the link), so the
// step runs on the host cores, rows of DM trials spread over threads like the per-stream copy threads of
// PAPER.md:63.  Neighbours: DM indices differ by at most 1 and the boxcars overlap or touch in raw samples
// (t' <= t + w and t <= t' + w').  A candidate is a peak iff no neighbour has a larger stored S/N, ties going to
// the smaller (dm_index, t_start).  Shares nothing with oracle/ (which checks all pairs).
#include <algorithm>
#include <atomic>
#include <thread>
#include <vector>

#include "aa_internal.h"

namespace {

struct Row { uint32_t dm; uint64_t lo, hi; };

inline bool beats(const aa_candidate &a, const aa_candidate &b)   // a beats b
{
    if (a.snr != b.snr) return a.snr > b.snr;
    if (a.dm_index != b.dm_index) return a.dm_index < b.dm_index;
    return a.t_start < b.t_start;
}

}  // namespace

extern "C" int aa_find_peaks(const aa_candidate *c, uint64_t n, aa_candidate *out, uint64_t max_out, uint64_t *n_out,
                             int32_t nthreads)
{
    if (!n_out || (!c && n) || (!out && max_out)) return AA_ERR_INVALID;
    *n_out = 0;
    if (n == 0) return AA_OK;
    std::vector<Row> rows;
    uint64_t wmax = 0;
    for (uint64_t i = 0; i < n; ++i) {
        if (i && (c[i].dm_index < c[i - 1].dm_index || (c[i].dm_index == c[i - 1].dm_index && c[i].t_start < c[i - 1].t_start)))
            return AA_ERR_INVALID;                           // not sorted by (dm_index, t_start)
        if (rows.empty() || rows.back().dm != c[i].dm_index) {
            if (!rows.empty()) rows.back().hi = i;
            rows.push_back({c[i].dm_index, i, n});
        }
        wmax = std::max<uint64_t>(wmax, c[i].width);
    }
    std::vector<uint8_t> keep(n, 1);
    if (nthreads < 1) nthreads = (int32_t)std::max(1u, std::thread::hardware_concurrency());
    nthreads = (int32_t)std::min<uint64_t>((uint64_t)nthreads, rows.size());
    std::atomic<size_t> next{0};

    auto work = [&]() {
        for (;;) {
            const size_t r = next.fetch_add(1);
            if (r >= rows.size()) return;
            for (uint64_t i = rows[r].lo; i < rows[r].hi; ++i) {
                const aa_candidate &ci = c[i];
                const uint64_t t_hi = (uint64_t)ci.t_start + ci.width;                     // neighbours start at or before this
                const uint64_t t_lo = ci.t_start > wmax ? (uint64_t)ci.t_start - wmax : 0;   // ... and not before this
                bool peak = true;
                for (int dd = -1; dd <= 1 && peak; ++dd) {
                    const size_t q = r + (size_t)dd;                                       // rows are sorted by dm
                    if ((dd < 0 && r == 0) || q >= rows.size()) continue;
                    if ((int64_t)rows[q].dm != (int64_t)ci.dm_index + dd) continue;
                    const aa_candidate *b = c + rows[q].lo, *e = c + rows[q].hi;
                    const aa_candidate *j = std::lower_bound(b, e, t_lo, [](const aa_candidate &x, uint64_t t) { return x.t_start < t; });
                    for (; j < e && (uint64_t)j->t_start <= t_hi; ++j) {
                        if (j == &ci || (uint64_t)ci.t_start > (uint64_t)j->t_start + j->width) continue;
                        if (beats(*j, ci)) { peak = false; break; }
                    }
                }
                keep[i] = peak ? 1 : 0;
            }
        }
    };
    std::vector<std::thread> th;
    for (int k = 1; k < nthreads; ++k) th.emplace_back(work);
    work();
    for (auto &t : th) t.join();

    uint64_t m = 0;
    for (uint64_t i = 0; i < n; ++i)
        if (keep[i]) {
            if (m < max_out) out[m] = c[i];
            ++m;
        }
    *n_out = m;
    return m > max_out ? AA_ERR_OVERFLOW : AA_OK;
}
