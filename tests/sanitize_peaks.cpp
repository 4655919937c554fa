// Test infrastructure (not product code): drives aa_find_peaks (csrc/peaks.cu, the library's host thread pool for the
// peak rule) from a plain executable so that it can run under ThreadSanitizer, which a Python process cannot host.
// Built and run by tests/test_host_sanitizers.py.  Prints the number of peaks of each list; exit code 0 = ran through.
#include <algorithm>
#include <cstdint>
#include <cstdio>
#include <random>
#include <vector>

#include "../include/aa.h"

int main()
{
    std::mt19937_64 rng(2101);
    for (int round = 0; round < 6; ++round) {
        const uint32_t ndm = round % 2 ? 40 : 3, span = 20000;
        std::vector<aa_candidate> c(30000);
        for (auto &x : c) {
            x.dm_index = (uint32_t)(rng() % ndm);
            x.t_start = (uint32_t)(rng() % span);
            x.width = 1u << (rng() % 7);
            x.snr = 6.0f + (float)(rng() % 60) * 0.1f;           // many exact ties
        }
        std::sort(c.begin(), c.end(), [](const aa_candidate &a, const aa_candidate &b) {
            return a.dm_index != b.dm_index ? a.dm_index < b.dm_index : a.t_start < b.t_start;
        });
        c.erase(std::unique(c.begin(), c.end(), [](const aa_candidate &a, const aa_candidate &b) {
                    return a.dm_index == b.dm_index && a.t_start == b.t_start;
                }), c.end());
        std::vector<aa_candidate> out(c.size());
        uint64_t n1 = 0, n8 = 0;
        if (aa_find_peaks(c.data(), c.size(), out.data(), out.size(), &n1, 1) != AA_OK) return 2;
        std::vector<aa_candidate> out8(c.size());
        if (aa_find_peaks(c.data(), c.size(), out8.data(), out8.size(), &n8, 8) != AA_OK) return 3;
        if (n1 != n8) return 4;
        for (uint64_t i = 0; i < n1; ++i)
            if (out[i].dm_index != out8[i].dm_index || out[i].t_start != out8[i].t_start) return 5;
        std::printf("round %d: %zu candidates, %llu peaks\n", round, c.size(), (unsigned long long)n1);
    }
    return 0;
}
