"""Cost model report of the shared-pattern dedispersion kernels (aa_plan_dedisp_model; no GPU needed).

    python -m paper_2101_00941_b200.costmodel > profiles/r2_cost_model.md

For every range of the 4096-channel workloads: shared-memory wavefronts per (64 trials x 1024 samples) output tile
and 4 channels, by source, for the 4-channel x 64-trial stage of dedisp_ws_kernel, plus the readings that were not
built or were built and rejected (the 8-channel kernel of round 2 is no longer in the tree, its rows
in profiles/r2_cost_model.md are that round's record).
"""
from __future__ import annotations

from . import binding as B
from . import inputs as I


def rows(w, r):
    out = []
    for g in (4,):
        m = B.dedisp_model(w, r, g)
        if m is None:
            continue
        # normalise to one (4 channels x 64 trials x 1024 samples) unit block
        nblocks = (w.nchans / 4.0) * (m["tile_samples"] / 1024.0)
        f = 1.0 / nblocks
        out.append((g, m, {k: m[k] * f for k in ("wf_consumer", "wf_producer_load", "wf_producer_store", "wf_bulk")}))
    return out


def main():
    print("# Round 2: shared-memory cost model of the dedispersion kernels over the real delay tables\n")
    print("Command (no GPU): `python -m paper_2101_00941_b200.costmodel` (calls `aa_plan_dedisp_model` of `libaa.so`,")
    print("`csrc/cost_model.cu`, which builds the kernels' own plan-time tables and counts what they make the kernel do).")
    print("Unit: 128-byte shared-memory wavefronts per (4 channels x 64 trials x 1024 samples) block of work; the pipe")
    print("delivers one per clock per SM (`profiles/r2_microbench.md`).\n")
    print("| workload / range | stage | patterns mean (max) | consumer loads | producer loads | producer stores | bulk landings | total | "
          "stage KB mean (max) | ring KB | same row words as the previous trial |")
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    for k in (3, 4):
        w = I.workload(k)
        for r, rg in enumerate(w.ranges):
            for g, m, n in rows(w, r):
                tot = sum(n.values())
                print(f"| cfg{k} r{r} (step {rg.dm_step}, bin {rg.bin}) | {g} ch x {m['block_trials']} trials x {m['tile_samples']} | "
                      f"{m['patterns_mean']:.1f} ({m['patterns_max']}) | {n['wf_consumer']:.0f} | {n['wf_producer_load']:.0f} | "
                      f"{n['wf_producer_store']:.0f} | {n['wf_bulk']:.0f} | **{tot:.0f}** | {m['stage_bytes_mean'] / 1024:.0f} "
                      f"({m['stage_bytes_max'] / 1024:.0f}) | {m['ring_bytes'] / 1024:.0f} | {100 * m['shared_offset_fraction']:.1f} % |")
    print("""
Readings (VERDICT r1 item 4, (i)-(iv)):

* (i) the 4-channel x 64-trial stage that runs: 1024 consumer + about 440 producer wavefronts per block on cfg3; ncu measured 1577
  (the difference is plan-record and trial-offset reads and bank conflicts), 86 % of the pipe at 26.6 ms per launch.
* (iii) 8 channels x 32 trials, pattern rows built from (channels 0-3, channels 4-7) pairs: -17 % wavefronts on cfg3 by this model.
  Built (`kernels_dedisp_g8.cu`), bit-exact, and measured at 58.7 ms per launch: the model counts bytes, but the producers then need
  4666 instructions per stage and eight latency-bound warps deliver 1.2 per clock (`profiles/r2_dedisp_g8_ncu.txt`).  8 channels x
  64 trials would need 5 % fewer wavefronts still, but its stages (81 KB on average, 181 KB at the bottom of the band) do not fit
  the ring.
* (ii) skipping the load when a consumer warp's next trial reads the very same row words (same pattern, same offset): last column.
  2 % of the loads on cfg3 (the delay of most channels moves by more than a sample per trial), 13-36 % on cfg4's fine-step ranges.
* (iv) three 10-bit samples per row word (4-channel sums <= 1020): 2/3 of the consumer bytes (-23 % of the total on cfg3), but a
  16-bit accumulator lane holds only one 10-bit field without carry, so each word must be split before it is added: 5 issue slots per
  three samples instead of 2 per two, and rows need three alignments instead of two (+50 % producer stores).  With issue slots at
  68 % and the producers already the critical path, not built.
""")


if __name__ == "__main__":
    main()
