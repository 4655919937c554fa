"""Host logic of the timeline report (no GPU): interval unions and the copy/compute overlap figure."""
import pytest

from paper_2101_00941_b200 import timeline as T


def _entry(j, h0, h1, p1, c0, c1):
    return {"index": j, "stream": j % 2, "h2d_begin": h0, "h2d_end": h1, "prep_end": p1, "compute_begin": c0,
            "compute_end": c1, "d2h_end": c1, "dedisp_ms": c1 - c0, "sps_ms": 0.0}


def test_union_and_intersection():
    u = T._union([(0, 2), (1, 3), (5, 6), (6, 6)])
    assert u == [[0, 3], [5, 6]] and T._length(u) == 4
    assert T._intersect(u, T._union([(2, 5.5)])) == pytest.approx(1.5)
    assert T._intersect(u, []) == 0.0


def test_overlap_figures_of_a_hand_made_timeline():
    # copy 0 alone on the link (nothing to hide behind), copy 1 fully under sub-chunk 0's kernels
    tl = [_entry(0, 0.0, 10.0, 11.0, 11.0, 41.0), _entry(1, 12.0, 22.0, 23.0, 41.0, 71.0)]
    s = T.summarise(tl, wall_ms=72.0)
    assert s["link_busy_ms"] == pytest.approx(20.0)
    # kernels in flight: [10,11] + [11,41] + [22,23] + [41,71] -> [10,71]
    assert s["kernels_in_flight_ms"] == pytest.approx(61.0)
    assert s["overlap_pct"] == pytest.approx(50.0)
    assert s["kernel_idle_ms"] == pytest.approx(11.0)


def test_report_modules_refuse_to_run_without_cuda():
    import torch
    from paper_2101_00941_b200 import sweep
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(SystemExit):
        sweep.main(["--workload", "1", "--streams", "1"])
    with pytest.raises(SystemExit):
        T.main(["--workload", "1"])


def test_dedispersion_cost_model_on_the_headline_workload():
    """aa_plan_dedisp_model (aa_bench.h; no GPU): the consumer term is the definition (one 32-bit row word per trial, group
    and sample pair) less the words a trial shares with the previous trial of its warp, which the kernel does not load
    again; the pattern counts are those of the delay table; ranges the kernel family cannot serve are refused."""
    import numpy as np
    import oracle
    from paper_2101_00941_b200 import binding as B, inputs as I
    w = I.workload(3)
    m4 = B.dedisp_model(w, 0, 4)
    assert m4["stages_per_cta"] == w.nchans // 4
    full = 64 * 1024 * 2 / 128 * (w.nchans // 4)
    f = m4["shared_offset_fraction"]                             # of the 48 non-leading trials of a 64-trial block
    assert m4["wf_consumer"] == pytest.approx(full * (64 - 48 * f) / 64, rel=1e-12) and 0.97 * full < m4["wf_consumer"] < full
    # distinct relative-delay vectors of one (64 trials, 4 channels) block, counted from the oracle's delay table
    dl = oracle.delays(w, 0)
    blk = dl[:64, 2000:2004] - dl[:64, 2000:2001]
    assert 1 <= len(np.unique(blk, axis=0)) <= m4["patterns_max"] <= 8
    assert 4.0 < m4["patterns_mean"] < 5.5
    assert m4["stage_bytes_max"] <= m4["ring_bytes"] and 0.0 <= f < 0.1
    assert B.dedisp_model(w, 0, 8) is None                       # the 8-channel family is gone
    # fine DM steps: many trials share their row words, and the model counts what the kernel then skips
    w4 = I.workload(4)
    m = B.dedisp_model(w4, 1, 4)
    assert m is not None and m["shared_offset_fraction"] > 0.1
    assert m["wf_consumer"] < 0.93 * 64 * m["tile_samples"] * 2 / 128 * m["stages_per_cta"]
    # bin 32 runs the 32-bit-accumulator variant, which loads every word: no reduction there
    m5 = B.dedisp_model(w4, 5, 4)
    assert m5 is not None and m5["tile_samples"] == 512
    assert m5["wf_consumer"] == pytest.approx(64 * 512 * 2 / 128 * m5["stages_per_cta"])
    # binned input beyond 4 * 255 * bin < 2^16 runs on the plain kernel: no model of a kernel that never runs
    import dataclasses
    coarse = I.scaled(w4, ranges=(dataclasses.replace(w4.ranges[5], bin=128),), norm_block=65536, name="bin128")
    assert B.plan_geometry(coarse)["ndms_total"] == w4.ranges[5].ndms and B.dedisp_model(coarse, 0, 4) is None
