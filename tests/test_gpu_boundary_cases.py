"""Configurations of the C ABI that no other test runs ("parity tests" 1-4):
the library-owned arena and streams a plain C caller gets ("0/NULL -> library allocates with cudaMalloc /
non-blocking streams"; PAPER.md:41 step 1, "create CUDA streams"), and an output buffer smaller than the list in both
output modes.  Everything is compared with the oracle."""
import numpy as np
import pytest

import oracle
from paper_2101_00941_b200 import inputs as I
from _compare import compare_candidates, key
from test_gpu_parity import _pinned_fill, _tiny

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2101_00941_b200 import binding
    binding.load_library()
    return binding


def _against_oracle(B, w, **plan_kw):
    buf, x = _pinned_fill(B, w)
    with B.Plan(w, taps=list(range(w.ndms_total)), **plan_kw) as plan:
        cands, tap = plan.run(buf)
        assert not plan.overflow
    ref, dense, geo = oracle.run(x, w, keep_dense=True)
    base = 0
    for r, rg in enumerate(w.ranges):
        assert np.array_equal(tap[base:base + rg.ndms, :geo["nout"][r]], dense[r]), f"dedispersed series differ in range {r}"
        base += rg.ndms
    res = compare_candidates(cands, ref, w.snr_threshold)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0 and res["common"] > 0
    return cands


def test_library_owned_arena_and_streams_match_the_oracle(B):
    """device_arena = NULL, streams = NULL: aa_plan_create cudaMallocs the arena and creates its own non-blocking
    streams.  cfg1 (one stream) and a three-stream case with several chunks, against the oracle; the results equal the
    caller-owned (torch) resources' bit for bit."""
    w1 = I.workload(1)
    own = _against_oracle(B, w1, torch_resources=False)
    assert own.tobytes() == _against_oracle(B, w1).tobytes()
    top = own[np.argmax(own["snr"])]
    assert (top["dm_index"], top["t_start"], top["width"]) == (50, 40000, 8)
    w3 = _tiny(n_streams=3, chunk_len=3 * 2048, nsamp=30000, thr=4.0)
    own = _against_oracle(B, w3, torch_resources=False)
    assert own.tobytes() == _against_oracle(B, w3).tobytes()


def test_library_owned_resources_are_released(B):
    """Ten create / run / destroy rounds with library-owned resources leave the device's free memory where it was
    (cudaMemGetInfo): aa_destroy frees the arena, streams, events and pinned staging it made."""
    import torch
    w = _tiny(n_streams=3, chunk_len=3 * 2048, nsamp=30000, thr=4.0)
    buf, _ = _pinned_fill(B, w)
    with B.Plan(w, torch_resources=False) as plan:        # first round outside the measurement: lazy module loading
        first, _ = plan.run(buf, want_taps=False)
        arena = plan.info["arena_bytes"]
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(10):
        with B.Plan(w, torch_resources=False) as plan:
            got, _ = plan.run(buf, want_taps=False)
            assert got.tobytes() == first.tobytes()
            inside, _ = torch.cuda.mem_get_info()
            assert free0 - inside >= arena                # the arena really is the library's own cudaMalloc
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert abs(free0 - free1) <= (2 << 20), (free0, free1)  # the driver hands memory out in 2 MiB pages


@pytest.mark.parametrize("n_streams,chunk_len", [(1, 4096), (3, 3 * 2048)])
def test_output_buffer_smaller_than_the_candidate_list(B, n_streams, chunk_len):
    """output_mode 0 with max_cands below the total: AA_ERR_OVERFLOW (not fatal), *n_cands is the true total, `out`
    holds n_stored <= max_cands records, sorted by (dm_index, t_start), every one of them a record of the oracle's
    list.  With one stream the stored records are whole sub-chunks in time order."""
    w = _tiny(n_streams=n_streams, chunk_len=chunk_len, nsamp=30000, thr=3.5)
    buf, x = _pinned_fill(B, w)
    ref, _ = oracle.run(x, w)
    kr = key(ref)
    for max_cands in (len(ref) // 3, 1, len(ref) - 1):
        with B.Plan(w) as plan:
            got, _ = plan.run(buf, max_cands=max_cands, want_taps=False)
            st = plan.stats()
            assert plan.overflow and st["overflow"] == 1
            assert plan.n_found == len(ref) == st["n_candidates"]           # the true total
            assert len(got) == st["n_stored"] <= max_cands and len(got) > 0
        kg = key(got)
        assert np.all(np.diff(kg.astype(np.int64)) > 0)
        assert np.all(got["dm_index"] < w.ndms_total)                       # no flag bits
        idx = np.searchsorted(kr, kg)
        assert np.all(idx < len(ref)) and np.array_equal(kr[idx], kg), "stored records that the oracle does not have"
        compare_candidates(got, ref[idx], w.snr_threshold)
    # room for exactly the list: no overflow
    with B.Plan(w) as plan:
        got, _ = plan.run(buf, max_cands=len(ref), want_taps=False)
        assert not plan.overflow and len(got) == len(ref)


@pytest.mark.parametrize("n_streams,chunk_len", [(1, 4096), (3, 3 * 2048)])
def test_output_buffer_smaller_than_the_peak_list(B, n_streams, chunk_len):
    """output_mode 1 with max_cands below what the sub-chunks send (peaks + border records): AA_ERR_OVERFLOW, the
    records returned are sorted, carry no peak flag in dm_index (bits 30 and 31 are internal), and each is a candidate
    of the oracle's full list; n_found and n_stored agree with what `out` holds.  With room for everything the
    result is the peak rule on the oracle's list (checked elsewhere; repeated here as the control)."""
    w = _tiny(n_streams=n_streams, chunk_len=chunk_len, nsamp=30000, thr=3.2)
    buf, x = _pinned_fill(B, w)
    ref, _ = oracle.run(x, w)
    want = oracle.find_peaks_fast(ref)
    kr = key(ref)
    with B.Plan(w, peaks=True) as plan:
        got, _ = plan.run(buf, want_taps=False)
        assert not plan.overflow and got.tobytes() == want.tobytes()
        crossed = (plan.stats()["d2h_bytes"] - 8 * plan.info["n_subchunks"]) // 16   # records the sub-chunks sent
    assert crossed >= len(want)
    for max_cands in (crossed // 2, 7, crossed - 1):
        with B.Plan(w, peaks=True) as plan:
            got, _ = plan.run(buf, max_cands=max_cands, want_taps=False)
            st = plan.stats()
            assert plan.overflow and st["overflow"] == 1
            assert st["n_candidates"] == len(ref)
            assert len(got) == st["n_stored"] == st["n_peaks"] == plan.n_found <= max_cands
        assert np.all(got["dm_index"] < w.ndms_total), "peak flags left in dm_index"
        kg = key(got)
        assert np.all(np.diff(kg.astype(np.int64)) > 0)
        idx = np.searchsorted(kr, kg)
        assert np.all(idx < len(ref)) and np.array_equal(kr[idx], kg)
        compare_candidates(got, ref[idx], w.snr_threshold)
