"""aa_find_peaks_device_noalloc: device peak finding for callers that must not allocate device memory.

Some users of this library cannot call cudaMalloc while they work: a real-time ingest loop in its streamed phase
(cudaMalloc / cudaFree wait for the whole device, so one allocation stalls every other stream's copies and kernels),
or a process whose device memory all belongs to one owner such as a caching pool.  For them the library has one entry
point whose scratch memory (bucket grid + chains of the peak kernels) is a fixed 8 MiB array inside libaa.so instead of
a slice of a plan's arena.  The array is shared by every call and keeps the last call's contents, so the thing to
check is that a call is correct whatever the call before it left behind: each test below makes two (or more) calls in
a row, with different lists and different grid shapes, and compares every result with the library's existing peak
paths -- aa_find_peaks on the host, and aa_run's output_mode 1 on the device -- record for record (the peak rule is
exact: same set of 16-byte records, the tolerance every peak test in this suite uses).

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide other tests) and
passes alone in a fresh process as well as after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

from paper_2101_00941_b200 import inputs as I


@pytest.fixture(scope="module")
def B():
    from paper_2101_00941_b200 import binding, build
    build.build_cuda()
    binding.load_library()
    return binding


def _sorted(a):
    return a[np.lexsort((a["t_start"], a["dm_index"]))]


def _random_list(B, rng, n, ndms, t_end, wmax):
    c = np.zeros(n, dtype=B.CAND_DTYPE)
    c["dm_index"] = rng.integers(0, ndms, n)
    c["t_start"] = rng.integers(0, t_end, n)
    c["width"] = 2 ** rng.integers(0, int(np.log2(wmax)) + 1, n)
    c["snr"] = np.round(rng.uniform(6, 12, n), 1).astype(np.float32)            # many exact ties
    _, first = np.unique(np.stack([c["dm_index"], c["t_start"]]), axis=1, return_index=True)
    return _sorted(c[np.sort(first)])                                            # one record per (dm, t), as aa_run gives


def _device_peaks(B, torch, cands, ndms, t_end, wmax, order_rng=None, out_cap=None):
    """One call of the entry point; every buffer is the caller's (torch tensors made before the call)."""
    src = cands if order_rng is None else cands[order_rng.permutation(len(cands))]     # the call takes any order
    d_in = torch.from_numpy(np.frombuffer(src.tobytes(), dtype=np.uint8).copy()).cuda()
    cap = len(cands) if out_cap is None else out_cap
    d_out = torch.zeros(max(cap, 1) * 16, dtype=torch.uint8, device="cuda")
    d_n = torch.full((1,), 12345, dtype=torch.int32, device="cuda")              # garbage: the call must reset it
    B.find_peaks_device_noalloc(d_in, ndms, t_end, wmax, d_out[: cap * 16], d_n, n=len(cands))
    torch.cuda.synchronize()
    n = int(d_n.item())
    got = np.frombuffer(d_out.cpu().numpy().tobytes(), dtype=B.CAND_DTYPE)[: min(n, cap)]
    return n, _sorted(got)


def test_limits_are_refused_before_any_cuda_call(B):
    """Sizes beyond the fixed array are an error of their own (AA_ERR_LIMIT), never a hidden allocation; needs no GPU."""
    lib = B.load_library()
    dummy = ctypes.c_uint32(0)
    err = ctypes.c_int(7)
    call = lambda n, ndms, t_end: lib.aa_find_peaks_device_noalloc(ctypes.addressof(dummy), n, ndms, t_end, 8, ctypes.addressof(dummy),
                                                                   1, ctypes.addressof(dummy), None, ctypes.byref(err))
    assert call(B.PEAKS_NOALLOC_MAX_CANDS + 1, 16, 1000) == B.AA_ERR_LIMIT and err.value == 0
    assert call(10, B.PEAKS_NOALLOC_MAX_CELLS + 1, 1000) == B.AA_ERR_LIMIT
    assert call(10, 0, 1000) == B.AA_ERR_INVALID and call(10, 16, 0) == B.AA_ERR_INVALID
    assert lib.aa_find_peaks_device_noalloc(None, 10, 16, 1000, 8, None, 0, ctypes.addressof(dummy), None, None) == B.AA_ERR_INVALID
    assert lib.aa_find_peaks_device_noalloc(None, 0, 16, 1000, 8, None, 0, None, None, None) == B.AA_ERR_INVALID
    assert b"AA_PEAKS_NOALLOC_MAX" in lib.aa_strerror(B.AA_ERR_LIMIT)


@pytest.mark.gpu
def test_two_calls_in_a_row_equal_the_host_peak_finder(B):
    """Back-to-back calls on the shared array: a large list on a fine grid, then a small one on a different grid shape
    (stale chains of the first call lie exactly where the second one looks), then the first again, then an empty one.
    Each must equal aa_find_peaks (the library's host path) of the same list."""
    import torch
    rng = np.random.default_rng(2101)
    cases = [(200_000, 500, 1 << 20, 64), (3_000, 40, 5_000, 256), (200_000, 500, 1 << 20, 64), (0, 7, 100, 4),
             (50_000, 3, 1 << 22, 16),                 # few rows, long span
             (60_000, 1 << 16, 4096, 8)]              # many rows: the grid is coarsened to fit the fixed array
    lists = [_random_list(B, rng, *c) for c in cases]
    lists[2] = lists[0]
    for k, (c, (n, ndms, t_end, wmax)) in enumerate(zip(lists, cases)):
        want = B.find_peaks(c)
        n_got, got = _device_peaks(B, torch, c, ndms, t_end, wmax, order_rng=rng)
        assert n_got == len(want), (k, n_got, len(want))
        assert got.tobytes() == want.tobytes(), k
        assert n == 0 or 0 < len(want) < len(c)


@pytest.mark.gpu
def test_same_peaks_as_the_plan_path_on_a_searched_observation(B):
    """The list a real search produces (cfg1-shaped noise + a pulse, low threshold): the entry point, fed aa_run's
    candidates, must return what aa_run itself returns in output_mode 1 (the arena-backed device kernels + host border
    settling), twice in a row, with a different list in between."""
    import torch
    w = I.scaled(I.workload(1), nsamp=1 << 16, norm_block=1 << 14, chunk_len=1 << 15, n_streams=2, snr_threshold=3.5,
                 pulses=(I.Pulse(dm=50.0, t0=20000, width=8, amp=3.0),), name="noalloc")
    host = B.pinned_empty(w.nbytes)
    I.fill(w, host.numpy().reshape(w.nsamp, w.nchans))
    with B.Plan(w) as plan:
        cands, _ = plan.run(host, want_taps=False)
    with B.Plan(w, peaks=True) as plan:
        want, _ = plan.run(host, want_taps=False)
    wmax = max(w.widths) * max(r.bin for r in w.ranges)
    assert 0 < len(want) < len(cands) <= B.PEAKS_NOALLOC_MAX_CANDS
    other = _random_list(B, np.random.default_rng(5), 20_000, w.ndms_total, 9_000, 32)
    for c, ref in ((cands, want), (other, B.find_peaks(other)), (cands, want)):
        t_end = int(c["t_start"].max()) + 1
        n_got, got = _device_peaks(B, torch, c, w.ndms_total, t_end, wmax)
        assert n_got == len(ref) and got.tobytes() == _sorted(ref).tobytes()


@pytest.mark.gpu
def test_small_output_buffer_and_out_of_range_records(B):
    """*n_out is the true number of peaks even when `out` is too small (the stored ones are peaks); records outside
    the declared rows / span are ignored instead of indexing past the grid."""
    import torch
    rng = np.random.default_rng(9)
    c = _random_list(B, rng, 5_000, 30, 20_000, 16)
    want = B.find_peaks(c)
    n_got, got = _device_peaks(B, torch, c, 30, 20_000, 16, out_cap=10)
    assert n_got == len(want) and len(got) == 10
    assert set(map(bytes, got)) <= set(map(bytes, want))
    bad = c.copy()
    bad["dm_index"][::7] += 1000                                  # rows that do not exist
    bad["t_start"][3::11] += 1 << 30                              # far outside the span
    keep = (bad["dm_index"] < 30) & (bad["t_start"] < 20_000)
    n_got, got = _device_peaks(B, torch, bad, 30, 20_000, 16)
    ref = B.find_peaks(_sorted(bad[keep]))
    assert n_got == len(ref) and got.tobytes() == ref.tobytes()
