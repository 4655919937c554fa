"""aa_find_peaks (host code of libaa, no GPU needed) against the oracle's all-pairs definition (reading A17)."""
import numpy as np
import pytest

import oracle
from paper_2101_00941_b200 import inputs as I


@pytest.fixture(scope="module")
def B():
    from paper_2101_00941_b200 import binding, build
    build.build_cuda()
    binding.load_library()
    return binding


def _sorted(a):
    return a[np.lexsort((a["t_start"], a["dm_index"]))]


def test_random_lists_match_the_oracle(B):
    rng = np.random.default_rng(17)
    for n, ndm, span, wmax in [(0, 1, 1, 1), (1, 1, 10, 4), (300, 6, 400, 16), (2000, 40, 3000, 64), (1500, 3, 500, 256)]:
        c = np.zeros(n, dtype=oracle.CAND_DTYPE)
        c["dm_index"] = rng.integers(0, ndm, n) * rng.choice([1, 1, 2], n)      # gaps between rows too
        c["t_start"] = rng.integers(0, span, n)
        c["width"] = 2 ** rng.integers(0, int(np.log2(wmax)) + 1, n)
        c["snr"] = np.round(rng.uniform(6, 12, n), 1).astype(np.float32)        # many exact ties
        # one record per (dm, t) as aa_run produces
        _, first = np.unique(np.stack([c["dm_index"], c["t_start"]]), axis=1, return_index=True)
        c = _sorted(c[np.sort(first)])
        want = oracle.find_peaks(c)
        for nthreads in (1, 3, 0):
            got = B.find_peaks(c, nthreads=nthreads)
            assert got.tobytes() == want.tobytes(), (n, nthreads)


def test_candidate_list_of_a_pulse(B):
    w = I.scaled(I.workload(1), nsamp=1 << 16, norm_block=1 << 14, pulses=(I.Pulse(dm=50.0, t0=20000, width=8, amp=3.0),))
    cands, _ = oracle.run(I.fill(w), w)
    got = B.find_peaks(cands)
    assert got.tobytes() == oracle.find_peaks(cands).tobytes() and 0 < len(got) < len(cands) // 20
    top = got[np.argmax(got["snr"])]
    assert (int(top["dm_index"]), int(top["t_start"]), int(top["width"])) == (50, 20000, 8)


def test_unsorted_input_and_small_output_are_reported(B):
    c = np.zeros(3, dtype=oracle.CAND_DTYPE)
    c["dm_index"] = [2, 1, 1]
    with pytest.raises(B.AAError):
        B.find_peaks(c)
    import ctypes
    c = _sorted(c)
    c["t_start"] = [0, 1000, 0]
    c = _sorted(c)
    lib = B.load_library()
    out = np.empty(1, dtype=oracle.CAND_DTYPE)
    n = ctypes.c_uint64(0)
    c["snr"] = 7.0
    rc = lib.aa_find_peaks(c.ctypes.data, 3, out.ctypes.data, 1, ctypes.byref(n), 1)
    assert rc == B.AA_ERR_OVERFLOW and n.value == 2
