"""The seeded generator: C and numpy statements agree; statistics and pulses are as described."""
import math

import numpy as np

from paper_2101_00941_b200 import inputs as I


def test_c_matches_numpy_restatement():
    w = I.scaled(I.workload(1), nsamp=4096, pulses=())
    x = I.fill(w)
    ref = I.noise_numpy(w.noise_seed, 0, w.nsamp * w.nchans).reshape(w.nsamp, w.nchans)
    assert np.array_equal(x, ref)


def test_noise_law():
    w = I.scaled(I.workload(2), nsamp=1 << 16, pulses=())
    x = I.fill(w).astype(np.float64)
    assert abs(x.mean() - 128.0) < 0.02
    assert abs(x.std() - np.sqrt(256.0 + 1.0 / 12.0)) < 0.02      # quantisation adds 1/12
    # neighbouring samples are uncorrelated
    a = x[:-1].ravel() - 128.0
    b = x[1:].ravel() - 128.0
    assert abs((a * b).mean() / 256.0) < 5e-3


def test_quantile_table_is_the_8bit_gaussian_law():
    cdf = I.quantile_table(128.0).astype(np.float64) / 2.0 ** 32
    assert np.all(np.diff(cdf) >= 0)
    assert abs(cdf[127] - 0.5 * (1 + math.erf(-0.5 / 16 / math.sqrt(2)))) < 1e-9   # P(X <= 127)
    assert abs(cdf[128 + 16] - 0.8490) < 2e-3     # Phi(16.5/16)


def test_pulse_is_where_the_recipe_says():
    w = I.workload(1)
    x = I.fill(w)
    p = w.pulses[0]
    off = I.pulse_offsets(w, p.dm)
    assert off[0] == 0 and np.all(np.diff(off) >= 0)
    on = np.array([x[p.t0 + off[c]: p.t0 + off[c] + p.width, c].mean() for c in range(w.nchans)])
    assert abs(on.mean() - (128 + 48)) < 2.0
    # sample() reproduces single elements without the buffer
    for t, c in [(0, 0), (p.t0, 0), (p.t0 + off[40] + 3, 40), (w.nsamp - 1, w.nchans - 1)]:
        assert I.sample(w, t, c) == x[t, c]


def test_workload_table_matches_baseline_configs():
    w3, w4, w5 = I.workload(3), I.workload(4), I.workload(5)
    assert (w3.nchans, w3.nsamp, w3.ndms_total, w3.snr_threshold) == (4096, 1 << 23, 2048, 7.0)
    assert w4.ndms_total == 6050 and [r.bin for r in w4.ranges] == [1, 2, 4, 8, 16, 32]
    assert w5.nsamp == 1 << 24 and len(w5.pulses) == 64 and w5.nbytes == 68719476736
    assert I.workload(2).widths == (1, 2, 4, 8, 16, 32, 64, 128)
    assert I.workload(1).widths == (1, 2, 4, 8, 16, 32)


def test_fill_span_equals_the_slice_of_the_whole():
    """A rank of a time-sharded run generates only its own rows (counter-based generator + clipped pulses)."""
    w = I.scaled(I.workload(1), nsamp=9000,
                 pulses=(I.Pulse(dm=50.0, t0=2990, width=8, amp=3.0), I.Pulse(dm=120.0, t0=5990, width=32, amp=2.0)))
    x = I.fill(w)
    for t_first, n in [(0, 9000), (3000, 3000), (2995, 10), (6000, 3000), (8999, 1)]:
        assert np.array_equal(I.fill_span(w, t_first, n), x[t_first:t_first + n]), (t_first, n)
