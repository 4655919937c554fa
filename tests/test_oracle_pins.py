"""Pins for the CPU oracle: what the problem statement and the mathematics fix.

Every check compares the oracle with something other than itself: exact rational
arithmetic, numpy reductions, closed forms, python-loop brute force on tiny
inputs, or values recorded in tests/golden/ with their citation.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2101_00941_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# --------------------------------------------------------------------------- delays
def _exact_delay(w, rg, c, i):
    """delay in exact rational arithmetic, rounded half up (north_star formula)."""
    F = lambda v: Fraction(repr(float(v)))
    f_c = F(w.f_top) + c * F(w.foff)
    dm = F(rg.dm_low) + i * F(rg.dm_step)
    v = Fraction("4148.808") * dm * (1 / (f_c * f_c) - 1 / (F(w.f_top) ** 2)) / (F(w.tsamp) * rg.bin)
    return math.floor(v + Fraction(1, 2))


@pytest.mark.parametrize("k", [1, 2, 3, 4])
def test_delays_against_exact_rationals(k):
    w = I.workload(k)
    rng = np.random.default_rng(k)
    for r, rg in enumerate(w.ranges):
        dl = oracle.delays(w, r)
        assert dl.shape == (rg.ndms, w.nchans)
        assert np.all(dl[:, 0] == 0)                      # reference frequency is f_top (A4)
        if rg.dm_low == 0.0:
            assert np.all(dl[0] == 0)                     # DM = 0 has no delay
        assert np.all(np.diff(dl, axis=1) >= 0)           # later at lower frequency
        assert np.all(np.diff(dl, axis=0) >= 0)           # later at higher DM
        for _ in range(40):
            i = int(rng.integers(0, rg.ndms)); c = int(rng.integers(0, w.nchans))
            assert dl[i, c] == _exact_delay(w, rg, c, i)
        assert dl[-1, -1] == _exact_delay(w, rg, w.nchans - 1, rg.ndms - 1)


def test_delay_maxima_golden():
    rows = [l.split() for l in open(os.path.join(GOLD, "delay_maxima.txt")) if l.strip() and l[0] != "#"]
    for k, r, mx in rows:
        w = I.workload(int(k))
        assert int(oracle.delays(w, int(r)).max()) == int(mx), (k, r)


def test_textbook_delay_value():
    # 4.15 ms * DM * (f_lo^-2 - f_hi^-2) with f in GHz: DM=100 between 1.5 and 1.2 GHz = 103.7 ms
    class W: nchans = 2; f_top = 1500.0; foff = -300.0; tsamp = 1e-3; ranges = (I.DMRange(100.0, 1.0, 1, 1),)
    assert int(oracle.delays(W, 0)[0, 1]) == 104


def test_geometry_matches_survey_sizes():
    # maxshift 159 / 1336 / 29660, cfg4 36224 (= 32*1132)
    for k, ms in [(1, 159), (2, 1336), (3, 29660), (4, 36224)]:
        g = oracle.geometry(I.workload(k))
        assert g["maxshift"] == ms
        assert g["t_valid"] == I.workload(k).nsamp - ms
    g4 = oracle.geometry(I.workload(4))
    assert g4["nout"] == [(8388608 - 36224) // b for b in (1, 2, 4, 8, 16, 32)]
    # W = sum ndms*nout = 1.92e10 for cfg4, 1.71e10 for cfg3
    W4 = sum(r.ndms * n for r, n in zip(I.workload(4).ranges, g4["nout"]))
    assert abs(W4 / 1.92e10 - 1) < 0.01


# --------------------------------------------------------------------------- dedispersion
def _tiny(nchans=8, nsamp=600, bins=(1,), ndms=6, dm_step=20.0, seed=0, **kw):
    ranges = tuple(I.DMRange(0.0 if j == 0 else 30.0 * j, dm_step, ndms, b) for j, b in enumerate(bins))
    w = I.Workload(name="tiny", nchans=nchans, nsamp=nsamp, tsamp=64e-6, f_top=1500.0, foff=-8.0,
                   ranges=ranges, widths=(1, 2, 4), snr_threshold=4.0, n_streams=1, chunk_len=nsamp,
                   noise_seed=1234 + seed, pulses=(), norm_block=kw.pop("norm_block", 64), **kw)
    return w


def test_dm0_row_is_the_channel_sum():
    w = I.scaled(I.workload(1), nsamp=8192, pulses=())
    x = I.fill(w)
    geo = oracle.geometry(w)
    D = oracle.dedisperse(x, w, 0, rows=[0], geo=geo)
    assert np.array_equal(D[0], x[:geo["nout"][0]].astype(np.uint32).sum(axis=1))


def test_constant_input():
    w = _tiny(bins=(1, 2, 4))
    x = np.full((w.nsamp, w.nchans), 7, dtype=np.uint8)
    for r, rg in enumerate(w.ranges):
        D = oracle.dedisperse(x, w, r)
        assert np.all(D == 7 * w.nchans * rg.bin)


def test_single_impulse_lands_at_t_minus_delay():
    w = _tiny(nchans=8, nsamp=900, ndms=8)
    geo = oracle.geometry(w)
    dl = geo["delays"][0]
    for c, t0 in [(0, 100), (3, 417), (7, 650)]:
        x = np.zeros((w.nsamp, w.nchans), dtype=np.uint8); x[t0, c] = 1
        D = oracle.dedisperse(x, w, 0, geo=geo)
        for d in range(dl.shape[0]):
            tau = t0 - dl[d, c]
            expect = np.zeros(geo["nout"][0], dtype=np.uint32)
            if 0 <= tau < geo["nout"][0]:
                expect[tau] = 1
            assert np.array_equal(D[d], expect), (c, d)


@pytest.mark.parametrize("bins", [(1,), (2,), (1, 4), (8,), (3,), (1, 6), (5, 10)])
def test_dedispersion_brute_force_python_loops(bins):
    w = _tiny(nchans=6, nsamp=520, bins=bins, ndms=5, seed=len(bins))
    x = I.fill(w)
    geo = oracle.geometry(w)
    for r, rg in enumerate(w.ranges):
        D = oracle.dedisperse(x, w, r, geo=geo)
        dl = geo["delays"][r]
        assert D.shape == (rg.ndms, geo["nout"][r])
        for d in range(rg.ndms):
            for tau in range(0, geo["nout"][r], 7):
                s = 0
                for c in range(w.nchans):
                    for i in range(rg.bin):
                        s += int(x[rg.bin * (tau + dl[d, c]) + i, c])
                assert D[d, tau] == s


def test_binned_zero_delay_is_the_pairwise_summed_channel_sum():
    w = _tiny(bins=(4,), ndms=1)      # one trial at DM 0
    x = I.fill(w)
    geo = oracle.geometry(w)
    D = oracle.dedisperse(x, w, 0, geo=geo)
    cs = x.astype(np.uint32).sum(axis=1)
    n = geo["nout"][0]
    assert np.array_equal(D[0], cs[:4 * n].reshape(n, 4).sum(axis=1))


def test_sub_range_equals_slice_of_whole():
    w = _tiny(nchans=8, nsamp=2000, ndms=6)
    x = I.fill(w)
    geo = oracle.geometry(w)
    D = oracle.dedisperse(x, w, 0, geo=geo)
    part = oracle.dedisperse(x, w, 0, rows=[1, 4], tau_first=300, ntau=500, geo=geo)
    assert np.array_equal(part, D[[1, 4], 300:800])


def test_total_is_conserved_away_from_edges():
    w = _tiny(nchans=8, nsamp=3000, ndms=4)
    geo = oracle.geometry(w)
    x = np.zeros((w.nsamp, w.nchans), dtype=np.uint8)
    rng = np.random.default_rng(3)
    lo, hi = geo["maxshift"], w.nsamp - geo["maxshift"] - 1
    x[lo:hi] = rng.integers(0, 256, size=(hi - lo, w.nchans))
    D = oracle.dedisperse(x, w, 0, geo=geo)
    assert np.all(D.sum(axis=1, dtype=np.uint64) == x.sum(dtype=np.uint64))


# --------------------------------------------------------------------------- other input bit depths (reading A19)
def test_unpack_hand_made_bytes():
    class W4: nsamp = 2; nchans = 4; nbits = 4
    x = np.array([[0x21, 0xF0], [0x0A, 0x37]], dtype=np.uint8)
    assert oracle.unpack(x, W4).tolist() == [[1, 2, 0, 15], [10, 0, 7, 3]]        # even channel = low nibble
    class W16: nsamp = 1; nchans = 2; nbits = 16
    x = np.array([[0x34, 0x12, 0xFF, 0xFF]], dtype=np.uint8)
    assert oracle.unpack(x, W16).tolist() == [[0x1234, 0xFFFF]]                    # little-endian words


@pytest.mark.parametrize("nbits,bins", [(4, (1, 2)), (16, (1,)), (16, (3,))])
def test_other_bit_depths_brute_force_and_linearity(nbits, bins):
    w = I.scaled(_tiny(nchans=6, nsamp=520, bins=bins, ndms=5, seed=nbits), nbits=nbits)
    x = I.fill(w)
    u = oracle.unpack(x, w).astype(np.int64)
    geo = oracle.geometry(w)
    for r, rg in enumerate(w.ranges):
        D = oracle.dedisperse(x, w, r, geo=geo)
        dl = geo["delays"][r]
        for d in range(rg.ndms):
            for tau in range(0, geo["nout"][r], 11):                                # python loops over the definition
                assert D[d, tau] == sum(int(u[rg.bin * (tau + dl[d, c]) + i, c]) for c in range(w.nchans) for i in range(rg.bin))
        # dedispersion is linear: the 16-bit result is 256 x (high bytes) + (low bytes), the 4-bit one that of the nibbles as bytes
        w8 = I.scaled(w, nbits=8)
        if nbits == 16:
            hi = oracle.dedisperse(np.ascontiguousarray(x[:, 1::2]), w8, r, geo=geo).astype(np.uint64)
            lo = oracle.dedisperse(np.ascontiguousarray(x[:, 0::2]), w8, r, geo=geo).astype(np.uint64)
            assert np.array_equal(D.astype(np.uint64), 256 * hi + lo)
        else:
            assert np.array_equal(D, oracle.dedisperse(u.astype(np.uint8), w8, r, geo=geo))


def test_stats_with_sums_of_squares_beyond_64_bits():
    """16-bit input on thousands of channels: 65536 samples near 2^28 have a sum of squares near 2^72."""
    rng = np.random.default_rng(5)
    d = (rng.integers(0, 1 << 20, size=70000) + (1 << 28)).astype(np.int64)
    d[rng.integers(0, d.size, 40)] += 1 << 27
    mu, sg, n = oracle.block_stats(d.astype(np.uint32))
    pm, ps, pn = _py_stats(d)
    assert sum(int(v) * int(v) for v in d) > 2 ** 64
    assert n == pn and mu == pm and abs(sg - ps) <= 1e-12 * ps


# --------------------------------------------------------------------------- statistics
def _py_stats(d):
    """Python restatement with exact integers (fractions) and numpy selection."""
    d = np.asarray(d, dtype=np.int64)
    sel = np.ones(d.size, dtype=bool)
    mu = sg = 0.0
    for it in range(4):
        if it:
            sel = np.abs(d.astype(np.float64) - mu) <= 3.0 * sg
        v = [int(a) for a in d[sel]]
        m = len(v)
        if m == 0:
            break
        S1, S2 = sum(v), sum(a * a for a in v)
        mu = float(Fraction(S1, m))
        sg = math.sqrt(float(Fraction(m * S2 - S1 * S1, m * m)))
    return mu, sg, int(sel.sum())


def test_stats_without_outliers_is_numpy_mean_std():
    rng = np.random.default_rng(0)
    d = rng.integers(1000, 2000, size=5000).astype(np.uint32)      # uniform: max dev = 1.73 sigma < 3 sigma
    mu, sg, n = oracle.block_stats(d)
    assert n == d.size
    assert abs(mu - d.mean()) < 1e-9 and abs(sg - d.std()) < 1e-9


def test_stats_matches_python_restatement_with_outliers():
    rng = np.random.default_rng(1)
    for trial in range(5):
        d = np.rint(rng.normal(8192, 128, size=4000)).astype(np.int64)
        d[rng.integers(0, d.size, 30)] += rng.integers(500, 5000, 30)
        mu, sg, n = oracle.block_stats(d.astype(np.uint32))
        pm, ps, pn = _py_stats(d)
        assert n == pn and mu == pm and abs(sg - ps) <= 1e-12 * ps


def test_stats_clipped_gaussian_fixed_point():
    # three 3-sigma clips of a Gaussian: sigma -> 0.98487 sigma0 (closed form below)
    phi = lambda k: math.exp(-k * k / 2) / math.sqrt(2 * math.pi)
    Phi = lambda k: 0.5 * (1 + math.erf(k / math.sqrt(2)))
    f = 1.0
    for _ in range(3):
        k = 3.0 * f
        f = math.sqrt(1 - 2 * k * phi(k) / (2 * Phi(k) - 1))
    assert abs(f - 0.98487) < 1e-4
    rng = np.random.default_rng(2)
    d = np.rint(rng.normal(1 << 20, 4096.0, size=1 << 18)).astype(np.uint32)
    mu, sg, n = oracle.block_stats(d)
    assert abs(sg / 4096.0 - f) < 0.004
    assert abs(mu - (1 << 20)) < 40
    assert abs(n / d.size - (2 * Phi(3 * 0.98505) - 1)) < 0.002


def test_stats_constant_block_and_outlier_rejection():
    mu, sg, n = oracle.block_stats(np.full(100, 77, dtype=np.uint32))
    assert (mu, sg, n) == (77.0, 0.0, 100)
    d = np.tile(np.array([99, 101], dtype=np.uint32), 500)
    d[10] = 100000; d[11] = 100000                     # removes one 99 and one 101
    mu, sg, n = oracle.block_stats(d)
    assert (mu, sg, n) == (100.0, 1.0, 998)


# --------------------------------------------------------------------------- S/N and candidates
class _W:
    """Minimal workload for sps_row: one un-binned range."""
    def __init__(self, widths, thr, norm_block, b=1):
        self.widths = tuple(widths); self.snr_threshold = thr; self.norm_block = norm_block
        self.ranges = (I.DMRange(0.0, 1.0, 1, b),)


def test_snr_closed_form_on_a_hand_made_row():
    # alternating 99/101 -> mu = 100, sigma = 1 once the two spikes are clipped away
    d = np.tile(np.array([99, 101], dtype=np.uint32), 64)
    d[40] = 100 + 20; d[41] = 100 + 20
    w = _W((1, 2, 4), 5.0, 128)
    tau, ww, sn = oracle.sps_row(d, w, 0, nout=d.size)
    got = {int(t): (int(a), float(s)) for t, a, s in zip(tau, ww, sn)}
    # tau=40: S_1 = 20, S_2 = 40/sqrt2 = 28.28 (best), S_4 = (20+20-1+1)/2 = 20
    assert got[40][0] == 2 and abs(got[40][1] - 40 / math.sqrt(2)) < 1e-12
    # tau=41: S_1 = 20, S_2 = (20-1)/sqrt2 = 13.4, S_4 = (20 -1 +1 -1)/2 = 9.5 -> w = 1
    assert got[41] == (1, 20.0)
    # tau=39: S_1 = +1, S_2 = 21/sqrt2 = 14.85, S_4 = (1+20+20-1)/2 = 20 -> w = 4
    assert got[39] == (4, 20.0)
    # tau=38: S_4 = (-1+1+20+20)/2 = 20; tau=37: S_4 = (1-1+1+20)/2 = 10.5
    assert got[38] == (4, 20.0) and got[37] == (4, 10.5)
    assert sorted(got) == [37, 38, 39, 40, 41]


def _py_candidates(d, widths, thr, L, nout):
    out = []
    for b0 in range(0, nout, L):
        b1 = min(b0 + L, nout)
        mu, sg, _ = _py_stats(d[b0:b1])
        if not sg > 0 or b1 - b0 < 32:
            continue
        for tau in range(b0, b1):
            best = None
            for wd in widths:
                if tau + wd > nout:
                    continue
                S = (float(sum(int(v) for v in d[tau:tau + wd])) - wd * mu) / (sg * math.sqrt(wd))
                if best is None or S > best[1]:
                    best = (wd, S)
            if best is not None and best[1] >= thr:
                out.append((tau, best[0], best[1]))
    return out


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_candidate_rule_brute_force(seed):
    rng = np.random.default_rng(seed)
    nout, L = 300, 64                      # last block has 44 samples; with nout=270 it would have 14
    nout = 300 if seed != 2 else 270
    d = np.rint(rng.normal(5000, 50, size=nout)).astype(np.uint32)
    d[70:74] += 120; d[200] += 400; d[nout - 2:] += 300
    widths = (1, 2, 3, 8)
    w = _W(widths, 3.0, L)
    tau, ww, sn = oracle.sps_row(d, w, 0, nout=nout)
    ref = _py_candidates(d, widths, 3.0, L, nout)
    assert [int(t) for t in tau] == [r[0] for r in ref]
    assert [int(a) for a in ww] == [r[1] for r in ref]
    assert np.allclose(sn, [r[2] for r in ref], rtol=1e-13, atol=0)
    if seed == 2:
        assert all(t < 256 for t in tau)       # the 14-sample last block emits nothing (A13)


# ---- readings A20 (long boxcars on a coarser time grid) and A18 (statistics of each width's own series) ----------
def _dec(wd, wdec):
    dec = 1
    while wdec > 0 and wd > wdec * dec:
        dec *= 2
    return dec


def _py_candidates_variants(d, widths, thr, L, nout, wdec, sigma_mode):
    """The definition in python loops: exact integer boxcars, statistics through the exact-fraction restatement."""
    out = []
    for b0 in range(0, nout, L):
        b1 = min(b0 + L, nout)
        mu, sg, _ = _py_stats(d[b0:b1])
        if not sg > 0 or b1 - b0 < 32:
            continue
        ws = {}
        if sigma_mode:
            for wd in widths:
                series = [sum(int(v) for v in d[t:t + wd]) for t in range(b0, b1) if t % _dec(wd, wdec) == 0 and t + wd <= nout]
                ws[wd] = _py_stats(np.array(series, dtype=np.int64))[:2] if len(series) >= 32 else (0.0, 0.0)
        for tau in range(b0, b1):
            best = None
            for wd in widths:
                if tau + wd > nout or tau % _dec(wd, wdec) != 0:
                    continue
                B = float(sum(int(v) for v in d[tau:tau + wd]))
                if sigma_mode:
                    if not ws[wd][1] > 0:
                        continue
                    S = (B - ws[wd][0]) / ws[wd][1]
                else:
                    S = (B - wd * mu) / (sg * math.sqrt(wd))
                if best is None or S > best[1]:
                    best = (wd, S)
            if best is not None and best[1] >= thr:
                out.append((tau, best[0], best[1]))
    return out


class _WV(_W):
    def __init__(self, widths, thr, norm_block, wdec=0, sigma_mode=0):
        super().__init__(widths, thr, norm_block)
        self.wdec = wdec; self.sigma_mode = sigma_mode


@pytest.mark.parametrize("wdec,sigma_mode", [(2, 0), (4, 0), (0, 1), (2, 1), (3, 1)])
def test_search_variants_brute_force(wdec, sigma_mode):
    rng = np.random.default_rng(10 * wdec + sigma_mode)
    nout, L = 900, 256                     # last block has 132 samples: on a grid of 8 that is 17 < 32 boxcars
    d = np.rint(rng.normal(5000, 50, size=nout)).astype(np.uint32)
    d[71:79] += 90; d[200] += 400; d[250:266] += 60; d[600:605] += 110; d[nout - 3:] += 300
    widths = (1, 2, 5, 8, 16)
    tau, ww, sn = oracle.sps_row(d, _WV(widths, 3.0, L, wdec, sigma_mode), 0, nout=nout)
    ref = _py_candidates_variants(d, widths, 3.0, L, nout, wdec, sigma_mode)
    assert len(ref) > 10 and len({r[1] for r in ref}) >= 3
    assert [int(t) for t in tau] == [r[0] for r in ref]
    assert [int(a) for a in ww] == [r[1] for r in ref]
    assert np.allclose(sn, [r[2] for r in ref], rtol=1e-12, atol=0)


def test_decimated_widths_are_the_full_search_on_a_coarser_grid():
    rng = np.random.default_rng(3)
    d = np.rint(rng.normal(9000, 70, size=2048)).astype(np.uint32)
    d[1001:1017] += 150                                             # 16-sample pulse starting at an odd sample
    widths = (1, 2, 4, 8, 16, 32)
    full = oracle.sps_row(d, _WV(widths, 5.0, 1024), 0, nout=d.size)
    assert np.array_equal(oracle.sps_row(d, _WV(widths, 5.0, 1024, wdec=32), 0, nout=d.size)[0], full[0])   # wdec >= wmax: nothing changes
    tau, ww, sn = oracle.sps_row(d, _WV(widths, 5.0, 1024, wdec=4), 0, nout=d.size)        # dec = 1 1 1 2 4 8
    for t, a in zip(tau, ww):
        assert t % _dec(int(a), 4) == 0
    best_full = int(full[0][np.argmax(full[2])]), int(full[1][np.argmax(full[2])])
    assert best_full == (1001, 16)                                   # the full search finds the pulse where it is
    k = np.argmax(sn)
    assert int(ww[k]) == 16 and int(tau[k]) in (1000, 1004) and sn[k] < full[2].max()    # the grid of width 16 is 4 samples
    # a candidate of the decimated search at a tau on every grid has exactly the S/N of the full search there
    both = {int(t): float(s) for t, a, s in zip(full[0], full[1], full[2])}
    for t, a, s in zip(tau, ww, sn):
        if t % 8 == 0 and int(t) in both:
            assert s == both[int(t)]


def test_series_statistics():
    rng = np.random.default_rng(8)
    d = rng.integers(1000, 2000, size=5000).astype(np.uint32)
    assert oracle.series_stats(d.astype(np.uint64)) == oracle.block_stats(d)      # width 1: the block statistics themselves
    v = (rng.integers(0, 1 << 22, size=3000) + (1 << 35)).astype(np.int64)        # boxcar sums of 16-bit data: past 2^32
    v[rng.integers(0, v.size, 25)] += 1 << 30
    mu, sg, n = oracle.series_stats(v.astype(np.uint64))
    pm, ps, pn = _py_stats(v)
    assert n == pn and mu == pm and abs(sg - ps) <= 1e-12 * ps


def test_measured_sigma_of_white_noise_follows_sqrt_w():
    """Reading A18 on Gaussian noise: the boxcar series of width w has sigma_w = 0.98487 sigma sqrt(w) (three 3-sigma
    clips) and mean w mu, so the two S/N scalings agree to a few per cent; they differ when the noise is not white."""
    rng = np.random.default_rng(12)
    d = np.rint(rng.normal(50000, 300, size=1 << 16)).astype(np.uint32)
    d[30000:30008] += 1500
    widths = (1, 4, 16)
    a = oracle.sps_row(d, _WV(widths, 8.0, 1 << 16), 0, nout=d.size)
    b = oracle.sps_row(d, _WV(widths, 8.0, 1 << 16, sigma_mode=1), 0, nout=d.size)
    ta, tb = int(a[0][np.argmax(a[2])]), int(b[0][np.argmax(b[2])])
    assert abs(ta - 30000) <= 4 and abs(tb - 30000) <= 4
    assert abs(a[2].max() / b[2].max() - 1) < 0.05
    for w_ in widths:
        series = np.convolve(d.astype(np.int64), np.ones(w_, dtype=np.int64), "valid")
        mu, sg, _ = oracle.series_stats(series.astype(np.uint64))
        # overlapping boxcars are correlated samples of the same Gaussian: the clip factor is still 0.98487
        assert abs(mu / (w_ * 50000.0) - 1) < 1e-3 and abs(sg / (0.98487 * 300 * math.sqrt(w_)) - 1) < 0.03


def test_boxcar_may_run_into_the_next_block_but_not_past_the_end():
    d = np.tile(np.array([99, 101], dtype=np.uint32), 64)     # two blocks of 64
    d[62:66] = 140
    w = _W((4,), 5.0, 64)
    tau, ww, sn = oracle.sps_row(d, w, 0, nout=128)
    assert 62 in tau and 61 in tau                 # boxcars starting in block 0 use samples of block 1
    tau2, _, _ = oracle.sps_row(d[:126], w, 0, nout=126)
    assert np.all(tau2 + 4 <= 126)


def test_cfg1_injected_pulse_recovered_exactly():
    w = I.workload(1)
    x = I.fill(w)
    c, geo = oracle.run(x, w)
    top = c[np.argmax(c["snr"])]
    p = w.pulses[0]
    assert (top["dm_index"], top["t_start"], top["width"]) == (50, p.t0, p.width)
    expect = p.amp * math.sqrt(w.nchans * p.width) / 0.98487           # SURVEY §8(c) pin table
    assert abs(top["snr"] - expect) < 3.0
    # sorted by (dm_index, t_start), one per (dm, t)
    key = c["dm_index"].astype(np.int64) << 32 | c["t_start"]
    assert np.all(np.diff(key) > 0)
    # noise-only: Gaussian tail gives ~0.1 expected candidates at 6 sigma
    w0 = I.scaled(w, pulses=())
    c0, _ = oracle.run(I.fill(w0), w0)
    assert len(c0) <= 3


def test_binned_range_units_are_raw_samples():
    w = _tiny(nchans=8, nsamp=6000, bins=(1, 4), ndms=3, norm_block=256)
    x = I.fill(w)
    geo = oracle.geometry(w)
    t0 = 2000
    for c in range(w.nchans):
        x[t0 + 4 * geo["delays"][1][1, c]: t0 + 4 * geo["delays"][1][1, c] + 8, c] = 255
    c, _ = oracle.run(x, w)
    hit = c[(c["dm_index"] == 3 + 1)]
    top = hit[np.argmax(hit["snr"])]
    assert top["t_start"] == t0 and top["width"] == 8 and top["t_start"] % 4 == 0


# ---- peak finding (reading A17) ----------------------------------------------------------------------------
def _cl(rows):
    a = np.zeros(len(rows), dtype=oracle.CAND_DTYPE)
    for i, r in enumerate(rows):
        a[i] = r
    return a


def test_peaks_hand_made_cases():
    # an isolated candidate is a peak; a clump keeps its maximum only
    c = _cl([(5, 100, 4, 7.0), (5, 102, 4, 9.0), (6, 101, 8, 8.0), (5, 300, 1, 6.5)])
    assert [tuple(x) for x in oracle.find_peaks(c)] == [(5, 102, 4, 9.0), (5, 300, 1, 6.5)]
    # touching boxcars (t' == t + w) are neighbours, a gap of one sample is not
    c = _cl([(0, 10, 5, 8.0), (0, 15, 2, 7.0), (0, 18, 2, 6.0)])
    assert [int(x["t_start"]) for x in oracle.find_peaks(c)] == [10, 18]
    # DM distance 2 is not a neighbour, distance 1 is
    c = _cl([(3, 50, 4, 9.0), (5, 50, 4, 8.0), (4, 50, 4, 7.0)])
    assert [int(x["dm_index"]) for x in oracle.find_peaks(c)] == [3, 5]
    # equal S/N: the smaller (dm_index, t_start) wins, so exactly one of a tie survives
    c = _cl([(7, 20, 4, 8.0), (7, 22, 4, 8.0), (6, 23, 4, 8.0)])
    assert [tuple(x)[:2] for x in oracle.find_peaks(c)] == [(6, 23)]
    # the rule is a local maximum, not a transitive clustering: a chain 9 > 8 > 7 with the ends apart keeps 9 and 7's
    # other-side survivor only if nothing beats it
    c = _cl([(1, 0, 4, 9.0), (1, 4, 4, 8.0), (1, 8, 4, 7.0), (1, 100, 4, 6.1)])
    assert [int(x["t_start"]) for x in oracle.find_peaks(c)] == [0, 100]
    assert len(oracle.find_peaks(_cl([]))) == 0


def test_fast_peak_finding_is_the_all_pairs_rule():
    """aaor_find_peaks (rows dm-1..dm+1, starts in [t - wmax, t + w]) against the all-pairs definition on random lists
    with clumps, exact S/N ties, touching boxcars and gaps of one sample."""
    rng = np.random.default_rng(17)
    for trial in range(6):
        n = 400
        a = np.zeros(n, dtype=oracle.CAND_DTYPE)
        a["dm_index"] = rng.integers(0, 12, n)
        a["t_start"] = rng.integers(0, 300, n) * (1 if trial % 2 else 4)
        a["width"] = rng.choice([1, 2, 4, 8, 32], n)
        a["snr"] = rng.integers(6, 12, n).astype(np.float32) + (rng.random(n) < 0.5) * rng.random(n).astype(np.float32)
        key = (a["dm_index"].astype(np.uint64) << np.uint64(32)) | a["t_start"].astype(np.uint64)
        _, first = np.unique(key, return_index=True)                 # one candidate per (dm, t), sorted
        a = a[np.sort(first)]
        a = a[np.lexsort((a["t_start"], a["dm_index"]))]
        slow, fast = oracle.find_peaks(a), oracle.find_peaks_fast(a)
        assert 0 < len(slow) < len(a) and slow.tobytes() == fast.tobytes()


def test_peaks_invariants_on_a_real_candidate_list():
    """peaks are a subset; no two peaks are neighbours; every dropped candidate has a neighbour that beats it;
    the injected cfg1 pulse gives one peak at exactly (DM 50, t 20000, w 8)."""
    w = I.scaled(I.workload(1), nsamp=1 << 16, norm_block=1 << 14, pulses=(I.Pulse(dm=50.0, t0=20000, width=8, amp=3.0),))
    x = I.fill(w)
    cands, _ = oracle.run(x, w)
    assert len(cands) > 1000
    peaks = oracle.find_peaks(cands)
    assert 0 < len(peaks) < len(cands) // 20
    key = lambda a: set(zip(a["dm_index"].tolist(), a["t_start"].tolist()))
    assert key(peaks) <= key(cands)
    d, t, ww, s = (peaks[k].astype(np.float64) for k in ("dm_index", "t_start", "width", "snr"))
    for i in range(len(peaks)):
        nb = (np.abs(d - d[i]) <= 1) & (t <= t[i] + ww[i]) & (t[i] <= t + ww)
        assert nb.sum() == 1                                   # only itself
    top = peaks[np.argmax(peaks["snr"])]
    assert (int(top["dm_index"]), int(top["t_start"]), int(top["width"])) == (50, 20000, 8)
    near = peaks[(np.abs(peaks["dm_index"].astype(int) - 50) <= 1) & (np.abs(peaks["t_start"].astype(int) - 20000) <= 8)]
    assert len(near) == 1
