"""GPU parity on the BASELINE.json workloads: full cfg1/cfg2, sampled rows/blocks of cfg3-cfg5.

Sampled checks: the oracle dedisperses chosen DM rows over chosen normalisation blocks (rows and
blocks are independent) and runs its statistics / boxcars / candidate rule on them;
the GPU's tapped rows must match bit for bit and its candidates in those (row, block) cells must
match under the north_star tolerances.  cfg4 (6050 trials) and cfg5 (68.7 GB pinned) run at full size
when the host has the memory for them (AA_FULL=0 skips them, AA_FULL=1 forces them); reduced-length
variants of them always run.
"""
import os

import numpy as np
import pytest

import oracle
from paper_2101_00941_b200 import inputs as I
from _compare import compare_candidates

pytestmark = pytest.mark.gpu


def _host_gb():
    try:
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable:"):
                    return int(line.split()[1]) / 1e6
    except OSError:
        pass
    return 0.0


def _full(need_gb):
    v = os.environ.get("AA_FULL", "")
    return v == "1" or (v != "0" and _host_gb() >= need_gb)



@pytest.fixture(scope="module")
def B():
    from paper_2101_00941_b200 import binding
    binding.load_library()
    return binding


def _pinned_fill(B, w):
    buf = B.pinned_empty(w.nbytes)
    x = buf.numpy().reshape(w.nsamp, w.row_bytes)
    I.fill(w, x)
    return buf, x


def _global_rows(w, per_range):
    """{range: [local rows]} -> sorted global tap indices and a lookup (range, row) -> tap row."""
    taps, base = [], 0
    for r, rg in enumerate(w.ranges):
        taps += [base + d for d in per_range.get(r, [])]
        base += rg.ndms
    taps = sorted(set(taps))
    return taps, {g: k for k, g in enumerate(taps)}


def _check_cells(w, x, cands, tap, tapidx, cells):
    """cells: list of (range, [rows], block index)."""
    from concurrent.futures import ThreadPoolExecutor
    geo = oracle.geometry(w)
    base = np.cumsum([0] + [rg.ndms for rg in w.ranges])
    wmax = max(w.widths)
    n_checked = n_cands = 0
    # candidates of each tapped row, once (the list is sorted by (dm_index, t_start))
    lo = np.searchsorted(cands["dm_index"], np.arange(int(base[-1]) + 1))
    for r, rows, k in cells:
        rg = w.ranges[r]
        Lr = w.norm_block // rg.bin
        nout = geo["nout"][r]
        t0 = k * Lr
        if t0 >= nout:
            continue
        nblk = min(Lr, nout - t0)
        ntau = min(Lr + wmax - 1, nout - t0)
        D = oracle.dedisperse(x, w, r, rows=rows, tau_first=t0, ntau=ntau, geo=geo)

        def one(i):
            d = rows[i]
            g = int(base[r]) + d
            got = tap[tapidx[g], t0:t0 + nblk]
            assert np.array_equal(got, D[i, :nblk]), f"dedispersed row differs: range {r} dm {d} block {k}"
            tau, ww, sn = oracle.sps_row(D[i], w, r, d_first=t0, tau_a=t0, tau_b=t0 + nblk, nout=nout)
            ref = oracle.pack_candidates(g, rg.bin, tau, ww, sn)
            row = cands[lo[g]:lo[g + 1]]
            sel = (row["t_start"] >= t0 * rg.bin) & (row["t_start"] < (t0 + nblk) * rg.bin)
            compare_candidates(row[sel], ref, w.snr_threshold)
            return len(ref)

        with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
            for n in ex.map(one, range(len(rows))):
                n_checked += 1
                n_cands += n
    return n_checked, n_cands


def _stratified_cells(w, subchunk_len, n_rows=64, n_seams=3, n_random_blocks=2, seed=0, max_pulses=16):
    """SURVEY 8(d) / BASELINE.md section 3: at least `n_rows` DM rows (first and last trial, both trials at every
    range edge, every injected DM +-1, the rest seeded-random), each checked on normalisation blocks spread over the
    whole time span: the first block, the ragged last one, both blocks on either side of `n_seams` sub-chunk seams,
    and `n_random_blocks` seeded-random ones.  Returns the cell list for _check_cells."""
    geo = oracle.geometry(w)
    rng = np.random.default_rng(2101_00941 + seed)
    base = np.cumsum([0] + [rg.ndms for rg in w.ranges])
    rows = set()
    for r, rg in enumerate(w.ranges):
        rows |= {int(base[r]), int(base[r]) + rg.ndms - 1}
        for p in w.pulses[:max_pulses]:
            hi = rg.dm_low + rg.dm_step * (rg.ndms - 1)
            if rg.dm_low <= p.dm <= hi and rg.dm_step > 0:
                d = int(round((p.dm - rg.dm_low) / rg.dm_step))
                rows |= {int(base[r]) + min(max(d + e, 0), rg.ndms - 1) for e in (-1, 0, 1)}
    while len(rows) < n_rows:
        rows.add(int(rng.integers(0, base[-1])))
    per_range = {}
    for g in sorted(rows):
        r = int(np.searchsorted(base, g, side="right")) - 1
        per_range.setdefault(r, []).append(g - int(base[r]))
    nblocks = -(-geo["t_valid"] // w.norm_block)                  # blocks on the raw time axis (the last one ragged)
    per_sub = subchunk_len // w.norm_block
    n_sub = -(-geo["t_valid"] // subchunk_len)
    seams = sorted({int(v) for v in np.linspace(1, max(1, n_sub - 1), n_seams)}) if n_sub > 1 else []
    blocks = {0, nblocks - 1}
    for j in seams:                                               # sub-chunk j starts at block j * per_sub
        blocks |= {j * per_sub - 1, j * per_sub}
    while len(blocks) < 2 + 2 * len(seams) + n_random_blocks and len(blocks) < nblocks:
        blocks.add(int(rng.integers(0, nblocks)))
    blocks = sorted(b for b in blocks if 0 <= b < nblocks)
    cells = [(r, rws, k) for k in blocks for r, rws in sorted(per_range.items())]
    return cells, len(rows), blocks


def _pulse_cells(w, geo, max_pulses=4, extra=()):
    """(range, rows around the pulse's DM, block holding the pulse) for a few injected pulses."""
    cells = []
    for p in w.pulses[:max_pulses]:
        for r, rg in enumerate(w.ranges):
            hi = rg.dm_low + rg.dm_step * (rg.ndms - 1)
            if rg.dm_low <= p.dm <= hi and rg.dm_step > 0:
                d = int(round((p.dm - rg.dm_low) / rg.dm_step))
                rows = sorted({max(0, d - 1), d, min(rg.ndms - 1, d + 1)})
                cells.append((r, rows, p.t0 // w.norm_block))
                break
    return cells + list(extra)


def test_cfg2_full_streamed_equals_single_stream_and_oracle(B):
    w = I.workload(2)                                  # 4 streams x 4 time chunks
    buf, x = _pinned_fill(B, w)
    taps = list(range(w.ndms_total))
    with B.Plan(w, taps=taps) as plan:
        c4, t4 = plan.run(buf)
        assert plan.info["n_subchunks"] == 16 and not plan.overflow
        nout = plan.nout[0]
    with B.Plan(w, taps=taps, n_streams=1, chunk_len=1 << 20) as plan:
        c1, t1 = plan.run(buf)
    assert c4.tobytes() == c1.tobytes() and np.array_equal(t4, t1)     # streamed == single stream
    ref, dense, geo = oracle.run(x, w, keep_dense=True)
    assert np.array_equal(t4[:, :nout], dense[0])                      # bit-exact dedispersed series
    res = compare_candidates(c4, ref, w.snr_threshold)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0
    # every injected pulse is recovered near its DM / time with a width within a factor two
    for p in w.pulses:
        near = c4[(np.abs(c4["dm_index"].astype(float) - p.dm) <= 4) & (np.abs(c4["t_start"].astype(float) - p.t0) <= 2 * p.width + 2)]
        expect = p.amp * np.sqrt(w.nchans * p.width) / 0.98487
        if expect < 2 * w.snr_threshold:
            continue
        assert len(near), p
        top = near[np.argmax(near["snr"])]
        assert top["snr"] >= 0.6 * expect and 0.5 * p.width <= top["width"] <= 2 * max(p.width, 1), (p, top)


def test_cfg1_cfg2_peaks_on_the_device(B):
    """cfg1 and cfg2 in output_mode 1 return exactly the peaks of the oracle's candidate list."""
    for k in (1, 2):
        w = I.workload(k)
        buf, x = _pinned_fill(B, w)
        with B.Plan(w, peaks=True) as plan:
            got, _ = plan.run(buf, want_taps=False)
            st = plan.stats()
        ref, _ = oracle.run(x, w)
        want = oracle.find_peaks_fast(ref)
        assert st["n_candidates"] == len(ref) and len(want) < len(ref) / 10
        assert got.tobytes() == want.tobytes(), k
        # the strongest peak sits on the strongest injected pulse
        top = got[np.argmax(got["snr"])]
        assert any(abs(int(top["dm_index"]) - p.dm) <= 2 and abs(int(top["t_start"]) - p.t0) <= 2 * p.width + 2 for p in w.pulses)


def _run_sampled(B, w, cells_extra, max_pulses=4, also_streams=(), **plan_kw):
    buf, x = _pinned_fill(B, w)
    geo = oracle.geometry(w)
    cells = _pulse_cells(w, geo, max_pulses=max_pulses, extra=cells_extra)
    # one oracle call per (range, block): merge the row lists of cells that share them
    merged = {}
    for r, rows, k in cells:
        merged.setdefault((k, r), set()).update(rows)
    cells = [(r, sorted(rows), k) for (k, r), rows in sorted(merged.items())]
    per_range = {}
    for r, rows, _ in cells:
        per_range.setdefault(r, set()).update(rows)
    taps, tapidx = _global_rows(w, {r: sorted(v) for r, v in per_range.items()})
    with B.Plan(w, taps=taps, **plan_kw) as plan:
        cands, tap = plan.run(buf, max_cands=1 << 24)
        assert not plan.overflow
        assert plan.info["maxshift"] == geo["maxshift"] and plan.nout == geo["nout"]
        stats = plan.stats()
    for ns in also_streams:                                       # same buffer, other stream counts: identical output
        kw = dict(plan_kw, n_streams=ns)
        with B.Plan(w, taps=taps, **kw) as plan:
            c2, t2 = plan.run(buf, max_cands=1 << 24)
            assert not plan.overflow and plan.info["n_subchunks"] >= ns
            assert c2.tobytes() == cands.tobytes() and np.array_equal(t2, tap), f"{ns} streams differ"
        del c2, t2
    n_cells, n_ref = _check_cells(w, x, cands, tap, tapidx, cells)
    return cands, n_cells, n_ref, stats


def test_cfg3_full_size_sampled(B):
    """Workload and launch configuration bench.py times: 4096 x 2^23, 2048 trials, 8 streams.  >= 64 stratified DM
    rows, each on blocks over the whole time span (first, ragged last, both sides of sub-chunk seams, random), plus
    the block holding every injected pulse on the rows around its DM."""
    w = I.workload(3)
    extra, n_rows, blocks = _stratified_cells(w, w.chunk_len // w.n_streams)
    assert n_rows >= 64 and len(blocks) >= 9
    cands, n_cells, n_ref, stats = _run_sampled(B, w, extra, max_pulses=len(w.pulses))
    assert n_cells >= 64 * 9 and n_ref > 0
    assert stats["h2d_bytes"] == w.nbytes                     # every input byte crosses the link once


def test_cfg4_reduced_length_sampled(B):
    w = I.scaled(I.workload(4), nsamp=1 << 19, chunk_len=1 << 18, n_streams=4, name="cfg4_short")
    extra = [(r, [0, w.ranges[r].ndms // 2, w.ranges[r].ndms - 1], k) for r in range(6) for k in (0, 6)]
    w = I.scaled(w, pulses=(I.Pulse(dm=100.0, t0=70000, width=8, amp=0.3), I.Pulse(dm=700.4, t0=200000, width=64, amp=0.1),
                            I.Pulse(dm=2000.0, t0=300000, width=256, amp=0.05)))
    cands, n_cells, n_ref, _ = _run_sampled(B, w, extra)
    assert n_cells >= 36 and n_ref > 0


def test_cfg4_shape_measured_sigma_sampled(B):
    """Reading A18 on the multi-range plan (B:configs[3]): ranges 0-4 keep per-width statistics in the cluster kernel, range 5
    (bin 32: 255 * 4096 * 32 * 256 >= 2^32, 64-bit boxcar sums) in the generic kernel; sampled rows x blocks of every range
    against the oracle."""
    w = I.scaled(I.workload(4), nsamp=1 << 19, chunk_len=1 << 18, n_streams=4, name="cfg4_short_a18", sigma_mode=1)
    w = I.scaled(w, pulses=(I.Pulse(dm=100.0, t0=70000, width=8, amp=0.3), I.Pulse(dm=700.4, t0=200000, width=64, amp=0.1),
                            I.Pulse(dm=2000.0, t0=300000, width=256, amp=0.05)))
    extra = [(r, [0, w.ranges[r].ndms // 2, w.ranges[r].ndms - 1], k) for r in range(6) for k in (0, 6)]
    cands, n_cells, n_ref, _ = _run_sampled(B, w, extra)
    assert n_cells >= 36 and n_ref > 0


def test_cfg5_reduced_length_sampled_16_streams(B):
    w = I.scaled(I.workload(5), nsamp=1 << 21, chunk_len=1 << 20, n_streams=16, name="cfg5_short")
    extra = [(0, [0, 2047], 0), (0, [1000], 17), (0, [1, 2046], 31)]
    cands, n_cells, n_ref, _ = _run_sampled(B, w, extra)
    assert n_cells >= 5


@pytest.mark.parametrize("n_streams", [32, 64])
def test_cfg3_shape_many_streams_sampled(B, n_streams):
    """aa.h takes n_streams up to 64: the headline workload's shape with 65536-sample sub-chunks, one per stream, so
    that every one of the 32 / 64 streams (and host threads) runs a sub-chunk; stratified rows x blocks (first, ragged
    last, both sides of sub-chunk seams) against the oracle, and the whole list against the 4-stream run's."""
    w = I.scaled(I.workload(3), nsamp=n_streams << 16, chunk_len=n_streams << 16, n_streams=n_streams,
                 name=f"cfg3_{n_streams}streams")
    w = I.scaled(w, pulses=(I.Pulse(dm=300.0, t0=150000, width=16, amp=0.35), I.Pulse(dm=1500.0, t0=(n_streams << 16) // 2, width=128, amp=0.12)))
    extra, n_rows, blocks = _stratified_cells(w, 1 << 16, n_rows=12, n_seams=3, n_random_blocks=1, max_pulses=2)
    assert len(blocks) >= 7
    buf, x = _pinned_fill(B, w)
    taps, tapidx = _global_rows(w, {0: sorted({d for _, rows, _ in extra for d in rows})})
    with B.Plan(w, taps=taps, max_cands_per_subchunk=1 << 18) as plan:
        assert plan.info["n_subchunks"] == n_streams and plan.info["subchunk_len"] == 1 << 16
        cands, tap = plan.run(buf, max_cands=1 << 22)
        assert not plan.overflow and plan.stats()["n_streams"] == n_streams
    n_cells, n_ref = _check_cells(w, x, cands, tap, tapidx, extra)
    assert n_cells >= 12 * 7 and n_ref > 0
    with B.Plan(w, taps=taps, n_streams=4, max_cands_per_subchunk=1 << 18) as plan:
        c4, t4 = plan.run(buf, max_cands=1 << 22)
    assert c4.tobytes() == cands.tobytes() and np.array_equal(t4, tap)


@pytest.mark.parametrize("variant", [dict(nbits=4), dict(nbits=16), dict(sigma_mode=1), dict(wdec=16), dict(sigma_mode=1, wdec=16),
                                     dict(nbits=16, sigma_mode=1)],
                         ids=["4bit", "16bit", "measured-sigma", "decimated-widths", "measured-sigma+decimated", "16bit+measured-sigma"])
def test_cfg3_shape_search_variants_sampled(B, variant):
    """The S:8(f) rows (readings A18-A20) on the headline workload's shape: 4096 channels, 2048 trials, 131072-sample
    sub-chunks on 4 streams, the kernels bench.py times plus the ones these variants select (per-width statistics and
    coarse grids in the first cluster kernel, 64-bit boxcar sums for 16-bit input); sampled rows x blocks against the oracle."""
    w = I.scaled(I.workload(3), nsamp=1 << 19, chunk_len=1 << 19, n_streams=4, name="cfg3_short", **variant)
    w = I.scaled(w, pulses=(I.Pulse(dm=300.0, t0=150000, width=16, amp=0.35), I.Pulse(dm=1500.0, t0=300000, width=128, amp=0.12)))
    extra = [(0, [0, 1023, 2047], 0), (0, [7, 640], 3), (0, [0, 2047], 7)]      # block 7 is the ragged last one
    cands, n_cells, n_ref, _ = _run_sampled(B, w, extra, max_pulses=2)
    assert n_cells >= 10 and n_ref > 0


@pytest.mark.skipif(not _full(60), reason="needs 34.4 GB pinned + headroom (AA_FULL=1 forces it)")
def test_cfg4_full_size_sampled(B):
    w = I.workload(4)
    extra, n_rows, blocks = _stratified_cells(w, w.chunk_len // w.n_streams, n_seams=2, n_random_blocks=1)
    assert n_rows >= 64 and len(blocks) >= 6
    cands, n_cells, n_ref, _ = _run_sampled(B, w, extra, max_pulses=len(w.pulses))
    assert n_cells >= 64 * 6 and n_ref > 0


@pytest.mark.skipif(not _full(110), reason="needs 68.7 GB of pinned host memory + headroom (AA_FULL=1 forces it)")
def test_cfg5_full_size_sampled(B):
    w = I.workload(5)
    n_streams = 8
    extra, n_rows, blocks = _stratified_cells(w, w.chunk_len // n_streams, n_seams=2, n_random_blocks=1)
    assert n_rows >= 64 and len(blocks) >= 6
    # B:configs[4] asks for a stream sweep up to 16: the 16-stream run (65536-sample sub-chunks) must return the
    # 8-stream run's bytes, which are the ones compared with the oracle
    cands, n_cells, n_ref, stats = _run_sampled(B, w, extra, max_pulses=8, also_streams=(16,), n_streams=n_streams)
    assert n_cells >= 64 * 6 and n_ref > 0
    assert stats["h2d_bytes"] == w.nbytes
