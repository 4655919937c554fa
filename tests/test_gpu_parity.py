"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element."""
import numpy as np
import pytest

import oracle
from paper_2101_00941_b200 import inputs as I
from _compare import compare_candidates

pytestmark = pytest.mark.gpu


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


def _run_gpu(B, w, buf, *, taps="all", **kw):
    tap_list = list(range(w.ndms_total)) if taps == "all" else taps
    with B.Plan(w, taps=tap_list, **kw) as plan:
        cands, tap = plan.run(buf)
        assert not plan.overflow
        return cands, tap, plan.info, plan.nout, plan.stats()


def _check_against_oracle(B, w, mutate=None, **kw):
    buf, x = _pinned_fill(B, w)
    if mutate is not None:
        mutate(x)
    cands, tap, info, nout, _ = _run_gpu(B, w, buf, **kw)
    ref, dense, geo = oracle.run(x, w, keep_dense=True)
    assert info["maxshift"] == geo["maxshift"] and nout == geo["nout"]
    base = 0
    for r, rg in enumerate(w.ranges):
        got = tap[base:base + rg.ndms, :geo["nout"][r]]
        assert np.array_equal(got, dense[r]), f"dedispersed series differ in range {r}"
        base += rg.ndms
    res = compare_candidates(cands, ref, w.snr_threshold)
    return cands, ref, res


def _tiny(nchans=16, nsamp=20000, bins=(1,), ndms=40, dm_step=3.0, widths=(1, 2, 4, 8), thr=5.0,
          norm_block=1024, n_streams=1, chunk_len=4096, seed=0, f_top=1500.0, foff=-4.0):
    ranges, lo = [], 0.0
    for b in bins:
        ranges.append(I.DMRange(lo, dm_step, ndms, b))
        lo += dm_step * ndms
    w = I.Workload(name="tiny", nchans=nchans, nsamp=nsamp, tsamp=64e-6, f_top=f_top, foff=foff,
                   ranges=tuple(ranges), widths=tuple(widths), snr_threshold=thr, n_streams=n_streams,
                   chunk_len=chunk_len, noise_seed=99 + seed,
                   pulses=(I.Pulse(dm=dm_step * ndms * 0.4, t0=nsamp // 3, width=4, amp=4.0),
                           I.Pulse(dm=dm_step * ndms * len(bins) * 0.8, t0=nsamp // 2, width=16, amp=2.0)),
                   norm_block=norm_block)
    return w


def test_delay_tables_match_oracle_entry_by_entry(B):
    for k in (1, 2, 4):
        w = I.scaled(I.workload(k), nsamp=1 << 17, chunk_len=1 << 17, n_streams=1, pulses=())
        with B.Plan(w) as plan:
            for r in range(len(w.ranges)):
                assert np.array_equal(plan.delays(r), oracle.delays(w, r).astype(np.int32))


@pytest.mark.parametrize("case", [
    dict(),                                                     # one range, several sub-chunks
    dict(nchans=24, ndms=37, nsamp=15001),                      # ragged channels / trials / tail
    dict(bins=(1, 2, 4), nsamp=40000, chunk_len=8192),          # time decimation
    dict(bins=(8,), nsamp=60000, chunk_len=16384, ndms=20),
    dict(n_streams=3, chunk_len=3 * 2048, nsamp=30000),         # streams
    dict(widths=(1, 3, 5, 32), thr=4.0),                        # arbitrary widths
    dict(nchans=300, nsamp=12000, foff=-0.3, dm_step=4.0, chunk_len=4096, norm_block=2048),  # flushes of the 16-bit lanes
    # bins that are not 2..32 powers of two: the generic binning kernel
    dict(bins=(3,), norm_block=1536, chunk_len=3 * 1536, nsamp=30000),
    dict(bins=(1, 6), norm_block=1536, chunk_len=4 * 1536, nsamp=40000),
    dict(bins=(5, 10), norm_block=1280, chunk_len=5 * 1280, nsamp=50000, n_streams=5),
    dict(bins=(2, 3), norm_block=1536, chunk_len=4 * 1536, nsamp=40000, nchans=30),          # fused and generic binning together
    dict(bins=(64,), norm_block=4096, chunk_len=32768, nsamp=200000, ndms=12),
    dict(bins=(128,), norm_block=8192, chunk_len=65536, nsamp=400000, ndms=8, widths=(1, 2, 4)),
])
def test_small_cases_bit_exact(B, case):
    w = _tiny(**case)
    cands, ref, res = _check_against_oracle(B, w)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0 and res["width_ties"] == 0
    assert len(ref) > 0


@pytest.mark.parametrize("case", [
    dict(norm_block=32768, chunk_len=32768, nsamp=150000, ndms=6),            # SPS cluster of 2 CTAs per block
    dict(norm_block=65536, chunk_len=65536, nsamp=200001, ndms=5),            # cluster of 4, ragged last block
    dict(norm_block=131072, chunk_len=131072, nsamp=300000, ndms=4),          # cluster of 8
    dict(norm_block=131072, chunk_len=131072, nsamp=140000, ndms=4),          # ... most CTAs of the cluster hold no data
    dict(norm_block=262144, chunk_len=262144, nsamp=300000, ndms=3),          # too long for a cluster: generic kernel
    dict(bins=(8,), norm_block=1040, chunk_len=8 * 1040, nsamp=50000, ndms=12),   # block of 130 samples: generic kernel
    dict(widths=(2, 6, 7, 12, 20, 33), thr=4.5, norm_block=4096, chunk_len=8192),  # every width alignment
    dict(nchans=30, nsamp=20011, ndms=33),                                    # byte-wise corner turn (nchans % 4 != 0)
    dict(nchans=20, bins=(4,), widths=(1, 2, 4, 4096), nsamp=120000, chunk_len=32768, norm_block=32768, ndms=6, thr=4.0),  # long boxcar tail
])
def test_sps_and_corner_turn_variants(B, case):
    """Shapes that select each SPS kernel (cluster sizes 1-8, generic fallback) and each corner-turn kernel."""
    w = _tiny(**case)
    cands, ref, res = _check_against_oracle(B, w)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0 and res["width_ties"] == 0
    assert len(ref) > 0


def _interference(kind):
    """Input rows that defeat the fast statistics path of sps_cluster2_kernel (listed outliers + totals): the kernel
    must then walk the whole segment for the remaining clip passes and still return the oracle's numbers."""
    def mutate(x):
        nsamp = x.shape[0]
        if kind == "burst":            # 12 % of one stretch far above the noise: the outlier lists overflow
            a = nsamp // 3
            x[a:a + nsamp // 8, :] = 250
        elif kind == "spikes":         # a few enormous samples: sigma collapses after the first clip, the 3-sigma interval
            x[nsamp // 5::997, :] = 255    # of the next pass falls inside the core of the first guess
            x[nsamp // 7::1013, :] = 0
        elif kind == "constant":       # sigma = 0 over whole blocks: nothing may be emitted there
            x[: nsamp // 2, :] = 77
        elif kind == "steps":          # two levels: the plain moments put the core between them
            x[::2, :] = 10
            x[1::2, :] = 240
        elif kind == "dense_spikes":   # 5 % of the samples four sigma out: more listed samples than a cluster's lists hold
            x[3::20, :] = 255
        elif kind == "almost_constant":  # sigma far below one count: no integer lies within 2.75 sigma of the mean
            x[:, :] = 77
            x[nsamp // 3, 0] = 78
            x[nsamp // 3 + 40000, 1] = 79
    return mutate


@pytest.mark.parametrize("sps_variant", [0, 1])
@pytest.mark.parametrize("kind", ["burst", "spikes", "constant", "steps", "dense_spikes", "almost_constant"])
@pytest.mark.parametrize("case", [
    dict(norm_block=16384, chunk_len=16384, nsamp=70000, ndms=6),             # one CTA per block
    dict(norm_block=65536, chunk_len=65536, nsamp=200001, ndms=4),            # cluster of 4, ragged last block
    dict(norm_block=131072, chunk_len=131072, nsamp=300000, ndms=3),          # cluster of 8
])
def test_sps_statistics_under_interference(B, case, kind, sps_variant):
    """Both cluster kernels (sps_variant 1 keeps the first one) on rows whose statistics take the slow path."""
    w = _tiny(**case)
    cands, ref, res = _check_against_oracle(B, w, mutate=_interference(kind), sps_variant=sps_variant)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0 and res["width_ties"] == 0


@pytest.mark.parametrize("case", [
    dict(norm_block=32768, chunk_len=32768, nsamp=150000, ndms=6),
    dict(norm_block=65536, chunk_len=65536, nsamp=200001, ndms=5),
    dict(widths=(2, 6, 7, 12, 20, 33), thr=4.5, norm_block=4096, chunk_len=8192),
    dict(widths=(1, 2, 3, 4, 8, 9), thr=4.5, norm_block=8192, chunk_len=8192, nsamp=40000),
])
def test_first_cluster_kernel_still_matches(B, case):
    """aa_plan_desc.sps_variant = 1: sps_cluster_kernel where sps_cluster2_kernel would run."""
    w = _tiny(**case)
    cands, ref, res = _check_against_oracle(B, w, sps_variant=1)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0 and res["width_ties"] == 0
    assert len(ref) > 0


@pytest.mark.parametrize("variant,code", [("ws1024", 4), ("ws512", 3), ("sp1024", 2), ("sp512", 1), ("plain", 0), ("auto", None)])
@pytest.mark.parametrize("case", [
    dict(nchans=302, ndms=100, nsamp=21000, chunk_len=8192),                 # padded channel group, partial DM block, ragged tile
    dict(nchans=1024, ndms=64, nsamp=9000, chunk_len=4096, foff=-0.2),      # four flushes of the 16-bit lanes
    dict(nchans=1029, ndms=33, nsamp=9000, chunk_len=4096, foff=-0.2),      # second half of the DM block holds one trial
])
def test_every_dedispersion_kernel_bit_exact(B, variant, code, case):
    """Fine channels / fine DM steps so that the shared-pattern tables exist; aa_plan_desc.dedisp_variant picks the kernel."""
    kw = dict(f_top=1500.0, foff=-0.5, dm_step=0.25, norm_block=1024, widths=(1, 2, 4, 8), thr=5.0)
    kw.update(case)
    w = _tiny(**kw)
    buf, x = _pinned_fill(B, w)
    with B.Plan(w, taps=list(range(w.ndms_total)), dedisp_variant=variant) as plan:
        # the plan's own choice on these shapes is the warp-specialised kernel, with either tile length
        assert plan.dedisp_variant(0) == code or (code is None and plan.dedisp_variant(0) in (3, 4))
        cands, tap = plan.run(buf)
        nout = plan.nout
    ref, dense, geo = oracle.run(x, w, keep_dense=True)
    assert np.array_equal(tap[:, :geo["nout"][0]], dense[0])
    res = compare_candidates(cands, ref, w.snr_threshold)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0


@pytest.mark.parametrize("variant,code", [("ws1024", 4), ("ws512", 3)])
@pytest.mark.parametrize("case", [
    dict(bins=(2,), nchans=302, ndms=100, nsamp=40000, chunk_len=16384),                 # padded channel group, ragged everything
    dict(bins=(2,), nchans=1024, ndms=64, nsamp=30000, chunk_len=8192, foff=-0.2),       # 8 flushes of the 16-bit lanes
    dict(bins=(4,), nchans=1024, ndms=64, nsamp=40000, chunk_len=16384, foff=-0.2),      # 16 flushes of the 16-bit lanes
    dict(bins=(8,), nchans=512, ndms=130, nsamp=80000, chunk_len=32768, foff=-0.4),      # flush every 8 groups
    dict(bins=(1, 2, 8), nchans=256, ndms=70, nsamp=60000, chunk_len=16384),             # mixed 8-bit and binned ranges
    dict(bins=(16,), nchans=512, ndms=70, nsamp=160000, chunk_len=65536, foff=-0.4, norm_block=4096),   # flush every 4 groups
    dict(bins=(32,), nchans=516, ndms=66, nsamp=300000, chunk_len=131072, foff=-0.4, norm_block=8192),  # 32-bit accumulators
    dict(bins=(3,), nchans=302, ndms=100, nsamp=60000, chunk_len=4 * 3072, norm_block=3072),           # generic binning kernel
    dict(bins=(6, 12), nchans=512, ndms=70, nsamp=120000, chunk_len=8 * 3072, norm_block=3072, foff=-0.4),
    dict(bins=(48,), nchans=516, ndms=66, nsamp=400000, chunk_len=16 * 6144, foff=-0.4, norm_block=6144),  # 32-bit accumulators
    dict(bins=(64,), nchans=512, ndms=66, nsamp=500000, chunk_len=131072, foff=-0.4, norm_block=8192),    # 4*255*64 = 65280: the limit of the 16-bit rows
    dict(bins=(96,), nchans=512, ndms=40, nsamp=700000, chunk_len=16 * 12288, foff=-0.4, norm_block=12288),  # past it: plain kernel
])
def test_binned_input_on_the_shared_pattern_kernel(B, variant, code, case):
    """Time-binned (uint16) ranges on the warp-specialised shared-pattern kernel, against the oracle."""
    kw = dict(f_top=1500.0, foff=-0.5, dm_step=0.25, norm_block=2048, widths=(1, 2, 4, 8), thr=5.0)
    kw.update(case)
    w = _tiny(**kw)
    buf, x = _pinned_fill(B, w)
    with B.Plan(w, taps=list(range(w.ndms_total)), dedisp_variant=variant) as plan:
        # bins 32..64: the 32-bit-accumulator variant; coarser: four-channel sums overflow 16 bits -> plain kernel
        want = [0 if rg.bin > 64 else 5 if rg.bin >= 32 else code for rg in w.ranges]
        assert [plan.dedisp_variant(r) for r in range(len(w.ranges))] == want
        cands, tap = plan.run(buf)
    ref, dense, geo = oracle.run(x, w, keep_dense=True)
    base = 0
    for r, rg in enumerate(w.ranges):
        assert np.array_equal(tap[base:base + rg.ndms, :geo["nout"][r]], dense[r]), f"range {r}"
        base += rg.ndms
    res = compare_candidates(cands, ref, w.snr_threshold)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0


@pytest.mark.parametrize("nbits,case", [
    (4, dict(nchans=16, nsamp=20000)),                                                    # plain kernel
    (4, dict(nchans=30, nsamp=20011, ndms=33, bins=(1, 2))),                              # ragged, binned
    (4, dict(nchans=302, ndms=100, nsamp=21000, chunk_len=8192, foff=-0.5, dm_step=0.25, norm_block=1024)),   # shared-pattern kernel
    (16, dict(nchans=16, nsamp=20000)),
    (16, dict(nchans=24, ndms=37, nsamp=15001, bins=(1, 4), chunk_len=8192, n_streams=2)),
    (16, dict(nchans=302, ndms=100, nsamp=21000, chunk_len=8192, foff=-0.5, dm_step=0.25, norm_block=1024)),  # both planes on the shared-pattern kernel
    (16, dict(nchans=1024, ndms=40, nsamp=30000, chunk_len=8192, foff=-0.2, dm_step=0.25, norm_block=4096, widths=(1, 2, 4, 64))),  # 128-bit statistics, 64-bit boxcars
])
def test_other_input_bit_depths(B, nbits, case):
    """DESIGN.md reading A19: 4-bit (nibbles unpacked on the device) and 16-bit (two 8-bit planes, D = D(low) + 256 D(high))
    input against the oracle, dense plane bit for bit."""
    w = I.scaled(_tiny(**case), nbits=nbits)
    cands, ref, res = _check_against_oracle(B, w)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0 and res["width_ties"] == 0
    assert len(ref) > 0


@pytest.mark.parametrize("case", [
    dict(wdec=2),                                                                        # plain shapes, generic SPS kernel (block 1024 = 4 * 256: cluster of 1)
    dict(wdec=1, widths=(1, 2, 3, 8, 32), thr=4.0),
    dict(wdec=4, widths=(1, 2, 4, 8, 16, 32, 64), norm_block=65536, chunk_len=65536, nsamp=200001, ndms=5),     # cluster of 4, grids up to 16
    dict(wdec=2, widths=(2, 6, 7, 12, 20, 33), thr=4.5, norm_block=4096, chunk_len=8192),  # unaligned widths on coarse grids
    dict(wdec=1, widths=(1, 2, 4, 4096), bins=(4,), nchans=20, nsamp=120000, chunk_len=32768, norm_block=32768, ndms=6, thr=4.0),  # grid 4096 > the group distance
    dict(wdec=8, bins=(8,), norm_block=1040, chunk_len=8 * 1040, nsamp=50000, ndms=12, widths=(1, 4, 16, 32)),   # generic kernel (block of 130)
    dict(sigma_mode=1),
    dict(sigma_mode=1, wdec=2, widths=(1, 2, 4, 8, 16, 32), norm_block=4096, chunk_len=8192),
    dict(sigma_mode=1, norm_block=65536, chunk_len=65536, nsamp=200001, ndms=5, widths=(1, 2, 4, 8, 16, 32, 64, 128)),   # cluster of 4, ragged last block
    dict(sigma_mode=1, wdec=4, norm_block=131072, chunk_len=131072, nsamp=300000, ndms=4, widths=(1, 3, 8, 64)),        # cluster of 8
    dict(sigma_mode=1, bins=(1, 2, 4), nsamp=40000, chunk_len=8192, n_streams=2),
    dict(sigma_mode=1, nchans=302, ndms=100, nsamp=21000, chunk_len=8192, foff=-0.5, dm_step=0.25, norm_block=1024, n_streams=2),
    # A18 outside the cluster kernel: per-width statistics swept tile by tile in the generic kernel
    dict(sigma_mode=1, bins=(8,), norm_block=1040, chunk_len=8 * 1040, nsamp=50000, ndms=12, widths=(1, 4, 16, 32)),     # block of 130 samples: no cluster
    dict(sigma_mode=1, wdec=4, bins=(8,), norm_block=1040, chunk_len=8 * 1040, nsamp=50000, ndms=12, widths=(1, 4, 16, 32, 64)),
    dict(sigma_mode=1, bins=(8,), norm_block=20816, chunk_len=41632, nsamp=150000, ndms=6, widths=(1, 2, 3, 8, 100)),   # block of 2602 samples: two tiles per block, ragged
    dict(sigma_mode=1, nbits=16, nchans=300, nsamp=12000, foff=-0.3, dm_step=4.0, chunk_len=4096, norm_block=2048, widths=(1, 2, 4, 8, 256), thr=4.0),   # 64-bit boxcar sums
    dict(sigma_mode=1, wdec=2, nbits=16, nchans=1024, ndms=40, nsamp=30000, chunk_len=8192, foff=-0.2, dm_step=0.25, norm_block=4096, widths=(1, 2, 4, 64)),  # 128-bit block statistics too
    dict(sigma_mode=1, norm_block=2048, chunk_len=4096, nsamp=4096 * 3 + 40, widths=(1, 2, 4, 8, 64)),                  # last block shorter than 32 + w: widths without statistics
])
def test_search_variants_a18_a20(B, case):
    """Readings A20 (long boxcars on a coarser time grid) and A18 (S/N from each width's own statistics) against the
    oracle: dense plane bit for bit, candidates under the north_star tolerances."""
    case = dict(case)
    wdec, sm, nbits = case.pop("wdec", 0), case.pop("sigma_mode", 0), case.pop("nbits", 8)
    w = I.scaled(_tiny(**case), wdec=wdec, sigma_mode=sm, nbits=nbits)
    cands, ref, res = _check_against_oracle(B, w)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0 and res["width_ties"] == 0
    assert len(ref) > 0


def test_measured_sigma_is_accepted_on_every_range(B):
    """Round 2 refused sigma_mode 1 where the cluster kernel does not serve (64-bit boxcar sums, blocks it cannot split):
    cfg4 and 16-bit cfg3 could not run reading A18 at all.  Every such plan is accepted now (no GPU work here: geometry only);
    the results are compared with the oracle in test_search_variants_a18_a20 and the sampled cfg3 / cfg4 tests."""
    assert B.plan_geometry(I.scaled(I.workload(4), sigma_mode=1))["ndms_total"] == I.workload(4).ndms_total
    assert B.plan_geometry(I.scaled(I.workload(3), nbits=16, sigma_mode=1))["ndms_total"] == 2048
    with B.Plan(I.scaled(_tiny(bins=(8,), norm_block=1040, chunk_len=8 * 1040, nsamp=50000), sigma_mode=1)) as plan:   # block of 130 samples
        assert plan.info["n_subchunks"] >= 1


@pytest.mark.parametrize("case", [
    dict(thr=3.0),                                                              # 4 sub-chunks, dense noise candidates: many border records
    dict(thr=3.2, n_streams=3, chunk_len=3 * 2048, nsamp=30000, widths=(1, 2, 4, 8, 64)),
    dict(thr=3.5, bins=(1, 2, 4), nsamp=40000, chunk_len=8192, n_streams=2),   # ranges with different bins: neighbours across a range edge
    dict(thr=3.0, bins=(8,), nsamp=60000, chunk_len=16384, ndms=20, widths=(1, 2, 4, 8, 32)),   # boxcars of 256 raw samples
    dict(thr=4.0, nchans=302, ndms=100, nsamp=21000, chunk_len=4096, foff=-0.5, dm_step=0.25, norm_block=1024, n_streams=2),
    dict(thr=3.0, chunk_len=1024, norm_block=1024, nsamp=9000, widths=(1, 2, 4, 8, 16, 128)),   # boxcars longer than a tenth of a sub-chunk
])
def test_peaks_on_the_device_equal_the_rule_on_the_full_list(B, case):
    """output_mode 1 (reading A17): every sub-chunk's list is thinned on the device, borders are settled on the host;
    the result must be exactly the peak rule applied to the oracle's full candidate list."""
    w = _tiny(**case)
    buf, x = _pinned_fill(B, w)
    with B.Plan(w, peaks=True) as plan:
        got, _ = plan.run(buf, want_taps=False)
        st = plan.stats()
        assert not plan.overflow and plan.info["n_subchunks"] >= 3
    ref, _ = oracle.run(x, w)
    want = oracle.find_peaks_fast(ref)
    assert st["n_candidates"] == len(ref) and st["n_peaks"] == len(got)
    assert 0 < len(want) < len(ref)
    assert got.tobytes() == want.tobytes()
    assert B.find_peaks(ref).tobytes() == want.tobytes()        # the host post-step agrees as well
    with B.Plan(w) as plan:                                      # and fewer bytes crossed the link than in candidate mode
        plan.run(buf, want_taps=False)
        assert st["d2h_bytes"] < plan.stats()["d2h_bytes"]


def test_saturated_16_bit_input(B):
    w = I.scaled(_tiny(nchans=1024, ndms=70, nsamp=9000, chunk_len=4096, f_top=1500.0, foff=-0.2, dm_step=0.25, norm_block=1024), nbits=16)
    buf = B.pinned_empty(w.nbytes)
    buf.numpy()[:] = 255                                 # every sample 65535
    with B.Plan(w, taps=list(range(w.ndms_total))) as plan:
        cands, tap = plan.run(buf)
        assert len(cands) == 0
        assert np.all(tap[:, :plan.nout[0]] == 65535 * w.nchans)


def test_saturated_binned_input(B):
    for variant, b in (("ws1024", 8), ("ws512", 2), ("plain", 4), ("plain", 32), ("ws512", 32), ("ws512", 16),
                       ("auto", 64), ("plain", 64), ("auto", 128), ("auto", 48), ("auto", 96)):
        nb = 2048 if 2048 % b == 0 else 32 * b       # a multiple of the bin and of 16
        w = _tiny(bins=(b,), nchans=1024, ndms=70, nsamp=40000, chunk_len=8 * nb, f_top=1500.0, foff=-0.2, dm_step=0.25,
                  norm_block=nb)
        buf = B.pinned_empty(w.nbytes)
        buf.numpy()[:] = 255                         # every 16-bit lane at its limit before every flush
        with B.Plan(w, taps=list(range(w.ndms_total)), dedisp_variant=variant) as plan:
            cands, tap = plan.run(buf)
            assert len(cands) == 0
            assert np.all(tap[:, :plan.nout[0]] == 255 * w.nchans * b)


def test_saturated_input_every_kernel(B):
    for variant in ("ws1024", "ws512", "sp1024", "plain"):
        w = _tiny(nchans=1024, ndms=70, nsamp=9000, chunk_len=4096, f_top=1500.0, foff=-0.2, dm_step=0.25, norm_block=1024)
        buf = B.pinned_empty(w.nbytes)
        buf.numpy()[:] = 255                         # 16-bit lanes at their limit before every flush
        with B.Plan(w, taps=list(range(w.ndms_total)), dedisp_variant=variant) as plan:
            cands, tap = plan.run(buf)
            assert len(cands) == 0
            assert np.all(tap[:, :plan.nout[0]] == 255 * w.nchans)


def test_cfg1_full(B):
    w = I.workload(1)
    cands, ref, res = _check_against_oracle(B, w)
    top = cands[np.argmax(cands["snr"])]
    assert (top["dm_index"], top["t_start"], top["width"]) == (50, 40000, 8)
    assert np.array_equal(cands, ref) or res["max_rel"] <= 1e-5


def test_stream_and_chunk_invariance(B):
    w = I.scaled(I.workload(2), nsamp=1 << 18, name="cfg2_short")
    buf, x = _pinned_fill(B, w)
    outs = []
    for ns, cl in [(1, 1 << 18), (1, 1 << 16), (2, 1 << 17), (4, 1 << 18), (4, 1 << 19)]:
        cands, tap, _, nout, _ = _run_gpu(B, w, buf, taps=[0, 7, 300, 511], n_streams=ns, chunk_len=cl)
        outs.append((cands.tobytes(), tap.tobytes()))
    assert all(o == outs[0] for o in outs[1:])


def test_pageable_input_through_pinned_staging(B):
    """aa_run_staged (pageable observation, small pinned staging, one copy thread per stream)
    equals the oracle, and returns exactly what aa_run returns on the pinned copy; aa_run itself keeps refusing
    pageable memory."""
    w = _tiny(nchans=64, nsamp=70000, n_streams=3, chunk_len=3 * 4096, ndms=48)
    buf, x = _pinned_fill(B, w)
    taps = list(range(w.ndms_total))
    ref, dense, geo = oracle.run(x, w, keep_dense=True)
    with B.Plan(w, taps=taps) as plan:
        want, want_tap = plan.run(buf)
        with pytest.raises(B.AAError):
            plan.run_staged(np.array(x))                   # plan has no staging buffers
    pageable = np.array(x)                                 # ordinary numpy memory
    with B.Plan(w, taps=taps, stage_input=True) as plan:
        got, got_tap = plan.run_staged(pageable)
        st = plan.stats()
        assert st["h2h_bytes"] == w.nbytes == st["h2d_bytes"]
        with pytest.raises(B.AAError):
            plan.run(pageable)
        again, _ = plan.run(buf)                           # the same plan still takes pinned input directly
    assert np.array_equal(got_tap[:, :geo["nout"][0]], dense[0])            # staged path against the oracle
    res = compare_candidates(got, ref, w.snr_threshold)
    assert res["only_gpu"] == 0 and res["only_oracle"] == 0 and res["width_ties"] == 0 and len(ref) > 0
    assert got.tobytes() == want.tobytes() == again.tobytes() and len(want) > 0
    assert np.array_equal(got_tap, want_tap)


def test_time_sharded_observation_equals_the_whole(B):
    """one observation split by time over several GPUs (here: the shards one after the other on one
    GPU, through the same dist_util code the ranks use) gives the single-run candidate list, bit for bit."""
    from paper_2101_00941_b200 import dist_util
    w = _tiny(nchans=64, nsamp=90000, ndms=48, norm_block=2048, chunk_len=8192, n_streams=2, bins=(1, 2))
    buf, x = _pinned_fill(B, w)
    with B.Plan(w) as plan:
        whole, _ = plan.run(buf, want_taps=False)
        info = plan.info
    ref, _ = oracle.run(x, w)
    tail = info["halo"] - info["maxshift"]
    for world in (2, 3, 5):
        parts = []
        for shard in dist_util.time_shards(w.nsamp, info["maxshift"], w.norm_block, tail, world):
            if shard.nsamp == 0:
                continue
            ws = dist_util.shard_workload(w, shard)
            sbuf = B.pinned_empty(ws.nbytes)
            I.fill_span(w, shard.t_first, shard.nsamp, sbuf.numpy().reshape(shard.nsamp, w.nchans))
            with B.Plan(ws) as plan:
                c, _ = plan.run(sbuf, want_taps=False)
            parts.append(dist_util.merge_shards(c, shard))
        merged = np.concatenate(parts)
        merged = merged[np.lexsort((merged["t_start"], merged["dm_index"]))]
        res = compare_candidates(merged, ref, w.snr_threshold)                 # the merged shards against the oracle
        assert res["only_gpu"] == 0 and res["only_oracle"] == 0 and res["width_ties"] == 0 and len(ref) > 0, world
        assert merged.tobytes() == whole.tobytes() and len(whole) > 0, world


def test_timeline_of_a_streamed_run(B):
    """aa_get_timeline: one entry per sub-chunk, on its own stream, events in pipeline order; dedispersion kernels of
    successive sub-chunks do not overlap (they are ordered across streams)."""
    w = _tiny(nchans=64, nsamp=70000, n_streams=3, chunk_len=3 * 4096, ndms=48)
    buf, _ = _pinned_fill(B, w)
    with B.Plan(w) as plan:
        plan.run(buf, want_taps=False)
        tl = plan.timeline()
        assert len(tl) == plan.info["n_subchunks"] > 6
    for j, t in enumerate(tl):
        assert t["index"] == j and t["stream"] == j % 3
        assert 0 <= t["h2d_begin"] <= t["h2d_end"] <= t["prep_end"] <= t["compute_begin"] <= t["compute_end"] <= t["d2h_end"]
        assert t["dedisp_ms"] > 0 and t["sps_ms"] > 0
    for a, b in zip(tl[:-1], tl[1:]):
        assert b["compute_end"] >= a["compute_end"] - a["sps_ms"] - 1e-3     # sub-chunk order on the device


def test_saturated_input_and_constant_input(B):
    w = _tiny(nchans=300, nsamp=9000, foff=-0.3, dm_step=4.0, chunk_len=4096, norm_block=2048)
    buf = B.pinned_empty(w.nbytes)
    x = buf.numpy().reshape(w.nsamp, w.nchans)
    x[:] = 255                                       # 16-bit lanes at their limit before every flush
    with B.Plan(w, taps=list(range(w.ndms_total))) as plan:
        cands, tap = plan.run(buf)
        assert len(cands) == 0                       # sigma = 0 everywhere
        assert np.all(tap[:, :plan.nout[0]] == 255 * w.nchans)


def test_errors(B):
    w = _tiny()
    x = I.fill(w)                                    # pageable
    with B.Plan(w) as plan:
        with pytest.raises(B.AAError) as e:
            plan.run(x)
        assert e.value.status == B.AA_ERR_NOT_PINNED
    with pytest.raises(B.AAError):
        B.Plan(I.scaled(w, chunk_len=1000))          # not a multiple of norm_block
    with pytest.raises(B.AAError):
        B.Plan(I.scaled(w, widths=(4, 2)))
    # candidate overflow is reported, not fatal
    buf, _ = _pinned_fill(B, I.scaled(w, snr_threshold=1.0))
    with B.Plan(I.scaled(w, snr_threshold=1.0), max_cands_per_subchunk=64) as plan:
        cands, _ = plan.run(buf, max_cands=1 << 20)
        assert plan.overflow and plan.n_found > len(cands)
