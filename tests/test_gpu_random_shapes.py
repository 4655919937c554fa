"""GPU parity on seeded random shapes: channels, trials, DM step, band, time bins, normalisation block, streams, width
lists, thresholds, bit depth, the A18 / A20 search variants, both cluster SPS kernels and rows of interference, drawn
from one seeded generator and compared with the oracle element by element (dense plane bit-exact, candidates by
tests/_compare.py).  The fixed cases of test_gpu_parity.py name what they cover; these cover what nobody thought of."""
import random

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


def _draw(rng, it):
    bins = rng.choice([(1,), (1,), (2,), (4,), (1, 2), (8,)])
    nb = max(rng.choice([1024, 2048, 4096, 8192, 16384, 32768, 65536, 131072]), 128 * max(bins))
    n_streams = rng.choice([1, 1, 2, 3])
    nchans = rng.choice([8, 16, 30, 64, 100, 300, 512])
    ndms = rng.choice([5, 17, 40, 64, 70, 130])
    dm_step = rng.choice([0.25, 1.0, 3.0])
    foff = rng.choice([-4.0, -0.5, -0.2])
    widths = rng.choice([(1, 2, 4, 8), (1, 2, 4, 8, 16, 32, 64), (1, 3, 5, 32), (2, 6, 7, 12, 20, 33), (4, 8, 256), (1, 2, 3), (1,),
                         (8, 16, 24), (1, 2, 4, 8, 16, 32, 64, 128, 256)])
    thr = rng.choice([4.0, 5.0, 6.0])
    chunk = nb * rng.choice([1, 1, 2]) * n_streams
    nsamp = rng.randint(chunk + 3000, 3 * chunk + 20000)
    kind = rng.choice([None, None, None, "spikes", "burst", "constant"])
    sps_variant = rng.choice([0, 0, 1])
    nbits = rng.choice([8, 8, 8, 4, 16])
    wdec = rng.choice([0, 0, 0, 2, 8])
    sigma_mode = rng.choice([0, 0, 0, 1])
    if nbits == 4 and nchans % 2:
        nchans += 1
    if nbits != 8:
        kind = None
    ranges, lo = [], 0.0
    for b in bins:
        ranges.append(I.DMRange(lo, dm_step, ndms, b))
        lo += dm_step * ndms
    w = I.Workload(name=f"random{it}", nchans=nchans, nsamp=nsamp, tsamp=64e-6, f_top=1500.0, foff=foff, ranges=tuple(ranges),
                   widths=widths, snr_threshold=thr, n_streams=n_streams, chunk_len=chunk, noise_seed=1000 + it,
                   pulses=(I.Pulse(dm=dm_step * ndms * 0.4, t0=nsamp // 3, width=4, amp=4.0),), norm_block=nb)
    return I.scaled(w, nbits=nbits, wdec=wdec, sigma_mode=sigma_mode), kind, sps_variant


@pytest.mark.parametrize("seed", [2, 3, 4, 5])
def test_random_shapes_match_the_oracle(B, seed):
    rng = random.Random(seed)
    ran = 0
    skipped = []
    for it in range(40):
        w, kind, sps_variant = _draw(rng, it)
        if w.f_top + (w.nchans - 1) * w.foff <= 100.0:
            continue                                   # the band would reach zero frequency
        buf = B.pinned_empty(w.nbytes)
        x = buf.numpy().reshape(w.nsamp, w.row_bytes)
        I.fill(w, x)
        if kind == "spikes":
            x[w.nsamp // 5::997, :] = 255
        elif kind == "burst":
            x[w.nsamp // 3: w.nsamp // 3 + w.nsamp // 8, :] = 250
        elif kind == "constant":
            x[: w.nsamp // 2, :] = 77
        try:
            plan = B.Plan(w, taps=list(range(w.ndms_total)), sps_variant=sps_variant, max_cands_per_subchunk=1 << 23)
        except B.AAError as e:
            # the only expected refusal: a descriptor the plan does not take (sub-chunk shorter than the DM sweep, A18 on
            # a block no cluster takes).  A CUDA error, an allocation failure or anything else is a failure of the test.
            if e.status != B.AA_ERR_INVALID:
                raise
            skipped.append((it, w.name))
            continue
        with plan:
            cands, tap = plan.run(buf, max_cands=1 << 24)
            assert not plan.overflow, (seed, it)
        ref, dense, geo = oracle.run(x, w, keep_dense=True)
        base = 0
        for r, rg in enumerate(w.ranges):
            assert np.array_equal(tap[base:base + rg.ndms, :geo["nout"][r]], dense[r]), (seed, it, r)
            base += rg.ndms
        res = compare_candidates(cands, ref, w.snr_threshold)
        assert res["only_gpu"] == 0 and res["only_oracle"] == 0, (seed, it, res)
        ran += 1
    assert ran >= 25, (ran, skipped)


def _draw_fine(B, rng, it):
    """Fine channels and fine DM steps: the delay tables the shared-pattern dedispersion kernels are built for."""
    bins = rng.choice([(1,), (1,), (2,), (4,), (1, 2, 4), (16,), (32,), (8, 16)])
    nchans = rng.choice([256, 302, 600, 1024, 1029, 2048, 4096])
    f_top = rng.choice([1500.0, 1550.0, 800.0])
    foff = -rng.choice([100.0, 300.0, 200.0]) / nchans
    ndms = rng.choice([33, 64, 70, 128, 200])
    dm_step = rng.choice([0.1, 0.25, 0.5, 1.0])
    nb = max(rng.choice([1024, 4096, 16384]), 128 * max(bins))
    n_streams = rng.choice([1, 2])
    chunk = nb * rng.choice([1, 2, 4]) * n_streams
    variant = rng.choice(["auto", "auto", "ws1024", "ws512", "sp1024", "plain"])
    peaks = rng.choice([False, False, True])
    ranges, lo = [], rng.choice([0.0, 50.0, 300.0])
    for b in bins:
        ranges.append(I.DMRange(lo, dm_step, ndms, b))
        lo += dm_step * ndms
    w = I.Workload(name=f"fine{it}", nchans=nchans, nsamp=10 * chunk + 10 ** 6, tsamp=64e-6, f_top=f_top, foff=foff,
                   ranges=tuple(ranges), widths=(1, 2, 4, 8, 16), snr_threshold=5.0, n_streams=n_streams, chunk_len=chunk,
                   noise_seed=3000 + it, pulses=(), norm_block=nb)
    try:
        g = B.plan_geometry(w)
    except RuntimeError:
        return None
    if g["halo"] > chunk // n_streams:                 # sub-chunks must hold the DM sweep
        chunk = -(-g["halo"] // (nb * n_streams)) * nb * n_streams
    nsamp = chunk + g["maxshift"] + rng.randint(2000, max(chunk, 4000))
    if nsamp * nchans > 3e8:                           # keep the oracle to seconds
        nsamp = max(chunk // n_streams + g["maxshift"] + 1000, int(3e8 // nchans))
    w = I.scaled(w, nsamp=nsamp, chunk_len=chunk, pulses=(I.Pulse(dm=lo * 0.5, t0=nsamp // 4, width=4, amp=2.0),))
    return w, variant, peaks


@pytest.mark.parametrize("seed", [11, 12])
def test_random_fine_channel_shapes_match_the_oracle(B, seed):
    rng = random.Random(seed)
    ran = shared_pattern = 0
    skipped = []
    for it in range(30):
        drawn = _draw_fine(B, rng, it)
        if drawn is None:
            continue
        w, variant, peaks = drawn
        buf = B.pinned_empty(w.nbytes)
        x = buf.numpy().reshape(w.nsamp, w.row_bytes)
        I.fill(w, x)
        try:
            plan = B.Plan(w, taps=list(range(w.ndms_total)), dedisp_variant=variant, peaks=peaks, max_cands_per_subchunk=1 << 22)
        except B.AAError as e:
            if e.status != B.AA_ERR_INVALID:           # only "descriptor not accepted" may skip a draw
                raise
            skipped.append((it, w.name))
            continue
        with plan:
            shared_pattern += any(plan.dedisp_variant(r) in (1, 2, 3, 4, 5) for r in range(len(w.ranges)))
            cands, tap = plan.run(buf, max_cands=1 << 24)
            assert not plan.overflow, (seed, it)
        ref, dense, geo = oracle.run(x, w, keep_dense=True)
        base = 0
        for r, rg in enumerate(w.ranges):
            assert np.array_equal(tap[base:base + rg.ndms, :geo["nout"][r]], dense[r]), (seed, it, r, variant)
            base += rg.ndms
        if peaks:
            assert cands.tobytes() == oracle.find_peaks_fast(ref).tobytes(), (seed, it)
        else:
            res = compare_candidates(cands, ref, w.snr_threshold)
            assert res["only_gpu"] == 0 and res["only_oracle"] == 0, (seed, it, res)
        ran += 1
    assert ran >= 20 and shared_pattern >= 8, (ran, shared_pattern, skipped)
