"""Seeded synthetic inputs for the streamed dedispersion + single-pulse-search path.

This is the INPUT GENERATOR module: the only code that both the CUDA path's
tests/bench and the CPU oracle's tests use.  It holds none of the method's
arithmetic (no dedispersion, binning, statistics, boxcars or candidate logic):
it describes the five workloads of BASELINE.json (`configs`) and writes seeded
8-bit filterbank buffers.  It imports neither `oracle/` nor the CUDA binding.

Recipe (BASELINE.json configs):
  * layout: time-major ``x[t][c]`` uint8, channel 0 at ``f_top``, ``foff < 0``;
  * noise: ``clip(rint(128 + 16 z), 0, 255)``, z ~ N(0,1), drawn through the
    quantile table of that 8-bit law from a counter-based 32-bit uniform
    ``u(seed, t*nchans + c)`` -- integer-only, so any thread count or device
    reproduces the same bytes;
  * pulses: a boxcar of ``amp`` sigma per channel, ``width`` samples long, whose
    arrival time in channel c follows the cold-plasma dispersion law for the
    pulse's own DM.  Samples under a pulse are re-drawn from the same uniform
    through the table of the shifted mean ``128 + 16*sum(amp)`` ("adds A*16
    counts before rounding/clipping").

These synthetic buffers stand in for the paper's "SKA-like input signal"
(PAPER.md:77), which is not available.
"""
from __future__ import annotations

import ctypes
import dataclasses
import math
import os
import subprocess
from typing import List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libaa_inputs.so")
_lib = None

NOISE_MEAN = 128.0
NOISE_SIGMA = 16.0
#: dispersion constant of the signal model, s MHz^2 / (pc cm^-3)
_K_DISP = 4.148808e3


# ----------------------------------------------------------------------------
# workload descriptions
# ----------------------------------------------------------------------------
@dataclasses.dataclass(frozen=True)
class DMRange:
    dm_low: float
    dm_step: float
    ndms: int
    bin: int = 1


@dataclasses.dataclass(frozen=True)
class Pulse:
    dm: float       # pc cm^-3
    t0: int         # arrival sample in channel 0 (raw samples)
    width: int      # raw samples
    amp: float      # sigma per channel


@dataclasses.dataclass(frozen=True)
class Workload:
    """One row of BASELINE.json `configs` (or a scaled-down test variant)."""
    name: str
    nchans: int
    nsamp: int
    tsamp: float            # seconds
    f_top: float            # MHz, centre of channel 0
    foff: float             # MHz, negative
    ranges: Tuple[DMRange, ...]
    widths: Tuple[int, ...]  # boxcar widths, in binned samples of each range
    snr_threshold: float
    n_streams: int
    chunk_len: int          # raw samples per time chunk
    noise_seed: int
    pulses: Tuple[Pulse, ...]
    norm_block: int = 65536
    nbits: int = 8          # bits per input sample: 8 (BASELINE.json configs), 4 or 16 (reading A19)
    wdec: int = 0           # > 0: widths above it are searched on a coarser time grid (reading A20)
    sigma_mode: int = 0     # 1: S/N from the statistics of each width's own boxcar series (reading A18)

    @property
    def ndms_total(self) -> int:
        return sum(r.ndms for r in self.ranges)

    @property
    def row_bytes(self) -> int:
        return self.nchans * self.nbits // 8

    @property
    def nbytes(self) -> int:
        return self.row_bytes * self.nsamp


def _pow2_upto(n: int) -> Tuple[int, ...]:
    out, w = [], 1
    while w <= n:
        out.append(w)
        w *= 2
    return tuple(out)


def _max_delay_samples(nchans, f_top, foff, tsamp, dm) -> int:
    f_lo = f_top + (nchans - 1) * foff
    return int(math.ceil(_K_DISP * dm * (f_lo ** -2 - f_top ** -2) / tsamp)) + 1


def _draw_pulses(seed: int, n: int, nchans: int, nsamp: int, tsamp: float, f_top: float,
                 foff: float, dm_lo: float, dm_hi: float, dm_plan_max: float,
                 width_choices: Sequence[int], amp_mode: str) -> Tuple[Pulse, ...]:
    """Seeded pulse parameters (SURVEY.md §8(d) 'Synthetic inputs')."""
    rng = np.random.Generator(np.random.PCG64(seed))
    guard = _max_delay_samples(nchans, f_top, foff, tsamp, dm_plan_max) + 64
    out = []
    for _ in range(n):
        dm = float(rng.uniform(dm_lo, dm_hi))
        w = int(width_choices[int(rng.integers(0, len(width_choices)))])
        t0 = int(rng.integers(0, max(1, nsamp - guard - w)))
        if amp_mode == "u1_4":
            amp = float(rng.uniform(1.0, 4.0))
        else:  # target S/N in U[15,60] -> per-channel amplitude
            s_target = float(rng.uniform(15.0, 60.0))
            amp = s_target / math.sqrt(nchans * w)
        out.append(Pulse(dm=dm, t0=t0, width=w, amp=amp))
    return tuple(out)


_SEED0 = 2101_00941_0
_PSEED0 = 2101_00941_100


def workload(k: int) -> Workload:
    """Workload k = 1..5 <-> BASELINE.json configs[k-1]."""
    if k == 1:
        return Workload(
            name="cfg1_tiny", nchans=64, nsamp=131072, tsamp=64e-6, f_top=1500.0, foff=-0.5,
            ranges=(DMRange(0.0, 1.0, 128, 1),), widths=(1, 2, 4, 8, 16, 32), snr_threshold=6.0,
            n_streams=1, chunk_len=131072, noise_seed=_SEED0 + 1,
            pulses=(Pulse(dm=50.0, t0=40000, width=8, amp=3.0),))
    if k == 2:
        nch, ns, ts, ft, fo = 256, 1 << 20, 64e-6, 1500.0, -0.25
        return Workload(
            name="cfg2_small_streamed", nchans=nch, nsamp=ns, tsamp=ts, f_top=ft, foff=fo,
            ranges=(DMRange(0.0, 1.0, 512, 1),), widths=_pow2_upto(128), snr_threshold=6.0,
            n_streams=4, chunk_len=1 << 18, noise_seed=_SEED0 + 2,
            pulses=_draw_pulses(_PSEED0 + 2, 8, nch, ns, ts, ft, fo, 10.0, 500.0, 511.0,
                                tuple(range(1, 65)), "u1_4"))
    if k in (3, 4, 5):
        nch, ts, ft, fo = 4096, 64e-6, 1550.0, -0.0732
        ns = (1 << 24) if k == 5 else (1 << 23)
        if k == 4:
            ranges = (DMRange(0.0, 0.1, 1500, 1), DMRange(150.0, 0.2, 750, 2),
                      DMRange(300.0, 0.25, 800, 4), DMRange(500.0, 0.4, 1000, 8),
                      DMRange(900.0, 0.6, 1000, 16), DMRange(1500.0, 1.0, 1000, 32))
            dm_plan_max = 2499.0
        else:
            ranges = (DMRange(0.0, 1.0, 2048, 1),)
            dm_plan_max = 2047.0
        npulses = 64 if k == 5 else 16
        return Workload(
            name={3: "cfg3_ska_wideband", 4: "cfg4_multirange_binned", 5: "cfg5_out_of_core"}[k],
            nchans=nch, nsamp=ns, tsamp=ts, f_top=ft, foff=fo, ranges=ranges,
            widths=_pow2_upto(256), snr_threshold=7.0, n_streams=8, chunk_len=1 << 20,
            noise_seed=_SEED0 + k,
            pulses=_draw_pulses(_PSEED0 + k, npulses, nch, ns, ts, ft, fo, 50.0, 2000.0,
                                dm_plan_max, _pow2_upto(64), "starget"))
    raise ValueError("workload index must be 1..5")


def scaled(w: Workload, *, nsamp: Optional[int] = None, name: Optional[str] = None,
           **changes) -> Workload:
    """A variant of a workload (shorter observation, other stream split...)."""
    if nsamp is not None:
        guard = max(_max_delay_samples(w.nchans, w.f_top, w.foff, w.tsamp,
                                       r.dm_low + r.dm_step * (r.ndms - 1)) for r in w.ranges)
        pulses = tuple(p for p in w.pulses if p.t0 + p.width + guard + 64 < nsamp)
        changes.setdefault("pulses", pulses)
        changes["nsamp"] = nsamp
    if name is not None:
        changes["name"] = name
    return dataclasses.replace(w, **changes)


# ----------------------------------------------------------------------------
# the generator
# ----------------------------------------------------------------------------
def build(force: bool = False) -> str:
    """Compile gen.c into libaa_inputs.so (gcc, OpenMP)."""
    src = os.path.join(_HERE, "gen.c")
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB_PATH, src])
    return _LIB_PATH


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB_PATH)
        u64, vp = ctypes.c_uint64, ctypes.c_void_p
        lib.aain_uniform32.restype = ctypes.c_uint32
        lib.aain_uniform32.argtypes = [u64, u64]
        lib.aain_fill_noise.restype = None
        lib.aain_fill_noise.argtypes = [vp, u64, u64, u64, vp, vp]
        lib.aain_patch.restype = None
        lib.aain_patch.argtypes = [vp, u64, u64, u64, ctypes.c_int64, ctypes.c_int64, u64, vp]
        _lib = lib
    return _lib


def quantile_table(mean: float, sigma: float = NOISE_SIGMA) -> np.ndarray:
    """32-bit thresholds cdf[v] = floor(2^32 * P(clip(rint(mean + sigma z)) <= v)), v=0..254."""
    out = np.empty(255, dtype=np.uint32)
    for v in range(255):
        p = 0.5 * math.erfc(-((v + 0.5 - mean) / sigma) / math.sqrt(2.0))
        out[v] = min(0xFFFFFFFF, int(math.floor(p * 4294967296.0)))
    return out


def _lut16(cdf: np.ndarray) -> np.ndarray:
    lo = np.searchsorted(cdf, (np.arange(65536, dtype=np.uint64) << np.uint64(16)).astype(np.uint32), side="right")
    hi = np.searchsorted(cdf, ((np.arange(65536, dtype=np.uint64) << np.uint64(16)) + np.uint64(0xFFFF)).astype(np.uint32), side="right")
    lut = np.where(lo == hi, lo, 0xFFFF).astype(np.uint16)
    return lut


def uniform32_numpy(seed: int, idx: np.ndarray) -> np.ndarray:
    """Pure-numpy restatement of the counter-based uniform (cross-check of gen.c)."""
    with np.errstate(over="ignore"):
        z = np.uint64(seed) * np.uint64(0x9E3779B97F4A7C15) + idx.astype(np.uint64)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(32)).astype(np.uint32)


def noise_numpy(seed: int, first: int, n: int, mean: float = NOISE_MEAN) -> np.ndarray:
    """Pure-numpy noise samples for flat indices first..first+n (slow; for checks)."""
    u = uniform32_numpy(seed, np.arange(first, first + n, dtype=np.uint64))
    return np.searchsorted(quantile_table(mean), u, side="right").astype(np.uint8)


def pulse_offsets(w: Workload, dm: float) -> np.ndarray:
    """Arrival-time offset (raw samples) of a pulse of dispersion measure `dm` in each channel.

    Signal model, not the search: cold-plasma law, rounded to the nearest sample.
    """
    f = w.f_top + np.arange(w.nchans, dtype=np.float64) * w.foff
    return np.rint(_K_DISP * dm * (f ** -2.0 - w.f_top ** -2.0) / w.tsamp).astype(np.int64)


def _fill_packed(w: Workload, out: Optional[np.ndarray], t_first: int, n: int) -> np.ndarray:
    """Other bit depths, derived from the seeded 8-bit stream so that the pulses stay where they are:
    4 bits: the 8-bit sample >> 4 (0..15, mean 8), two per byte, even channel in the low nibble;
    16 bits: 256 * (8-bit sample) + a second seeded 8-bit noise stream, little-endian words (mean 32896, sigma 4097)."""
    w8 = dataclasses.replace(w, nbits=8)
    hi = fill_span(w8, t_first, n)
    if out is None:
        out = np.empty((n, w.row_bytes), dtype=np.uint8)
    assert out.dtype == np.uint8 and out.shape == (n, w.row_bytes) and out.flags.c_contiguous
    if w.nbits == 4:
        assert w.nchans % 2 == 0
        np.bitwise_or(hi[:, 0::2] >> 4, hi[:, 1::2] & 0xF0, out=out)
    elif w.nbits == 16:
        lo = fill_span(dataclasses.replace(w8, noise_seed=w.noise_seed + 7777, pulses=()), t_first, n)
        out[:, 0::2] = lo
        out[:, 1::2] = hi
    else:
        raise ValueError("nbits must be 4, 8 or 16")
    return out


def fill(w: Workload, out: Optional[np.ndarray] = None) -> np.ndarray:
    """Write workload `w`'s filterbank into `out` (uint8, shape [nsamp, row_bytes]); returns it.

    `out` may be a view of pinned host memory; it is written in place.
    """
    if w.nbits != 8:
        return _fill_packed(w, out, 0, w.nsamp)
    lib = _load()
    if out is None:
        out = np.empty((w.nsamp, w.nchans), dtype=np.uint8)
    assert out.dtype == np.uint8 and out.shape == (w.nsamp, w.nchans) and out.flags.c_contiguous
    cdf = quantile_table(NOISE_MEAN)
    lut = _lut16(cdf)
    lib.aain_fill_noise(out.ctypes.data, 0, w.nsamp * w.nchans, w.noise_seed,
                        cdf.ctypes.data, lut.ctypes.data)
    _inject(lib, w, out)
    return out


def fill_span(w: Workload, t_first: int, n: int, out: Optional[np.ndarray] = None) -> np.ndarray:
    """Rows [t_first, t_first + n) of workload `w`'s filterbank (what `fill(w)[t_first:t_first+n]` holds) without
    generating the rest: the generator is counter-based, so a rank of a time-sharded run makes only its span."""
    assert 0 <= t_first and t_first + n <= w.nsamp
    if w.nbits != 8:
        return _fill_packed(w, out, t_first, n)
    lib = _load()
    if out is None:
        out = np.empty((n, w.nchans), dtype=np.uint8)
    assert out.dtype == np.uint8 and out.shape == (n, w.nchans) and out.flags.c_contiguous
    cdf = quantile_table(NOISE_MEAN)
    lut = _lut16(cdf)
    lib.aain_fill_noise(out.ctypes.data, t_first * w.nchans, n * w.nchans, w.noise_seed, cdf.ctypes.data, lut.ctypes.data)
    _inject(lib, w, out, t_first, n)
    return out


def _inject(lib, w: Workload, out: np.ndarray, t_first: int = 0, n: Optional[int] = None) -> None:
    """Pulse samples of rows [t_first, t_first + n) (default: the whole observation) re-drawn in `out`."""
    if not w.pulses:
        return
    if n is None:
        n = w.nsamp
    # aain_patch indexes rows by absolute time: hand it the address row 0 would have
    base = out.ctypes.data - t_first * w.nchans
    offs = [pulse_offsets(w, p.dm) for p in w.pulses]
    tables = {}
    for c in range(w.nchans):
        # elementary intervals of this channel's pulse segments, amplitudes added on overlap
        segs = [(p.t0 + int(o[c]), p.t0 + int(o[c]) + p.width, p.amp) for p, o in zip(w.pulses, offs)]
        cuts = sorted({s for s, _, _ in segs} | {e for _, e, _ in segs})
        for a, b in zip(cuts[:-1], cuts[1:]):
            amp = sum(A for s, e, A in segs if s <= a and b <= e)
            if amp == 0.0:
                continue
            tab = tables.get(amp)
            if tab is None:
                tab = tables[amp] = quantile_table(NOISE_MEAN + NOISE_SIGMA * amp)
            a, b = max(a, t_first), min(b, t_first + n)
            if a >= b:
                continue
            lib.aain_patch(base, w.nchans, t_first + n, c, a, b - a, w.noise_seed, tab.ctypes.data)


def sample(w: Workload, t: int, c: int) -> int:
    """The value of x[t][c] of workload `w` without materialising the buffer (spot checks)."""
    amp = 0.0
    for p in w.pulses:
        o = int(pulse_offsets(w, p.dm)[c])
        if p.t0 + o <= t < p.t0 + o + p.width:
            amp += p.amp
    u = uniform32_numpy(w.noise_seed, np.array([t * w.nchans + c], dtype=np.uint64))
    return int(np.searchsorted(quantile_table(NOISE_MEAN + NOISE_SIGMA * amp), u, side="right")[0])
