"""Thin ctypes binding of the C-ABI library (include/aa.h): argument marshalling only.

Every step of the path runs in libaa's CUDA kernels.  PyTorch supplies device memory (the plan's
arena is a torch uint8 tensor), streams and pinned host tensors; there is no CPU fallback: if
libaa.so is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libaa.so")

AA_OK, AA_ERR_INVALID, AA_ERR_NOT_PINNED, AA_ERR_OOM, AA_ERR_CUDA, AA_ERR_OVERFLOW = 0, -1, -2, -3, -4, -5
AA_ERR_LIMIT = -6
#: fixed capacity of aa_find_peaks_device_noalloc (aa.h)
PEAKS_NOALLOC_MAX_CANDS, PEAKS_NOALLOC_MAX_CELLS = 1 << 20, 1 << 20
#: aa_dedisp_choice (aa_plan_desc.dedisp_variant)
DEDISP_CHOICE = {"auto": 0, "plain": 1, "sp512": 2, "sp1024": 3, "ws512": 4, "ws1024": 5}

CAND_DTYPE = np.dtype([("dm_index", np.uint32), ("t_start", np.uint32),
                       ("width", np.uint32), ("snr", np.float32)])

EXPORTS = ["aa_plan_arena_bytes", "aa_plan_create", "aa_plan_query", "aa_plan_nout", "aa_plan_delays",
           "aa_plan_dedisp_variant",
           "aa_plan_geometry", "aa_run", "aa_run_staged", "aa_run_resident", "aa_get_stats", "aa_get_timeline", "aa_find_peaks", "aa_find_peaks_device_noalloc", "aa_destroy", "aa_host_alloc", "aa_host_free",
           "aa_strerror", "aa_last_cuda_error",
           "aa_plan_dedisp_model", "aa_microbench_count", "aa_microbench_name", "aa_microbench", "aa_microbench_link"]


class DMRangeC(ctypes.Structure):
    _fields_ = [("dm_low", ctypes.c_double), ("dm_step", ctypes.c_double),
                ("ndms", ctypes.c_int32), ("bin", ctypes.c_int32)]


class PlanDescC(ctypes.Structure):
    _fields_ = [("nchans", ctypes.c_int32), ("nsamp", ctypes.c_uint64), ("tsamp", ctypes.c_double),
                ("f_top", ctypes.c_double), ("foff", ctypes.c_double),
                ("nranges", ctypes.c_int32), ("ranges", ctypes.POINTER(DMRangeC)),
                ("nwidths", ctypes.c_int32), ("widths", ctypes.POINTER(ctypes.c_int32)),
                ("snr_threshold", ctypes.c_double),
                ("n_streams", ctypes.c_int32), ("chunk_len", ctypes.c_uint64), ("norm_block", ctypes.c_uint32),
                ("device_arena", ctypes.c_void_p), ("device_arena_bytes", ctypes.c_uint64),
                ("streams", ctypes.POINTER(ctypes.c_void_p)),
                ("ntap", ctypes.c_int32), ("tap_dm_indices", ctypes.POINTER(ctypes.c_uint32)),
                ("max_cands_per_subchunk", ctypes.c_uint64), ("stage_input", ctypes.c_int32),
                ("dedisp_variant", ctypes.c_int32), ("nbits", ctypes.c_int32),
                ("width_decimation", ctypes.c_int32), ("sigma_mode", ctypes.c_int32), ("output_mode", ctypes.c_int32),
                ("sps_variant", ctypes.c_int32), ("reserved0", ctypes.c_int32)]


class PlanInfoC(ctypes.Structure):
    _fields_ = [(n, ctypes.c_uint64) for n in
                ("maxshift", "t_valid", "halo", "subchunk_len", "n_subchunks", "ndms_total",
                 "dm_trial_samples", "arena_bytes", "pinned_bytes", "tap_row_len")]


class DedispModelC(ctypes.Structure):
    _fields_ = [("group_channels", ctypes.c_int32), ("block_trials", ctypes.c_int32), ("tile_samples", ctypes.c_int32),
                ("stages_per_cta", ctypes.c_int32), ("wf_consumer", ctypes.c_double), ("wf_producer_load", ctypes.c_double),
                ("wf_producer_store", ctypes.c_double), ("wf_bulk", ctypes.c_double), ("patterns_mean", ctypes.c_double),
                ("patterns_max", ctypes.c_int32), ("pad", ctypes.c_int32), ("stage_bytes_mean", ctypes.c_double),
                ("stage_bytes_max", ctypes.c_uint64), ("ring_bytes", ctypes.c_uint64),
                ("shared_offset_fraction", ctypes.c_double)]


class StatsC(ctypes.Structure):
    _fields_ = [("wall_ms", ctypes.c_double), ("sort_ms", ctypes.c_double),
                ("h2d_bytes", ctypes.c_uint64), ("d2h_bytes", ctypes.c_uint64),
                ("h2d_ms", ctypes.c_double), ("d2h_ms", ctypes.c_double), ("prep_ms", ctypes.c_double),
                ("dedisp_ms", ctypes.c_double), ("sps_ms", ctypes.c_double),
                ("dedisp_launches", ctypes.c_uint64), ("sps_launches", ctypes.c_uint64),
                ("prep_launches", ctypes.c_uint64), ("n_candidates", ctypes.c_uint64), ("n_stored", ctypes.c_uint64),
                ("overflow", ctypes.c_int32), ("n_streams", ctypes.c_int32),
                ("h2h_bytes", ctypes.c_uint64), ("h2h_ms", ctypes.c_double), ("n_peaks", ctypes.c_uint64)]


class SubchunkTimesC(ctypes.Structure):
    _fields_ = [("index", ctypes.c_uint32), ("stream", ctypes.c_uint32)] + [(n, ctypes.c_double) for n in
                ("h2d_begin", "h2d_end", "prep_end", "compute_begin", "compute_end", "d2h_end", "dedisp_ms", "sps_ms")]


class AAError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"libaa status {status}: {msg}")
        self.status = status


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libaa.so and declare every symbol of include/aa.h.  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2101_00941_b200.build` "
                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, u64, i32 = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int32
    lib.aa_plan_arena_bytes.restype = u64
    lib.aa_plan_arena_bytes.argtypes = [ctypes.POINTER(PlanDescC)]
    lib.aa_plan_create.restype = ctypes.c_int
    lib.aa_plan_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(PlanDescC)]
    lib.aa_plan_query.restype = ctypes.c_int
    lib.aa_plan_query.argtypes = [vp, ctypes.POINTER(PlanInfoC)]
    lib.aa_plan_nout.restype = u64
    lib.aa_plan_nout.argtypes = [vp, i32]
    lib.aa_plan_delays.restype = ctypes.c_int
    lib.aa_plan_delays.argtypes = [vp, i32, vp]
    lib.aa_plan_dedisp_variant.restype = ctypes.c_int
    lib.aa_plan_dedisp_variant.argtypes = [vp, i32]
    for f in (lib.aa_run, lib.aa_run_staged, lib.aa_run_resident):
        f.restype = ctypes.c_int
        f.argtypes = [vp, vp, vp, u64, ctypes.POINTER(u64), vp]
    lib.aa_get_stats.restype = ctypes.c_int
    lib.aa_get_stats.argtypes = [vp, ctypes.POINTER(StatsC)]
    lib.aa_destroy.restype = None
    lib.aa_destroy.argtypes = [vp]
    lib.aa_plan_geometry.restype = ctypes.c_int
    lib.aa_plan_geometry.argtypes = [ctypes.POINTER(PlanDescC), ctypes.POINTER(PlanInfoC)]
    lib.aa_plan_dedisp_model.restype = ctypes.c_int
    lib.aa_plan_dedisp_model.argtypes = [ctypes.POINTER(PlanDescC), i32, i32, ctypes.POINTER(DedispModelC)]
    lib.aa_find_peaks.restype = ctypes.c_int
    lib.aa_find_peaks.argtypes = [vp, u64, vp, u64, ctypes.POINTER(u64), ctypes.c_int32]
    lib.aa_find_peaks_device_noalloc.restype = ctypes.c_int
    lib.aa_find_peaks_device_noalloc.argtypes = [vp, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32,
                                                 vp, ctypes.c_uint32, vp, vp, ctypes.POINTER(ctypes.c_int)]
    lib.aa_get_timeline.restype = ctypes.c_int
    lib.aa_get_timeline.argtypes = [vp, ctypes.POINTER(SubchunkTimesC), u64, ctypes.POINTER(u64)]
    lib.aa_host_alloc.restype = ctypes.c_int
    lib.aa_host_alloc.argtypes = [ctypes.POINTER(vp), u64]
    lib.aa_host_free.restype = None
    lib.aa_host_free.argtypes = [vp]
    lib.aa_strerror.restype = ctypes.c_char_p
    lib.aa_strerror.argtypes = [ctypes.c_int]
    lib.aa_last_cuda_error.restype = ctypes.c_int
    lib.aa_last_cuda_error.argtypes = []
    lib.aa_microbench_count.restype = ctypes.c_int
    lib.aa_microbench_count.argtypes = []
    lib.aa_microbench_name.restype = ctypes.c_char_p
    lib.aa_microbench_name.argtypes = [ctypes.c_int]
    dp = ctypes.POINTER(ctypes.c_double)
    lib.aa_microbench.restype = ctypes.c_int
    lib.aa_microbench.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp]
    lib.aa_microbench_link.restype = ctypes.c_int
    lib.aa_microbench_link.argtypes = [u64, ctypes.c_int, ctypes.c_int, dp]
    _lib = lib
    return lib


def _check(lib, rc: int, allow_overflow: bool = False) -> int:
    if rc == AA_OK or (allow_overflow and rc == AA_ERR_OVERFLOW):
        return rc
    msg = lib.aa_strerror(rc).decode()
    if rc == AA_ERR_CUDA:
        msg += f" (cudaError {lib.aa_last_cuda_error()})"
    raise AAError(rc, msg)


def pinned_empty(nbytes: int):
    """Pinned host uint8 tensor (torch owns it)."""
    import torch
    return torch.empty(int(nbytes), dtype=torch.uint8, pin_memory=True)


def find_peaks(cands: np.ndarray, nthreads: int = 0) -> np.ndarray:
    """aa_find_peaks on a candidate array sorted by (dm_index, t_start) (what Plan.run returns)."""
    lib = load_library()
    cands = np.ascontiguousarray(cands, dtype=CAND_DTYPE)
    out = np.empty(len(cands), dtype=CAND_DTYPE)
    n = ctypes.c_uint64(0)
    _check(lib, lib.aa_find_peaks(cands.ctypes.data, len(cands), out.ctypes.data, len(out), ctypes.byref(n), int(nthreads)))
    return out[:int(n.value)]


def find_peaks_device_noalloc(cands_dev, ndms: int, t_end: int, wmax: int, out_dev, n_out_dev, stream=None,
                              n: Optional[int] = None) -> None:
    """aa_find_peaks_device_noalloc: peak finding on a device-resident candidate list without any device allocation,
    for callers that must not allocate while they run (a streamed real-time loop that one cudaMalloc would stall, a
    process whose device memory all belongs to a caching pool).  The caller brings everything: `cands_dev` (torch
    uint8/any tensor holding n 16-byte records), `out_dev` (room for the peaks, unordered) and `n_out_dev` (one
    uint32); the scratch is a fixed 8 MiB array inside libaa.so (limits: PEAKS_NOALLOC_MAX_*; AAError(AA_ERR_LIMIT)
    beyond).  Asynchronous on `stream` (a torch stream, default: the current one); calls that could overlap on the
    GPU share that scratch and must be ordered by the caller."""
    import torch
    lib = load_library()
    if n is None:
        n = cands_dev.numel() * cands_dev.element_size() // CAND_DTYPE.itemsize
    max_out = out_dev.numel() * out_dev.element_size() // CAND_DTYPE.itemsize
    st = stream if stream is not None else torch.cuda.current_stream()
    err = ctypes.c_int(0)
    rc = lib.aa_find_peaks_device_noalloc(cands_dev.data_ptr() if n else None, int(n), int(ndms), int(t_end), int(wmax),
                                          out_dev.data_ptr() if max_out else None, int(max_out), n_out_dev.data_ptr(),
                                          st.cuda_stream, ctypes.byref(err))
    if rc != AA_OK:
        raise AAError(rc, lib.aa_strerror(rc).decode() + (f" (cudaError {err.value})" if rc == AA_ERR_CUDA else ""))


def microbench(ctas_per_sm: int = 2, trips: int = 2000, link_bytes: int = 1 << 30) -> dict:
    """aa_microbench / aa_microbench_link: measured rates of the units the hot path is bound by (per SM and clock),
    and the pinned host link.  {name: {"per_clk_sm", "ms", "sm_mhz"}} plus "h2d_gbs" / "d2h_gbs"."""
    lib = load_library()
    out = {}
    for k in range(lib.aa_microbench_count()):
        r, ms, mhz = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
        _check(lib, lib.aa_microbench(k, ctas_per_sm, trips, ctypes.byref(r), ctypes.byref(ms), ctypes.byref(mhz)))
        out[lib.aa_microbench_name(k).decode()] = {"per_clk_sm": r.value, "ms": ms.value, "sm_mhz": mhz.value}
    for d, name in ((0, "h2d_gbs"), (1, "d2h_gbs")):
        g = ctypes.c_double()
        _check(lib, lib.aa_microbench_link(int(link_bytes), 5, d, ctypes.byref(g)))
        out[name] = g.value
    return out


def _desc_for(w, n_streams=None, chunk_len=None):
    ranges = (DMRangeC * len(w.ranges))(*[DMRangeC(r.dm_low, r.dm_step, r.ndms, r.bin) for r in w.ranges])
    widths = (ctypes.c_int32 * len(w.widths))(*w.widths)
    d = PlanDescC()
    d.nchans, d.nsamp, d.tsamp, d.f_top, d.foff = w.nchans, w.nsamp, w.tsamp, w.f_top, w.foff
    d.nranges, d.ranges, d.nwidths, d.widths = len(w.ranges), ranges, len(w.widths), widths
    d.snr_threshold = float(w.snr_threshold)
    d.n_streams = int(n_streams if n_streams is not None else w.n_streams)
    d.chunk_len = int(chunk_len if chunk_len is not None else w.chunk_len)
    d.norm_block = int(getattr(w, "norm_block", 65536))
    d.nbits = int(getattr(w, "nbits", 8))
    d.width_decimation = int(getattr(w, "wdec", 0))
    d.sigma_mode = int(getattr(w, "sigma_mode", 0))
    d._keep = (ranges, widths)
    return d


def dedisp_model(w, r: int, group_channels: int = 4):
    """aa_plan_dedisp_model for range r of workload w: dict of the model's fields, or None if the range does not fit
    that kernel family (no GPU needed)."""
    lib = load_library()
    d = _desc_for(w)
    m = DedispModelC()
    rc = lib.aa_plan_dedisp_model(ctypes.byref(d), int(r), int(group_channels), ctypes.byref(m))
    if rc == AA_ERR_INVALID:
        return None
    _check(lib, rc)
    return {n: getattr(m, n) for n, _ in DedispModelC._fields_ if n != "pad"}


def plan_geometry(w, *, n_streams: Optional[int] = None, chunk_len: Optional[int] = None) -> dict:
    """aa_plan_geometry: maxshift, halo, sub-chunks, work units and memory of the plan for workload `w`, without
    creating it (no GPU needed)."""
    lib = load_library()
    d = _desc_for(w, n_streams, chunk_len)
    info = PlanInfoC()
    _check(lib, lib.aa_plan_geometry(ctypes.byref(d), ctypes.byref(info)))
    return {n: int(getattr(info, n)) for n, _ in PlanInfoC._fields_}


class Plan:
    """aa_plan_create / aa_run / aa_destroy with torch-owned device memory and streams."""

    def __init__(self, w, *, n_streams: Optional[int] = None, chunk_len: Optional[int] = None,
                 taps: Optional[Sequence[int]] = None, max_cands_per_subchunk: int = 0,
                 torch_resources: bool = True, stage_input: bool = False, dedisp_variant="auto", peaks: bool = False,
                 sps_variant: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the path has no CPU fallback")
        self.lib = load_library()
        self.w = w
        self._ranges = (DMRangeC * len(w.ranges))(*[DMRangeC(r.dm_low, r.dm_step, r.ndms, r.bin) for r in w.ranges])
        self._widths = (ctypes.c_int32 * len(w.widths))(*w.widths)
        taps = sorted(int(t) for t in (taps or []))
        self._taps = (ctypes.c_uint32 * max(1, len(taps)))(*taps)
        self.taps = taps
        d = PlanDescC()
        d.nchans, d.nsamp, d.tsamp, d.f_top, d.foff = w.nchans, w.nsamp, w.tsamp, w.f_top, w.foff
        d.nranges, d.ranges = len(w.ranges), self._ranges
        d.nwidths, d.widths = len(w.widths), self._widths
        d.snr_threshold = float(w.snr_threshold)
        d.n_streams = int(n_streams if n_streams is not None else w.n_streams)
        d.chunk_len = int(chunk_len if chunk_len is not None else w.chunk_len)
        d.norm_block = int(getattr(w, "norm_block", 65536))
        d.ntap = len(taps)
        d.tap_dm_indices = self._taps if taps else None
        d.max_cands_per_subchunk = int(max_cands_per_subchunk)
        d.stage_input = 1 if stage_input else 0
        d.dedisp_variant = DEDISP_CHOICE[dedisp_variant] if isinstance(dedisp_variant, str) else int(dedisp_variant)
        d.nbits = int(getattr(w, "nbits", 8))
        d.width_decimation = int(getattr(w, "wdec", 0))
        d.sigma_mode = int(getattr(w, "sigma_mode", 0))
        d.output_mode = 1 if peaks else 0
        d.sps_variant = int(sps_variant)
        self._arena = None
        self._streams = None
        if torch_resources:
            need = self.lib.aa_plan_arena_bytes(ctypes.byref(d))
            if need == 0:
                raise AAError(AA_ERR_INVALID, "invalid plan descriptor")
            self._arena = torch.empty(int(need) + 256, dtype=torch.uint8, device="cuda")
            base = (self._arena.data_ptr() + 255) & ~255
            d.device_arena = base
            d.device_arena_bytes = need
            self._streams = [torch.cuda.Stream() for _ in range(d.n_streams)]
            self._stream_arr = (ctypes.c_void_p * d.n_streams)(*[s.cuda_stream for s in self._streams])
            d.streams = self._stream_arr
        self.desc = d
        self.handle = ctypes.c_void_p()
        _check(self.lib, self.lib.aa_plan_create(ctypes.byref(self.handle), ctypes.byref(d)))
        info = PlanInfoC()
        _check(self.lib, self.lib.aa_plan_query(self.handle, ctypes.byref(info)))
        self.info = {n: int(getattr(info, n)) for n, _ in PlanInfoC._fields_}
        self.nout = [int(self.lib.aa_plan_nout(self.handle, r)) for r in range(len(w.ranges))]
        self.overflow = False

    # ------------------------------------------------------------------
    def delays(self, r: int) -> np.ndarray:
        out = np.empty((self.w.ranges[r].ndms, self.w.nchans), dtype=np.int32)
        _check(self.lib, self.lib.aa_plan_delays(self.handle, r, out.ctypes.data))
        return out

    def dedisp_variant(self, r: int) -> int:
        """0 plain, 1/2 shared-pattern 512/1024, 3/4 warp-specialised shared-pattern 512/1024, 5 the latter with
        32-bit accumulators (coarse time bins)."""
        v = self.lib.aa_plan_dedisp_variant(self.handle, r)
        if v < 0:
            _check(self.lib, v)
        return v

    def _run(self, fn, ptr: int, max_cands: int, want_taps: bool, tap_out=None, out=None):
        # `out`: the caller's candidate array (CAND_DTYPE, C-contiguous), reused across calls; the returned list is then
        # a view of it.  Without it every call makes a fresh np.empty(max_cands): up to 268 MB of new virtual memory
        # whose first touch (page faults) lands inside aa_run's host stage -- fine for tests, not for a timed loop.
        if out is not None:
            assert out.dtype == CAND_DTYPE and out.flags.c_contiguous and out.ndim == 1
            max_cands = len(out)
        else:
            out = np.empty(int(max_cands), dtype=CAND_DTYPE)
        n = ctypes.c_uint64(0)
        tap = None
        if tap_out is not None:                      # caller's buffer (e.g. a 68 GB dense plane, touched once)
            assert tap_out.dtype == np.uint32 and tap_out.flags.c_contiguous
            assert tap_out.shape == (len(self.taps), self.info["tap_row_len"])
            tap = tap_out
        elif want_taps and self.taps:
            tap = np.zeros((len(self.taps), self.info["tap_row_len"]), dtype=np.uint32)
        rc = fn(self.handle, ptr, out.ctypes.data, int(max_cands), ctypes.byref(n),
                tap.ctypes.data if tap is not None else None)
        _check(self.lib, rc, allow_overflow=True)
        self.overflow = rc == AA_ERR_OVERFLOW
        self.n_found = int(n.value)
        return out[:int(self.stats()["n_stored"])], tap

    def run(self, host_input, max_cands: int = 1 << 22, want_taps: bool = True, tap_out=None, out=None):
        """aa_run on a pinned host buffer (torch pinned tensor or its numpy view)."""
        ptr = host_input.data_ptr() if hasattr(host_input, "data_ptr") else host_input.ctypes.data
        return self._run(self.lib.aa_run, ptr, max_cands, want_taps, tap_out, out)

    def run_staged(self, host_input, max_cands: int = 1 << 22, want_taps: bool = True, tap_out=None, out=None):
        """aa_run_staged on an ordinary (pageable) numpy uint8 array; needs Plan(stage_input=True)."""
        ptr = host_input.data_ptr() if hasattr(host_input, "data_ptr") else host_input.ctypes.data
        return self._run(self.lib.aa_run_staged, ptr, max_cands, want_taps, tap_out, out)

    def run_resident(self, device_input, max_cands: int = 1 << 22, want_taps: bool = True, out=None):
        """aa_run_resident on a torch CUDA uint8 tensor holding the whole observation."""
        return self._run(self.lib.aa_run_resident, device_input.data_ptr(), max_cands, want_taps, None, out)

    def stats(self) -> dict:
        s = StatsC()
        _check(self.lib, self.lib.aa_get_stats(self.handle, ctypes.byref(s)))
        return {n: getattr(s, n) for n, _ in StatsC._fields_}

    def timeline(self) -> list:
        """Per-sub-chunk device timeline of the last run (ms after its start), as dicts."""
        n = ctypes.c_uint64(0)
        cap = int(self.info["n_subchunks"])
        arr = (SubchunkTimesC * max(cap, 1))()
        _check(self.lib, self.lib.aa_get_timeline(self.handle, arr, cap, ctypes.byref(n)))
        return [{f: getattr(arr[i], f) for f, _ in SubchunkTimesC._fields_} for i in range(min(cap, int(n.value)))]

    def close(self):
        if getattr(self, "handle", None) is not None and self.handle:
            self.lib.aa_destroy(self.handle)
            self.handle = ctypes.c_void_p()
        self._arena = None
        self._streams = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
