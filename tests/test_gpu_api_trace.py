"""SURVEY.md T5 / VERDICT r1 item 4: the automated replacement for the paper's "visual inspection of the timeline"
(PAPER.md:45).  A CUPTI runtime-API callback records every CUDA runtime call made while aa_run executes; the property
the paper's recipe is about (PAPER.md:41 step 5, :71: no allocation, no blocking copy, no device-wide wait inside the
streamed phase) is asserted on the list of calls."""
import ctypes
import os
import subprocess

import numpy as np
import pytest

from paper_2101_00941_b200 import inputs as I

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")

# runtime calls that allocate, free, create, or wait for the whole device / block the host on a copy
FORBIDDEN = ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaHostRegister", "cudaHostUnregister", "cudaDeviceSynchronize",
             "cudaStreamCreate", "cudaStreamDestroy", "cudaEventCreate", "cudaEventDestroy", "cudaMemGetInfo",
             "cudaFuncSetAttribute", "cudaDeviceReset")
FORBIDDEN_EXACT = ("cudaMemcpy", "cudaMemcpy2D", "cudaMemset", "cudaMemcpyToSymbol")   # the blocking forms


@pytest.fixture(scope="module")
def tracer(tmp_path_factory):
    so = str(tmp_path_factory.mktemp("cupti") / "libcupti_trace.so")
    inc = [p for p in (f"{CUDA}/include", f"{CUDA}/extras/CUPTI/include") if os.path.isdir(p)]
    lib = [p for p in (f"{CUDA}/lib64", f"{CUDA}/targets/x86_64-linux/lib", f"{CUDA}/extras/CUPTI/lib64")
           if os.path.exists(os.path.join(p, "libcupti.so"))]
    if not lib:
        pytest.skip("libcupti.so not found in the toolkit")
    cmd = ["gcc", "-O1", "-shared", "-fPIC", os.path.join(HERE, "cupti_trace.c"), "-o", so] + [f"-I{p}" for p in inc] + \
          [f"-L{lib[0]}", f"-Wl,-rpath,{lib[0]}", "-lcupti", "-lpthread"]
    subprocess.check_call(cmd)
    t = ctypes.CDLL(so)
    t.trace_begin.restype = ctypes.c_int
    t.trace_end.restype = ctypes.c_int
    t.trace_end.argtypes = [ctypes.c_char_p, ctypes.c_int]
    return t


def _trace(tracer, fn):
    rc = tracer.trace_begin()
    if rc != 0:
        pytest.skip(f"CUPTI callbacks are closed on this box (cuptiSubscribe -> {rc})")
    try:
        fn()
    finally:
        buf = ctypes.create_string_buffer(1 << 16)
        tracer.trace_end(buf, len(buf))
    return {l.split()[0]: int(l.split()[1]) for l in buf.value.decode().splitlines() if l.strip()}


def _assert_clean(calls):
    bad = {k: v for k, v in calls.items() if k.startswith(FORBIDDEN) or k.split("_v")[0] in FORBIDDEN_EXACT}
    assert not bad, f"aa_run made blocking / allocating CUDA calls: {bad} (all calls: {calls})"


@pytest.mark.parametrize("mode", ["pinned", "staged", "resident", "dense"])
def test_no_alloc_no_device_sync_in_run(tracer, mode):
    from paper_2101_00941_b200 import binding as B
    import torch
    w = I.scaled(I.workload(2), nsamp=1 << 18, chunk_len=1 << 16, n_streams=4, norm_block=1 << 14, name="trace")
    host = B.pinned_empty(w.nbytes)
    x = host.numpy().reshape(w.nsamp, w.nchans)
    I.fill(w, x)
    taps = list(range(w.ndms_total)) if mode == "dense" else []
    with B.Plan(w, taps=taps, stage_input=(mode == "staged")) as plan:
        lib = plan.lib
        out = np.empty(1 << 22, dtype=B.CAND_DTYPE)
        n = ctypes.c_uint64(0)
        tap = np.zeros((len(taps), plan.info["tap_row_len"]), dtype=np.uint32) if taps else None
        pageable = np.array(x) if mode == "staged" else None
        dev = torch.empty(w.nbytes, dtype=torch.uint8, device="cuda") if mode == "resident" else None
        if dev is not None:
            dev.copy_(host)
        torch.cuda.synchronize()
        fn, src = {"pinned": (lib.aa_run, host.data_ptr()), "dense": (lib.aa_run, host.data_ptr()),
                   "staged": (lib.aa_run_staged, pageable.ctypes.data if pageable is not None else 0),
                   "resident": (lib.aa_run_resident, dev.data_ptr() if dev is not None else 0)}[mode]
        args = (plan.handle, src, out.ctypes.data, len(out), ctypes.byref(n), tap.ctypes.data if tap is not None else None)
        assert fn(*args) == 0                                   # first run outside the trace: lazy module loading is not aa_run's
        first = int(n.value)
        rc = []
        calls = _trace(tracer, lambda: rc.append(fn(*args)))
        assert rc == [0] and int(n.value) == first > 0
    # the run did go through the CUDA runtime, asynchronously ...
    assert calls.get("cudaLaunchKernel_v7000", 0) + sum(v for k, v in calls.items() if k.startswith("cudaLaunchKernel")) > 0
    if mode != "resident":
        assert any(k.startswith("cudaMemcpyAsync") for k in calls)
    assert any(k.startswith("cudaStreamWaitEvent") for k in calls) and any(k.startswith("cudaStreamSynchronize") for k in calls)
    # ... and never allocated, freed, created, or waited for the whole device
    _assert_clean(calls)


def test_the_tracer_sees_what_it_should_forbid(tracer):
    """Control: an allocation and a device-wide wait made on purpose are seen and rejected."""
    import torch
    from paper_2101_00941_b200 import binding as B
    lib = B.load_library()

    def naughty():
        p = ctypes.c_void_p()
        assert lib.aa_host_alloc(ctypes.byref(p), 4096) == 0     # cudaHostAlloc
        lib.aa_host_free(p)                                      # cudaFreeHost
        torch.cuda.synchronize()                                 # cudaDeviceSynchronize
    calls = _trace(tracer, naughty)
    assert any(k.startswith("cudaHostAlloc") for k in calls) and any(k.startswith("cudaFreeHost") for k in calls)
    with pytest.raises(AssertionError):
        _assert_clean(calls)
