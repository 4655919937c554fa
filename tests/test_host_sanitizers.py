"""The host half under sanitizers ("TSan/ASan on host scheduler + oracle").

compute-sanitizer covers device code (and is closed on this pool); the host code has its own hazards: plan-time table
builders that index delay tables, a thread pool in the peak finder, the oracle's C loops.  Three legs, all without a GPU:

  1. the oracle built with gcc -fsanitize=address,undefined, driven by the same Python entry points the pins use, on small
     workloads that reach every C function (all bit depths, both sigma modes, decimated widths, peak finding);
  2. a test-only copy of libaa.so built with nvcc -Xcompiler -fsanitize=address,undefined, host-only entry points:
     aa_plan_geometry and aa_plan_dedisp_model on the five BASELINE.json shapes (delay tables, shared-pattern and
     warp-specialised table builders), aa_find_peaks, the limit checks of aa_find_peaks_device_noalloc;
  3. csrc/peaks.cu built as C++ with -fsanitize=thread and driven by tests/sanitize_peaks.cpp (1 and 8 threads).

Legs 1 and 2 run in a child Python with the sanitizer runtimes preloaded (leak checking off: the interpreter itself
never frees everything).  A sanitizer report fails the test.  What this cannot cover: the stream worker threads of
aa_run, which need a device; their ordering is exercised by the -m gpu parity tests only.
"""
import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2101_00941_b200", "csrc")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
BAD = ("ERROR: AddressSanitizer", "runtime error:", "WARNING: ThreadSanitizer", "ERROR: LeakSanitizer")


def _runtime(name):
    p = subprocess.check_output(["gcc", f"-print-file-name={name}"], text=True).strip()
    if not os.path.isabs(p) or not os.path.exists(p):
        pytest.skip(f"{name} not installed with this gcc")
    return p


def _child(code, preload, extra_env=None):
    env = dict(os.environ, LD_PRELOAD=":".join(preload), ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:halt_on_error=1",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1", PYTHONPATH=ROOT + os.pathsep + os.path.join(ROOT, "tests"),
               OMP_NUM_THREADS="4")
    env.update(extra_env or {})
    r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=900)
    report = r.stdout[-3000:] + r.stderr[-6000:]
    assert not any(b in r.stderr for b in BAD), report
    assert r.returncode == 0, report
    return r.stdout


def test_oracle_under_asan_and_ubsan(tmp_path):
    so = str(tmp_path / "libaa_oracle_san.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-ffp-contract=off", "-fopenmp", "-fsanitize=address,undefined",
                           "-fno-omit-frame-pointer", "-shared", "-fPIC", "-o", so,
                           os.path.join(ROOT, "oracle", "aa_oracle.c"), "-lm"])
    code = f'''
import numpy as np
import oracle
oracle._LIB_PATH = {so!r}; oracle._lib = None
from paper_2101_00941_b200 import inputs as I
def tiny(**kw):
    base = dict(name="san", nchans=24, nsamp=15001, tsamp=64e-6, f_top=1500.0, foff=-4.0,
                ranges=(I.DMRange(0.0, 3.0, 37, 1), I.DMRange(111.0, 3.0, 20, 4)), widths=(1, 2, 4, 8, 32), snr_threshold=4.0,
                n_streams=1, chunk_len=4096, noise_seed=7, pulses=(I.Pulse(dm=40.0, t0=5000, width=4, amp=4.0),), norm_block=1024)
    base.update(kw)
    return I.Workload(**base)
n = 0
for kw in (dict(), dict(nbits=4), dict(nbits=16), dict(sigma_mode=1), dict(wdec=4), dict(sigma_mode=1, wdec=2)):
    w = tiny(**kw)
    x = I.fill(w)
    cands, dense, geo = oracle.run(x, w, keep_dense=True)
    peaks = oracle.find_peaks_fast(cands)
    assert 0 < len(peaks) <= len(cands)
    n += len(cands)
print("oracle ran under the sanitizers:", n, "candidates")
'''
    out = _child(code, [_runtime("libasan.so"), _runtime("libubsan.so")])
    assert "oracle ran under the sanitizers" in out


@pytest.fixture(scope="module")
def libaa_asan(tmp_path_factory):
    d = tmp_path_factory.mktemp("libaa_san")
    flags = ["-O1", "-g", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler",
             "-fPIC,-ffp-contract=off,-pthread,-fsanitize=address,-fsanitize=undefined,-fno-omit-frame-pointer"]
    srcs = sorted(glob.glob(os.path.join(CSRC, "*.cu")))

    def cc(src):
        obj = str(d / (os.path.basename(src)[:-3] + ".o"))
        subprocess.run([NVCC] + flags + ["-c", src, "-o", obj], check=True, capture_output=True)
        return obj
    with ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 1)) as ex:
        objs = list(ex.map(cc, srcs))
    so = str(d / "libaa_san.so")
    subprocess.run([NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler",
                    "-fsanitize=address,-fsanitize=undefined,-pthread", "-o", so] + objs + ["-ldl"], check=True, capture_output=True)
    return so


def test_libaa_host_entry_points_under_asan_and_ubsan(libaa_asan):
    code = f'''
import ctypes
import numpy as np
from paper_2101_00941_b200 import binding as B, inputs as I
B.LIB_PATH = {libaa_asan!r}; B._lib = None
lib = B.load_library()
done = []
for k in (1, 2, 3, 4, 5):
    w = I.workload(k)
    g = B.plan_geometry(w)
    assert g["ndms_total"] == w.ndms_total and g["dm_trial_samples"] > 0
    for r in range(len(w.ranges)):
        m = B.dedisp_model(w, r, 4)
        done.append((k, r, None if m is None else round(m["patterns_mean"], 2)))
for ns in (3, 16, 64):                                     # other stream splits of the headline shape, 4- and 16-bit input
    for nbits in (4, 8, 16):
        B.plan_geometry(I.scaled(I.workload(3), nbits=nbits), n_streams=ns, chunk_len=ns << 17)
# rejected descriptors take the error paths
d = B.PlanDescC()
assert lib.aa_plan_arena_bytes(ctypes.byref(d)) == 0
rng = np.random.default_rng(3)
c = np.zeros(20000, dtype=B.CAND_DTYPE)
c["dm_index"] = rng.integers(0, 50, len(c)); c["t_start"] = rng.integers(0, 30000, len(c))
c["width"] = 2 ** rng.integers(0, 7, len(c)); c["snr"] = np.round(rng.uniform(6, 12, len(c)), 1)
_, first = np.unique(np.stack([c["dm_index"], c["t_start"]]), axis=1, return_index=True)
c = c[np.sort(first)]; c = c[np.lexsort((c["t_start"], c["dm_index"]))]
a, b = B.find_peaks(c, nthreads=1), B.find_peaks(c, nthreads=5)
assert a.tobytes() == b.tobytes() and 0 < len(a) < len(c)
x = ctypes.c_uint32(0)
assert lib.aa_find_peaks_device_noalloc(ctypes.addressof(x), B.PEAKS_NOALLOC_MAX_CANDS + 1, 4, 100, 8, ctypes.addressof(x), 1,
                                        ctypes.addressof(x), None, None) == B.AA_ERR_LIMIT
print("libaa host entry points ran under the sanitizers:", len(done), "ranges modelled")
'''
    out = _child(code, [_runtime("libasan.so"), _runtime("libubsan.so")])
    assert "libaa host entry points ran under the sanitizers" in out


def test_peak_finder_thread_pool_under_tsan(tmp_path):
    exe = str(tmp_path / "sanitize_peaks")
    cuda_inc = os.path.join(os.path.dirname(os.path.dirname(NVCC)), "include")
    subprocess.run(["g++", "-O1", "-g", "-std=c++17", "-fsanitize=thread", "-pthread", f"-I{cuda_inc}", "-x", "c++",
                    os.path.join(CSRC, "peaks.cu"), os.path.join(ROOT, "tests", "sanitize_peaks.cpp"), "-o", exe],
                   check=True, capture_output=True)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=600, env=dict(os.environ, TSAN_OPTIONS="halt_on_error=1"))
    assert not any(b in r.stderr for b in BAD), r.stderr[-6000:]
    assert r.returncode == 0 and r.stdout.count("peaks") == 6, (r.returncode, r.stdout, r.stderr[-2000:])
