#!/usr/bin/env python
"""bench.py -- throughput of the streamed dedispersion + single-pulse-search path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 1..5] [--impl ours|reference]

A "step" is one pass of the whole hot path (H2D, corner turn, binning, dedispersion, SPS,
candidate D2H, host merge) over one synthetic observation.  The default workload is the one
BASELINE.json's north_star quotes its targets on, configs[2] (SKA-like 4096 channels x 2^23
samples x 2048 DM trials); the metric is DM-trial*samples/s (plan.dm_trial_samples / time).

  value : inputs already resident in HBM (aa_run_resident), one stream            (`ms_per_step` belongs to it)
  e2e   : aa_run on the pinned HOST buffer, H2D/D2H inside the timed region, n_streams streams: BASELINE.json's
          end-to-end metric, the headline (`e2e.ms_per_step`)
  roofline : dedispersion kernel, CUDA-event duration of each launch (stream of the launch)
  cpu_baseline : the oracle, as it stands, on a bounded sample of the same workload

Prints one JSON line (rank 0).  Under torchrun each rank processes its own observation (weak
scaling, no collective on the data path); the time is the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

# one hardware work queue per stream: with the default of 8 connections the streams of a 8- or 16-stream plan
# share queues and a stream's small D2H copy waits behind another stream's kernels (false dependency)
os.environ.setdefault("CUDA_DEVICE_MAX_CONNECTIONS", "32")

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2101_00941_b200 import inputs as I  # noqa: E402

# BASELINE.json's metric is the end-to-end rate; the bench contract puts the resident-input rate in `value` and the
# end-to-end rate (host buffer, H2D/D2H inside the timed region) in `e2e`: the label says which is which
METRIC = ("DM-trial*samples/s: `value` = observation resident in HBM, `e2e.value` = end to end incl. H2D/D2H "
          "(BASELINE.json's metric); real-time factor; overlap %")
UNIT = "DM-trial*samples/s"
N_SM = 148


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return p, "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


def ncu_profile(kernel_name):
    """Per-launch counters of the dominant kernel from this round's committed `ncu --set full` summary
    (profiles/r2_dedisp_ws_ncu.json, written by `python -m paper_2101_00941_b200.profile_meta`).  The summary names the
    kernel and the sha256 of the kernel sources it was taken from; if either differs from what runs now the counters
    are stale and (None, reason) is returned."""
    from paper_2101_00941_b200 import profile_meta
    path = os.path.join(ROOT, "profiles", "r2_dedisp_ws_ncu.json")
    if not os.path.exists(path):
        return None, "no ncu summary committed for this kernel"
    with open(path) as f:
        p = json.load(f)
    if p.get("kernel") != kernel_name:
        return None, f"summary is for {p.get('kernel')}, the bench ran {kernel_name}"
    if p.get("source_sha256") != profile_meta.kernel_source_hash():
        return None, "kernel sources changed since the summary was taken"
    return p, f"profiles/r2_dedisp_ws_ncu.json (sources {p['source_sha256'][:12]})"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def dist_env():
    from paper_2101_00941_b200 import dist_util
    return dist_util.env()


def pick_workload(k: int, world: int):
    w = I.workload(k)
    note = None
    if world > 1:
        # weak scaling: every rank searches its own observation; keep N pinned copies within host RAM
        try:
            avail = os.sysconf("SC_PHYS_PAGES") * os.sysconf("SC_PAGE_SIZE")
        except (ValueError, OSError):
            avail = 0
        ns = w.nsamp
        while avail and world * w.nchans * ns * 1.15 > 0.8 * avail and ns > (1 << 21):
            ns //= 2
        if ns != w.nsamp:
            w = I.scaled(w, nsamp=ns, name=w.name + f"_nsamp{ns}")
            note = f"observation shortened to {ns} samples per rank to fit {world} pinned copies in host RAM"
    return w, note


def cpu_baseline(w, x, budget_rows=48, budget_blocks=8):
    """The oracle, as it stands, on a bounded sample: `budget_rows` DM trials of range 0 over the first
    `budget_blocks` normalisation blocks (about 10-30 s of CPU work on the 4096-channel workloads)."""
    import oracle
    geo = oracle.geometry(w)
    r = 0
    rg = w.ranges[r]
    rows = sorted(set(np.linspace(0, rg.ndms - 1, budget_rows).astype(int).tolist()))
    L = w.norm_block // rg.bin
    # as many whole blocks as the rows of x that were generated allow
    have = (x.shape[0] - geo["maxshift"]) // rg.bin - (max(w.widths) - 1)
    nblocks = int(max(1, min(budget_blocks, have // L, geo["nout"][r] // L)))
    nemit = min(nblocks * L, geo["nout"][r])
    ntau = min(nemit + max(w.widths) - 1, geo["nout"][r])
    from concurrent.futures import ThreadPoolExecutor
    cores = oracle.num_threads()
    t0 = time.perf_counter()
    D = oracle.dedisperse(x, w, r, rows=rows, tau_first=0, ntau=ntau, geo=geo)         # OpenMP over DM rows
    with ThreadPoolExecutor(max_workers=cores) as ex:                                  # one DM row per host thread
        ncand = sum(ex.map(lambda k: len(oracle.sps_row(D[k], w, r, d_first=0, tau_a=0, tau_b=nemit, nout=geo["nout"][r])[0]),
                           range(len(rows))))
    dt = time.perf_counter() - t0
    units = len(rows) * nemit
    return {"value": units / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{len(rows)} DM trials x {nemit} output samples ({nblocks} normalisation blocks) "
                      f"of {w.name}, dedispersion + SPS, {dt:.1f} s", "seconds": dt}


def run_reference(args):
    rank, world, local = dist_env()
    if rank != 0:
        return 0
    w = I.workload(args.workload)
    # the oracle needs only the rows its sample touches: a short prefix of the observation
    import oracle
    geo_full = oracle.geometry(w)
    need = args.ref_blocks * w.norm_block + max(w.widths) * max(r.bin for r in w.ranges) + geo_full["maxshift"] + 64
    ws = I.scaled(w, nsamp=min(w.nsamp, int(need)), pulses=w.pulses)
    x = I.fill(ws)
    times, val = [], None
    for i in range(args.warmup + args.steps):
        cb = cpu_baseline(ws, x, budget_rows=args.ref_rows, budget_blocks=args.ref_blocks)
        if i >= args.warmup:
            times.append(cb["seconds"]); val = cb
    units = val["value"] * val["seconds"]
    v = units * len(times) / sum(times)
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8->u32 sums, f64 S/N",
            "data": "synthetic", "config": {"workload": w.name, "sample": val["sample"]},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": val["cores"], "kind": "oracle", "sample": val["sample"]},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def run_microbench():
    """The measured denominators: lane-operations per clock per SM of the integer instructions the
    kernels use, shared-memory bytes per clock per SM, pinned host-link GB/s.  profiles/r2_microbench.md is this output."""
    import torch
    from paper_2101_00941_b200 import binding as B
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --microbench needs a CUDA device")
    torch.cuda.set_device(0)
    B.load_library()
    sampler = ClockSampler(0)
    sampler.start()
    res = B.microbench()
    clocks = sampler.stop()
    nsm = torch.cuda.get_device_properties(0).multi_processor_count
    print(json.dumps({"microbench": res, "n_sm": nsm, "clocks": clocks, "gpu": torch.cuda.get_device_name(0),
                      "units": {"arithmetic": "lane-operations per clock per SM (a full-warp instruction = 32)",
                                "shared memory": "bytes per clock per SM, conflict-free accesses",
                                "link": "GB/s, 1 GiB pinned copies, best of 5"}}))
    return 0


def _timed(fn, plan_stats, steps, warmup, barrier, dist_util):
    """W untimed then exactly K timed calls, barrier + synchronize on both sides, CUDA events and wall clock, max over ranks."""
    import torch
    for _ in range(warmup):
        fn()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    t0 = time.perf_counter()
    acc = []
    for _ in range(steps):
        fn()
        acc.append(plan_stats())
    e1.record()
    barrier()
    wall = time.perf_counter() - t0
    dev = e0.elapsed_time(e1) / 1e3
    return dist_util.max_over_ranks(max(wall, dev)), acc


def _host_avail_gb():
    try:
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable:"):
                    return int(line.split()[1]) / 1e6
    except OSError:
        pass
    return 0.0


def _wall(fn):
    """One call, host clock, device idle on both sides."""
    import torch
    torch.cuda.synchronize()
    a = time.perf_counter()
    r = fn()
    torch.cuda.synchronize()
    return time.perf_counter() - a, r


def stream_sweep(B, w, host, obuf, streams, xfer_s, kernels_s, known=None):
    """The stream-count sweep BASELINE.json asks for (configs[2]: 1/2/4/8, configs[4]: 1/2/4/8/16; Fig. 2):
    the time chunk of the workload split into n sub-chunks, one per stream; aa_run from the pinned host buffer, one
    warm-up and one timed call per stream count.  `known` = {n: entry} for a count the caller has already timed.
    overlap_efficiency = max(transfer alone, kernels alone) / wall (north_star), with `kernels_s` = the kernels' own
    CUDA-event durations summed over the resident ONE-stream leg (with several streams a kernel's events also span the
    time it queues behind the other streams' kernels, so the sum of a streamed run is not a kernel time).
    The sorted candidate list must hash identically for every stream count: streams change scheduling, not results."""
    import hashlib
    out = {}
    for n in streams:
        if known and n in known:
            out[str(n)] = known[n]
            continue
        if w.chunk_len % n:
            out[str(n)] = {"skipped": f"chunk_len {w.chunk_len} is not a multiple of {n}"}
            continue
        with B.Plan(w, n_streams=n, chunk_len=w.chunk_len) as plan:
            def one():
                c, _ = plan.run(host, want_taps=False, out=obuf)
                return c
            one()
            dt, c = _wall(one)
            st = plan.stats()
            out[str(n)] = {"ms": 1e3 * dt, "subchunk_len": w.chunk_len // n,
                           "overlap_efficiency": max(kernels_s, xfer_s) / dt, "h2d_gbs_in_run": st["h2d_bytes"] / dt / 1e9,
                           "real_time_factor": w.nsamp * w.tsamp / dt, "candidates": int(len(c)),
                           "candidates_sha256": hashlib.sha256(c.tobytes()).hexdigest()[:16]}
    hashes = {v["candidates_sha256"] for v in out.values() if "candidates_sha256" in v}
    if len(hashes) > 1:
        raise SystemExit(f"stream sweep of {w.name}: candidate lists differ between stream counts: {out}")
    out["transfer_alone_s"] = xfer_s
    out["kernels_alone_s"] = kernels_s
    return out


def paper_path(B, w, host, x, obuf, ref_hash):
    """The paper's own data path, timed on the bench workload (one warm-up, one timed call each):
    staged -- the observation in ordinary PAGEABLE memory, copied by one host thread per stream into small pinned
              buffers and from there to the device (aa_run_staged);
    dense  -- the whole dedispersed DM x time plane returned to pageable host memory through per-stream pinned staging
              and the stream threads (all-rows tap).
    Needs host RAM beside the pinned observation; records {"skipped": reason} when there is not enough."""
    import hashlib
    out = {}
    need = w.nbytes / 1e9 * 1.1
    if _host_avail_gb() < need:
        out["staged"] = {"skipped": f"needs {need:.0f} GB of free host memory for the pageable copy"}
    else:
        pageable = np.array(x)
        with B.Plan(w, stage_input=True) as plan:
            def one():
                c, _ = plan.run_staged(pageable, want_taps=False, out=obuf)
                return c
            one()
            dt, c = _wall(one)
            st = plan.stats()
            h = hashlib.sha256(c.tobytes()).hexdigest()[:16]
            if h != ref_hash:
                raise SystemExit(f"aa_run_staged returned other candidates ({h}) than aa_run ({ref_hash})")
            out["staged"] = {"ms": 1e3 * dt, "n_streams": w.n_streams, "h2h_bytes": st["h2h_bytes"],
                             "h2h_gbs_per_thread": st["h2h_bytes"] / max(st["h2h_ms"], 1e-9) / 1e6,
                             "real_time_factor": w.nsamp * w.tsamp / dt, "candidates_sha256": h}
        del pageable
    g = B.plan_geometry(w)
    dense_gb = w.ndms_total * (g["t_valid"] // min(r.bin for r in w.ranges)) * 4 / 1e9
    if _host_avail_gb() < dense_gb * 1.05:
        out["dense"] = {"skipped": f"needs {dense_gb:.0f} GB of free host memory for the DM x time plane"}
    else:
        with B.Plan(w, taps=list(range(w.ndms_total))) as plan:
            dense = np.zeros((w.ndms_total, plan.info["tap_row_len"]), dtype=np.uint32)

            def one():
                c, _ = plan.run(host, want_taps=False, tap_out=dense, out=obuf)
                return c
            one()                                   # also touches the plane's pages
            dt, c = _wall(one)
            st = plan.stats()
            h = hashlib.sha256(c.tobytes()).hexdigest()[:16]
            if h != ref_hash:
                raise SystemExit(f"the dense run returned other candidates ({h}) than the plain run ({ref_hash})")
            out["dense"] = {"ms": 1e3 * dt, "n_streams": w.n_streams, "d2h_bytes": st["d2h_bytes"],
                            "d2h_gbs_in_run": st["d2h_bytes"] / dt / 1e9, "plane_checksum": int(dense[::97, ::4099].sum()),
                            "real_time_factor": w.nsamp * w.tsamp / dt, "candidates_sha256": h}
        del dense
    return out


def search_variants(B, w, host, obuf):
    """The SURVEY 8(f) variants on the bench workload's own buffer (one warm-up, two timed calls each): per-width measured
    sigma (A18), decimated long boxcars (A20)."""
    out = {}
    for name, ch in (("sigma_mode_1", dict(sigma_mode=1)), ("width_decimation_16", dict(wdec=16))):
        wv = I.scaled(w, name=w.name + "_" + name, **ch)
        try:
            with B.Plan(wv) as plan:
                def one():
                    c, _ = plan.run(host, want_taps=False, out=obuf)
                    return c
                one()
                ts = [_wall(one) for _ in range(2)]
                st = plan.stats()
                out[name] = {"ms": 1e3 * sum(t for t, _ in ts) / 2, "candidates": int(len(ts[-1][1])),
                             "sps_ms": st["sps_ms"], "dedisp_ms": st["dedisp_ms"], "real_time_factor": w.nsamp * w.tsamp * 2 / sum(t for t, _ in ts)}
        except Exception as e:
            out[name] = {"error": f"{type(e).__name__}: {e}"}
    return out


def bit_depth_variants(B, w, obuf):
    """4- and 16-bit input (A19) of the bench workload: own pinned buffer each (17 / 69 GB for cfg3), generated from the
    same seeded stream; one warm-up, two timed calls.  Call with the 8-bit buffer already released."""
    out = {}
    for nbits in (4, 16):
        wv = I.scaled(w, nbits=nbits, name=w.name + f"_{nbits}bit")
        if _host_avail_gb() < wv.nbytes / 1e9 * 1.1:
            out[f"nbits_{nbits}"] = {"skipped": f"needs {wv.nbytes / 1e9:.0f} GB of pinned host memory"}
            continue
        try:
            hv = B.pinned_empty(wv.nbytes)
            I.fill(wv, hv.numpy().reshape(wv.nsamp, wv.row_bytes))
            with B.Plan(wv) as plan:
                def one():
                    c, _ = plan.run(hv, want_taps=False, out=obuf)
                    return c
                one()
                ts = [_wall(one) for _ in range(2)]
                st = plan.stats()
                out[f"nbits_{nbits}"] = {"ms": 1e3 * sum(t for t, _ in ts) / 2, "candidates": int(len(ts[-1][1])),
                                         "h2d_bytes": st["h2d_bytes"], "h2d_gbs_in_run": st["h2d_bytes"] * 2 / sum(t for t, _ in ts) / 1e9,
                                         "dedisp_ms": st["dedisp_ms"], "sps_ms": st["sps_ms"]}
            del hv
        except Exception as e:
            out[f"nbits_{nbits}"] = {"error": f"{type(e).__name__}: {e}"}
    return out


def run_config(B, k, steps, warmup, link_gbs, max_cands=1 << 24, sweep=()):
    """One more BASELINE.json config end to end through aa_run (pinned host buffer, the workload's stream count):
    the `per_config` entries of the bench line.  Own pinned buffer, released before returning."""
    import hashlib
    import torch
    w = I.workload(k)
    t0 = time.perf_counter()
    host = B.pinned_empty(w.nbytes)
    t_pin = time.perf_counter() - t0
    I.fill(w, host.numpy().reshape(w.nsamp, w.row_bytes))
    out = {"workload": w.name, "n_streams": w.n_streams, "pin_s": t_pin}
    L = w.chunk_len // w.n_streams
    last = {}
    obuf = np.zeros(max_cands, dtype=B.CAND_DTYPE)     # the caller's output array: allocated and touched once, outside the timed region

    def leg(plan, fn, nsteps):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        ts, sts = [], []
        for _ in range(nsteps):
            a = time.perf_counter()
            fn()
            torch.cuda.synchronize()
            ts.append(time.perf_counter() - a)
            sts.append(plan.stats())
        return sum(ts) / len(ts), sts[-1]

    with B.Plan(w) as plan:
        def step():
            last["c"], _ = plan.run(host, want_taps=False, out=obuf)
        step_s, st = leg(plan, step, steps)
        last["c"] = last["c"].copy()
        units = plan.info["dm_trial_samples"]
        variants = [plan.dedisp_variant(r) for r in range(len(w.ranges))]
    # the same run with the lists thinned on the device (output_mode 1, reading A17): only peaks cross the link
    with B.Plan(w, peaks=True) as plan:
        def step_pk():
            last["p"], _ = plan.run(host, want_taps=False, out=obuf)
        pk_s, st_pk = leg(plan, step_pk, max(1, steps - 1))
    out["peaks_mode"] = {"ms_per_step": 1e3 * pk_s, "peaks": int(len(last["p"])), "d2h_bytes_per_step": st_pk["d2h_bytes"],
                         "sort_ms": st_pk["sort_ms"], "candidates_mode": {"d2h_bytes_per_step": st["d2h_bytes"], "sort_ms": st["sort_ms"]}}
    # the two things the end-to-end run overlaps, each alone: the copy of the observation, and the kernels on resident data
    dev_in = torch.empty(w.nbytes, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    a = time.perf_counter()
    dev_in.copy_(host, non_blocking=True)
    torch.cuda.synchronize()
    xfer_s = time.perf_counter() - a
    with B.Plan(w, n_streams=1, chunk_len=L) as plan:
        def step_res():
            last["r"], _ = plan.run_resident(dev_in, want_taps=False, out=obuf)
        kern_s, st_res = leg(plan, step_res, max(1, steps - 1))
    del dev_in
    kernels_s = (st_res["dedisp_ms"] + st_res["sps_ms"] + st_res["prep_ms"]) / 1e3
    c = last["c"]
    if sweep:
        known = {w.n_streams: {"ms": 1e3 * step_s, "subchunk_len": L,
                               "overlap_efficiency": max(kernels_s, xfer_s) / step_s, "h2d_gbs_in_run": st["h2d_bytes"] / step_s / 1e9,
                               "real_time_factor": w.nsamp * w.tsamp / step_s, "candidates": int(len(c)),
                               "candidates_sha256": hashlib.sha256(c.tobytes()).hexdigest()[:16]}}
        out["sweep"] = stream_sweep(B, w, host, obuf, sweep, xfer_s, kernels_s, known)
    if len(last["r"]) != len(c):
        raise RuntimeError(f"resident leg found {len(last['r'])} candidates, end-to-end leg {len(c)}")
    out.update({
        "steps": steps, "ms_per_step": 1e3 * step_s,
        "e2e": {"value": units / step_s, "unit": UNIT, "h2d_bytes_per_step": st["h2d_bytes"], "d2h_bytes_per_step": st["d2h_bytes"]},
        "real_time_factor": w.nsamp * w.tsamp / step_s,
        # north_star: wall within 10 % of max(transfer alone, kernels alone); "kernels alone" = the kernels' own CUDA-event
        # durations in the resident one-stream leg, not that leg's wall time (which holds the host output stage as well)
        "transfer_alone_s": xfer_s, "kernels_alone_s": kernels_s, "resident_wall_s": kern_s,
        "host_stage_ms": max(0.0, st_res["wall_ms"] - 1e3 * kernels_s - st_res["d2h_ms"]),
        "overlap_efficiency": max(kernels_s, xfer_s) / step_s,
        # resident leg, one stream: kernel durations from CUDA events on the launching stream, host sort inside the wall time
        "breakdown_ms": {"dedisp": st_res["dedisp_ms"], "sps": st_res["sps_ms"], "prep": st_res["prep_ms"],
                         "d2h": st_res["d2h_ms"], "sort": st_res["sort_ms"], "wall": st_res["wall_ms"]},
        "dedisp_variant": variants,
        "candidates": int(len(c)), "candidates_sha256": hashlib.sha256(c.tobytes()).hexdigest()[:16],
    })
    del host
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--streams", type=int, default=0, help="n_streams of the e2e leg (0: the workload's)")
    ap.add_argument("--ref-rows", type=int, default=48, help="DM trials of the oracle sample")
    ap.add_argument("--ref-blocks", type=int, default=8, help="normalisation blocks of the oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--per-config", default="auto",
                    help="comma-separated other configs to run end to end after the main workload (3 steps each) and "
                         "report under per_config; 'auto' = 1,2,4,5 for the default single-GPU run of workload 3, 'none' = skip")
    ap.add_argument("--extras", default="auto", choices=["auto", "all", "none"],
                    help="stream sweep 1/2/4/8, the paper's data path (aa_run_staged from pageable memory; dense DM x time "
                         "output) and the search variants (A18, A20, 4/16-bit input) on the bench workload, reported under "
                         "`sweep`, `paper_path`, `variants`; 'auto' = all for the default single-GPU run")
    ap.add_argument("--shard-observation", action="store_true",
                    help="strong scaling: ONE observation split by time over the ranks (whole normalisation blocks + halo "
                         "per rank, candidate lists gathered on rank 0); default: one observation per rank (weak)")
    ap.add_argument("--nbits", type=int, default=8, choices=[4, 8, 16],
                    help="bits per input sample (DESIGN.md reading A19); 8 is the BASELINE.json workload")
    ap.add_argument("--nsamp", type=int, default=0,
                    help="shorten the observation (profiling runs under ncu only; not a bench line)")
    ap.add_argument("--microbench", action="store_true",
                    help="measure the integer-ALU, shared-memory and host-link rates the rooflines are quoted against "
                         "(aa_microbench), print them as one JSON line and exit")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.microbench:
        return run_microbench()

    import torch
    from paper_2101_00941_b200 import binding as B

    rank, world, local = dist_env()
    from paper_2101_00941_b200 import dist_util
    affinity0 = os.sched_getaffinity(0) if hasattr(os, "sched_getaffinity") else None
    omp0 = os.environ.get("OMP_NUM_THREADS")
    placement = dist_util.place_rank(local, world)          # NUMA node of the GPU: host threads and first touch
    print(f"[bench] rank {rank}/{world} gpu {local}: {placement}", file=sys.stderr)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dist_util.init("nccl", device=torch.device("cuda", local))
    B.load_library()

    w, note = pick_workload(args.workload, world)
    if args.nsamp:
        w = I.scaled(w, nsamp=args.nsamp, name=w.name + f"_nsamp{args.nsamp}")
        note = "shortened observation for profiling; not a bench line"
    if args.nbits != 8:
        w = I.scaled(w, nbits=args.nbits, name=w.name + f"_{args.nbits}bit")
        note = f"{args.nbits}-bit input derived from the seeded 8-bit stream; not the BASELINE.json workload"
    n_streams = args.streams or w.n_streams
    L = w.chunk_len // w.n_streams                     # sub-chunk length of both legs
    shard = None
    if args.shard_observation:
        # one observation, rank r takes a contiguous run of whole normalisation blocks (+ DM sweep + boxcar tail)
        g = B.plan_geometry(w)
        shard = dist_util.time_shards(w.nsamp, g["maxshift"], w.norm_block, g["halo"] - g["maxshift"], world)[rank]
        if shard.nsamp == 0:
            raise SystemExit(f"rank {rank}: nothing to do ({world} ranks for {w.nsamp} samples)")
        w_full, w = w, dist_util.shard_workload(w, shard)
    else:
        w = dist_util.rank_workload(w, rank)

    # the measured denominators of this run: shared-memory and integer rates per clock and SM, pinned link GB/s
    mb = B.microbench(trips=500, link_bytes=1 << 28)

    t_gen0 = time.perf_counter()
    host = B.pinned_empty(w.nbytes)
    t_pin = time.perf_counter() - t_gen0
    x = host.numpy().reshape(w.nsamp, w.row_bytes)
    if shard is not None:
        I.fill_span(w_full, shard.t_first, shard.nsamp, x)
    else:
        I.fill(w, x)
    t_gen = time.perf_counter() - t_gen0 - t_pin

    def barrier():
        dist_util.barrier()
        torch.cuda.synchronize()

    max_cands = 1 << 24
    obuf = np.zeros(max_cands, dtype=B.CAND_DTYPE)     # output array of every timed call: allocated and touched once
    sampler = ClockSampler(local)

    # ---- leg 1: end to end from pinned host memory -------------------------------------------
    plan = B.Plan(w, n_streams=n_streams, chunk_len=L * n_streams)
    info = plan.info
    units = info["dm_trial_samples"]
    if shard is not None:
        # work units this rank owns: the output samples of its blocks (the tail belongs to the next rank)
        units = dist_util.sum_over_ranks(sum(r.ndms * (shard.keep // r.bin) for r in w.ranges)) // world
    last = {}

    def step_e2e():
        c, _ = plan.run(host, want_taps=False, out=obuf)
        if shard is not None:
            c = dist_util.merge_shards(c, shard)       # gather + sort on rank 0: part of the job
        last["n"] = len(c) if c is not None else 0
        last["c"] = c

    sampler.start()
    t_e2e, st_e2e = _timed(step_e2e, plan.stats, args.steps, args.warmup, barrier, dist_util)
    h2d = st_e2e[-1]["h2d_bytes"]; d2h = st_e2e[-1]["d2h_bytes"]
    launches_e2e = sum(s["dedisp_launches"] + s["sps_launches"] + s["prep_launches"] for s in st_e2e)
    n_cands = last["n"]
    # optional host post-step (outside the timed region): peak finding on the returned list (A17)
    peak_info = None
    if last.get("c") is not None:
        tp0 = time.perf_counter()
        n_peaks = len(B.find_peaks(last["c"]))
        peak_info = {"n": n_peaks, "ms": 1e3 * (time.perf_counter() - tp0), "where": "host threads, after aa_run, not in the timed region"}
    import hashlib
    e2e_hash = hashlib.sha256(last["c"].tobytes()).hexdigest()[:16] if last.get("c") is not None else None
    last.pop("c", None)
    plan.close()

    # ---- leg 2: observation resident in HBM, one stream (kernel-only; per-launch event times) --
    dev_in = torch.empty(w.nbytes, dtype=torch.uint8, device="cuda")
    torch.cuda.synchronize()
    tc0 = time.perf_counter()
    dev_in.copy_(host, non_blocking=True)
    torch.cuda.synchronize()
    t_copy = time.perf_counter() - tc0                 # the transfers alone
    plan = B.Plan(w, n_streams=1, chunk_len=L)
    variant = plan.dedisp_variant(0)
    kernel_name = {0: "dedisp_kernel", 1: "dedisp_sp_kernel<512>", 2: "dedisp_sp_kernel<1024>",
                   3: "dedisp_ws_kernel<512>", 4: "dedisp_ws_kernel<1024>", 5: "dedisp_ws_kernel<512, wide>"}.get(variant, "dedisp")

    def step_res():
        c, _ = plan.run_resident(dev_in, want_taps=False, out=obuf)
        last["n_res"] = len(c)

    t_res, st_res = _timed(step_res, plan.stats, args.steps, args.warmup, barrier, dist_util)
    clocks = sampler.stop()
    plan.close()
    del dev_in
    if shard is None and last["n_res"] != n_cands:
        raise SystemExit(f"resident leg found {last['n_res']} candidates, end-to-end leg {n_cands}")

    # ---- roofline of the dominant kernel (dedispersion) ---------------------------------------
    pk, pk_src = peaks()
    d_ms = sum(s["dedisp_ms"] for s in st_res); d_n = sum(s["dedisp_launches"] for s in st_res)
    s_ms = sum(s["sps_ms"] for s in st_res); p_ms = sum(s["prep_ms"] for s in st_res)
    s_n = sum(s["sps_launches"] for s in st_res)
    wall_ms = sum(s["wall_ms"] for s in st_res)
    avg_launch_s = d_ms / 1e3 / max(d_n, 1)
    sm_mhz = clocks.get("sm_mhz") or pk.get("sm_max_mhz", 1965.0)
    # (a) the binding resource: shared-memory wavefronts the kernel issues by design (aa_plan_dedisp_model over the
    #     plan's real tables) per launch, against the LDS rate measured in this run x the SM clock sampled in this run
    model = B.dedisp_model(w, 0, 4) if variant in (3, 4, 5) and len(w.ranges) == 1 else None
    nblk = -(-w.ranges[0].ndms // 64)
    ncols = L // w.ranges[0].bin + max(w.widths) - 1
    if model:
        wf_cta = model["wf_consumer"] + model["wf_producer_load"] + model["wf_producer_store"] + model["wf_bulk"]
        wf_launch = wf_cta * nblk * -(-ncols // model["tile_samples"])
        lds_b_clk = mb["lds32"]["per_clk_sm"]
        peak_gbs = N_SM * lds_b_clk * sm_mhz * 1e6 / 1e9
        achieved_gbs = wf_launch * 128 / avg_launch_s / 1e9
        prof, prof_src = ncu_profile(kernel_name)
        roofline = {"kernel": kernel_name, "bound": "smem", "achieved": achieved_gbs, "peak": peak_gbs,
                    "unit": "GB/s through shared memory (128-byte wavefronts)", "frac": achieved_gbs / peak_gbs,
                    "traffic": prof["dram_bytes_per_launch"] if prof else None, "traffic_source": prof_src,
                    "peak_source": f"measured in this run: {lds_b_clk:.1f} B/clk/SM (aa_microbench lds32) x {N_SM} SMs x "
                                   f"{sm_mhz:.0f} MHz (median SM clock sampled during the timed region)",
                    "algorithmic": {"wavefronts_per_launch": wf_launch, "per_cta": wf_cta,
                                    "source": "aa_plan_dedisp_model over the plan's tables: consumer row loads + producer window "
                                              "loads + pattern-row stores + bulk-copy landings (profiles/r2_cost_model.md)"},
                    "avg_launch_ms": avg_launch_s * 1e3, "launches": d_n}
        if prof:
            roofline["ncu_wavefronts_per_launch"] = prof["smem_wavefronts_per_launch"]
    else:
        roofline = {"kernel": kernel_name, "bound": "alu", "achieved": None, "peak": None, "unit": "T integer adds/s", "frac": None,
                    "traffic": None, "avg_launch_ms": avg_launch_s * 1e3, "launches": d_n}
    # (b) the algorithmic integer work (nchans adds per DM-trial*sample) against the measured integer rate:
    #     a work rate, not a utilisation -- the shared-pattern scheme performs about a quarter of these adds
    adds_per_step = sum(r.ndms * (info["t_valid"] // r.bin) for r in w.ranges) * w.nchans
    adds_rate = adds_per_step * args.steps / max(d_n, 1) / avg_launch_s / 1e12
    lane_clk = mb["iadd3"]["per_clk_sm"] + mb["imad"]["per_clk_sm"]
    alu_peak = N_SM * lane_clk * sm_mhz * 1e6 / 1e12
    roofline["alu"] = {"achieved": adds_rate, "peak": alu_peak, "unit": "T integer adds/s", "frac": adds_rate / alu_peak,
                       "peak_source": f"measured in this run: {mb['iadd3']['per_clk_sm']:.1f} (ALU pipe) + {mb['imad']['per_clk_sm']:.1f} "
                                      f"(FMA pipe) lane-ops/clk/SM x {N_SM} SMs x {sm_mhz:.0f} MHz",
                       "note": "algorithmic adds (nchans per unit) over time: above 1 is possible because shared pattern rows "
                               "replace four channel adds by one; the binding resource is shared memory (frac above)"}
    if roofline.get("frac") is None:
        roofline.update({"achieved": adds_rate, "peak": alu_peak, "frac": adds_rate / alu_peak})
    roofline["frac_algorithmic_adds"] = adds_rate / alu_peak
    roofline["note"] = ("frac = UTILISATION of the binding unit (shared-memory wavefronts the kernel issues / the measured pipe rate); "
                        "frac_algorithmic_adds = WORK RATE on SURVEY 8(d)'s object (nchans integer adds per DM-trial*sample / the "
                        "measured integer rate): it may exceed 1 because shared pattern rows do a quarter of the counted adds")
    roofline["share_of_step"] = {"dedisp": d_ms / wall_ms, "sps": s_ms / wall_ms, "prep": p_ms / wall_ms}
    # (c) the single-pulse-search kernel: HBM-bound by bytes (4 B read per DM-trial*sample)
    sps_gbs = 4.0 * units * args.steps / (s_ms / 1e3) / 1e9 if s_ms > 0 else 0.0
    roofline["sps_kernel"] = {"bound": "hbm", "achieved": sps_gbs, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": sps_gbs / pk["hbm_gbs"],
                              "avg_launch_ms": s_ms / max(s_n, 1), "peak_source": pk_src}

    if rank == 0:
        value = world * units * args.steps / t_res
        e2e_v = world * units * args.steps / t_e2e
        step_s = t_e2e / args.steps
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t_res / args.steps, "higher_is_better": True,
            "scaling": "strong" if shard is not None else "weak", "vs_baseline": None,
            "dtype": "u8 input, u32 exact sums, f64 S/N", "data": "synthetic",
            "legs": {"value": "observation resident in HBM, 1 stream (aa_run_resident): kernels + D2H of candidates + host merge; "
                              "top-level value and ms_per_step are this leg",
                     "e2e": f"aa_run on the pinned host buffer, {n_streams} streams: H2D and D2H inside the timed region; "
                            "BASELINE.json's end-to-end metric, the headline (e2e.value, e2e.ms_per_step)",
                     "resident": {"value": value, "ms_per_step": 1e3 * t_res / args.steps, "n_streams": 1},
                     "end_to_end": {"value": e2e_v, "ms_per_step": 1e3 * step_s, "n_streams": n_streams}},
            "config": {"workload": w.name, "nchans": w.nchans, "nsamp": w.nsamp, "nbits": w.nbits, "ndms": w.ndms_total,
                       "widths": list(w.widths), "n_streams_e2e": n_streams, "subchunk_len": L,
                       "chunk_len_e2e": L * n_streams, "l2": "inputs (34 GB) >> L2; no flush needed",
                       "note": note},
            "e2e": {"value": e2e_v, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": 1e3 * step_s, "n_streams": n_streams,
                    "real_time_factor": w.nsamp * w.tsamp / step_s,
                    "h2d_gbs_effective": h2d / step_s / 1e9,
                    "transfer_alone_s": t_copy, "kernels_alone_s": (d_ms + s_ms + p_ms) / 1e3 / args.steps,
                    "resident_wall_s": t_res / args.steps,
                    "overlap_efficiency": max(t_copy, (d_ms + s_ms + p_ms) / 1e3 / args.steps) / step_s,
                    "link": {"h2d_gbs": mb["h2d_gbs"], "d2h_gbs": mb["d2h_gbs"], "source": "aa_microbench_link, pinned, this run"}},
            "gpu_launches": int(launches_e2e),
            "candidates": n_cands, "peaks": peak_info, "clocks": clocks, "roofline": roofline,
            "microbench": {k: (v["per_clk_sm"] if isinstance(v, dict) else v) for k, v in mb.items()},
            "setup": {"pin_s": t_pin, "generate_s": t_gen, "placement": placement},
        }
        if not args.no_cpu_baseline:
            # the oracle baseline is quoted on the box's host cores, not on the GPU's NUMA share: undo the placement first
            if world == 1 and affinity0 is not None:
                try:
                    os.sched_setaffinity(0, affinity0)
                    if omp0 is None:
                        os.environ.pop("OMP_NUM_THREADS", None)
                    else:
                        os.environ["OMP_NUM_THREADS"] = omp0
                except OSError:
                    pass
            cb = cpu_baseline(w, x, budget_rows=args.ref_rows, budget_blocks=args.ref_blocks)
            cb.pop("seconds", None)
            line["cpu_baseline"] = cb
    # ---- on the bench workload itself: the stream sweep BASELINE.json asks for, the paper's own data path, the variants ----
    extras = args.extras
    if extras == "auto":
        extras = "all" if (world == 1 and not args.nsamp and not args.shard_observation and args.nbits == 8
                           and args.streams in (0, w.n_streams)) else "none"
    if rank == 0 and extras != "none":
        step_s = t_e2e / args.steps
        kern_alone_s = (d_ms + s_ms + p_ms) / 1e3 / args.steps      # resident one-stream leg: the kernels' own event times
        known = {n_streams: {"ms": 1e3 * step_s, "subchunk_len": L,
                             "overlap_efficiency": max(kern_alone_s, t_copy) / step_s, "h2d_gbs_in_run": h2d / step_s / 1e9,
                             "real_time_factor": w.nsamp * w.tsamp / step_s, "candidates": n_cands, "candidates_sha256": e2e_hash}}
        line["sweep"] = stream_sweep(B, w, host, obuf, [n for n in (1, 2, 4, 8) if w.chunk_len % n == 0], t_copy, kern_alone_s, known)
        try:
            line["paper_path"] = paper_path(B, w, host, x, obuf, e2e_hash)
        except MemoryError as e:
            line["paper_path"] = {"skipped": f"MemoryError: {e}"}
        line["variants"] = search_variants(B, w, host, obuf)
    del host, x
    if rank == 0 and extras != "none":
        line["variants"].update(bit_depth_variants(B, w, obuf))
    # ---- the other configs of BASELINE.json, end to end (north_star: "the 4096-channel configs") ----
    pcs = args.per_config
    if pcs == "auto":
        pcs = "1,2,4,5" if (world == 1 and args.workload == 3 and not args.nsamp and not args.shard_observation
                          and args.nbits == 8) else "none"
    if rank == 0 and pcs != "none":
        line["per_config"] = {}
        for k in [int(v) for v in pcs.split(",") if v]:
            try:
                line["per_config"][f"cfg{k}"] = run_config(B, k, 3, 1, mb["h2d_gbs"], sweep=(1, 2, 4, 8, 16) if k == 5 else ())
            except Exception as e:                      # e.g. not enough host memory to pin 68.7 GB
                line["per_config"][f"cfg{k}"] = {"error": f"{type(e).__name__}: {e}"}
    if rank == 0:
        print(json.dumps(line))
    dist_util.shutdown()
    return 0


if __name__ == "__main__":
    sys.exit(main())
