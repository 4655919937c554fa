"""Device timeline of one streamed run: the automated stand-in for the paper's visual inspection of the
profiler timeline (Fig. 3-4).

    python -m paper_2101_00941_b200.timeline --workload 3 --streams 8 [--rows 24] [--out FILE.md]

Runs aa_run once (after a warm-up run) and prints, per sub-chunk, when its host-to-device copy, corner turn,
dedispersion + SPS and candidate copy happened (CUDA events on the sub-chunk's stream, aa_get_timeline), then

  copy/compute overlap %  = time the link is busy while kernels of some stream are in flight / time the link is busy
  kernel idle time        = wall time during which no stream had kernels in flight

Needs libaa.so and a CUDA device (no CPU fallback).
"""
from __future__ import annotations

import argparse
import os
import sys


os.environ.setdefault("CUDA_DEVICE_MAX_CONNECTIONS", "32")   # one hardware queue per stream (scheduler)


def _union(intervals):
    out = []
    for a, b in sorted(i for i in intervals if i[1] > i[0]):
        if out and a <= out[-1][1]:
            out[-1][1] = max(out[-1][1], b)
        else:
            out.append([a, b])
    return out


def _length(u):
    return sum(b - a for a, b in u)


def _intersect(u, v):
    i = j = 0
    tot = 0.0
    while i < len(u) and j < len(v):
        a, b = max(u[i][0], v[j][0]), min(u[i][1], v[j][1])
        if b > a:
            tot += b - a
        if u[i][1] < v[j][1]:
            i += 1
        else:
            j += 1
    return tot


def summarise(tl, wall_ms):
    copies = _union([(t["h2d_begin"], t["h2d_end"]) for t in tl])
    kernels = _union([(t["h2d_end"], t["prep_end"]) for t in tl] + [(t["compute_begin"], t["compute_end"]) for t in tl])
    link = _length(copies)
    return {"link_busy_ms": link, "kernels_in_flight_ms": _length(kernels),
            "overlap_pct": 100.0 * _intersect(copies, kernels) / link if link else float("nan"),
            "kernel_idle_ms": wall_ms - _length(kernels)}


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--workload", type=int, default=3)
    ap.add_argument("--streams", type=int, default=0, help="0: the workload's")
    ap.add_argument("--nsamp", type=int, default=0)
    ap.add_argument("--rows", type=int, default=24, help="sub-chunks to list")
    ap.add_argument("--out", default="")
    args = ap.parse_args(argv)

    import torch
    from . import binding as B
    from . import inputs as I

    if not torch.cuda.is_available():
        raise SystemExit("timeline needs a CUDA device (no CPU fallback)")
    w = I.workload(args.workload)
    if args.nsamp:
        w = I.scaled(w, nsamp=args.nsamp, name=w.name + f"_nsamp{args.nsamp}")
    n = args.streams or w.n_streams
    host = B.pinned_empty(w.nbytes)
    I.fill(w, host.numpy().reshape(w.nsamp, w.nchans))
    with B.Plan(w, n_streams=n, chunk_len=w.chunk_len) as plan:
        plan.run(host, max_cands=1 << 24, want_taps=False)
        torch.cuda.synchronize()
        cands, _ = plan.run(host, max_cands=1 << 24, want_taps=False)
        st = plan.stats()
        tl = plan.timeline()
    sm = summarise(tl, st["wall_ms"])
    lines = [f"# Device timeline, workload {w.name}, {n} streams, sub-chunks of {w.chunk_len // n} samples",
             "",
             f"Command: `python -m paper_2101_00941_b200.timeline {' '.join(argv if argv is not None else sys.argv[1:])}`  ",
             f"GPU: {torch.cuda.get_device_name(0)}.  aa_run wall time {st['wall_ms']:.1f} ms, {len(cands)} candidates, "
             f"{st['h2d_bytes'] / 1e9:.2f} GB host-to-device.",
             "",
             f"* link busy {sm['link_busy_ms']:.1f} ms ({st['h2d_bytes'] / 1e6 / max(sm['link_busy_ms'], 1e-9):.1f} GB/s while busy); "
             f"kernels in flight {sm['kernels_in_flight_ms']:.1f} ms",
             f"* copy/compute overlap: **{sm['overlap_pct']:.1f} %** of the link-busy time has kernels of some stream in flight",
             f"* wall time with no kernel in flight: {sm['kernel_idle_ms']:.1f} ms "
             f"({100 * sm['kernel_idle_ms'] / st['wall_ms']:.1f} % of the run)",
             "",
             "Times in ms after the start of the run (CUDA events on the sub-chunk's own stream).",
             "",
             "| sub-chunk | stream | H2D begin | H2D end | corner turn end | compute begin | compute end | D2H end | dedisp ms | SPS ms |",
             "|---|---|---|---|---|---|---|---|---|---|"]
    for t in tl[:args.rows]:
        lines.append(f"| {t['index']} | {t['stream']} | {t['h2d_begin']:.1f} | {t['h2d_end']:.1f} | {t['prep_end']:.1f} | "
                     f"{t['compute_begin']:.1f} | {t['compute_end']:.1f} | {t['d2h_end']:.1f} | {t['dedisp_ms']:.2f} | {t['sps_ms']:.2f} |")
    if len(tl) > args.rows:
        lines.append(f"| ... {len(tl) - args.rows} more | | | | | | | | | |")
    text = "\n".join(lines) + "\n"
    print(text)
    if args.out:
        with open(args.out, "w") as f:
            f.write(text)
    return 0


if __name__ == "__main__":
    sys.exit(main())
