"""Tolerance-aware comparison of candidate lists (BASELINE.json north_star).

S/N must agree within 1e-5 relative; the sets must be identical except for entries whose S/N is
within 1e-4 of the threshold; where two widths tie within 1e-5 relative either width is accepted.
"""
import numpy as np


def key(c):
    return (c["dm_index"].astype(np.uint64) << np.uint64(32)) | c["t_start"].astype(np.uint64)


def compare_candidates(gpu, ref, thr, *, rtol=1e-5, thr_tol=1e-4):
    """Returns a dict of counts; raises AssertionError with a readable message on a mismatch."""
    kg, kr = key(gpu), key(ref)
    assert np.all(np.diff(kg.astype(np.int64)) > 0), "GPU candidates not sorted / not unique per (dm, t)"
    assert np.all(np.diff(kr.astype(np.int64)) > 0)
    both, ig, ir = np.intersect1d(kg, kr, return_indices=True)
    only_g = np.setdiff1d(np.arange(len(gpu)), ig)
    only_r = np.setdiff1d(np.arange(len(ref)), ir)
    # entries present on one side only must sit at the threshold
    for name, arr, idx in (("gpu", gpu, only_g), ("oracle", ref, only_r)):
        bad = idx[np.abs(arr["snr"][idx].astype(np.float64) - thr) > thr_tol]
        assert bad.size == 0, f"{bad.size} candidates only in {name}, e.g. {arr[bad[:5]]}"
    g, r = gpu[ig], ref[ir]
    rel = np.abs(g["snr"].astype(np.float64) - r["snr"]) / np.maximum(np.abs(r["snr"]), 1e-30)
    assert np.all(rel <= rtol), f"S/N mismatch: max rel {rel.max()} at {g[np.argmax(rel)]} vs {r[np.argmax(rel)]}"
    wdiff = np.nonzero(g["width"] != r["width"])[0]
    # a different width is only acceptable as an arg-max tie: both S/N equal within rtol (already checked)
    return {"common": int(both.size), "only_gpu": int(only_g.size), "only_oracle": int(only_r.size),
            "width_ties": int(wdiff.size), "max_rel": float(rel.max()) if rel.size else 0.0}
