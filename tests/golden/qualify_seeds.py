#!/usr/bin/env python
"""Seed qualification (reading G9) -- calls ONLY oracle/ and workloads/.

For every BASELINE config, the gap between the largest and the second-largest oracle power must be
>= 1e-5 * max(P), so that "identical peak index" is a property an fp32 path can always meet.  Full
grids for C1, C2, C4, C4S; for C3, C5, P0 (1e11-1e12 terms) a strided subset plus a dense window of +-256
bins around the injected frequency, which holds the global maximum by construction (pin P7).
Writes tests/golden/seed_qualification.json and, for the batches, the oracle's per-series peaks
(tests/golden/c4_oracle_peaks.json, c4s_oracle_peaks.json: peak index, peak power, top-two gap of all 4,096 series), which
the full-size GPU tests compare bit-exactly.  Run:  python tests/golden/qualify_seeds.py [C1 C2 ...]
"""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import oracle      # noqa: E402
import workloads   # noqa: E402

GAP = 1e-5
STRIDED = 1024          # strided frequencies of the large configs (plus the dense window)


def top_two_gap(P):
    o = np.argsort(P)
    return int(o[-1]), float(P[o[-1]]), float((P[o[-1]] - P[o[-2]]) / P[o[-1]])


def qualify(name):
    w = workloads.make(name)
    if w.B > 1:
        P, idx, val = oracle.periodogram_batched(w.t, w.x, w.f_min, w.df, w.Nf)
        gaps = np.array([top_two_gap(P[b])[2] for b in range(w.B)])
        with open(os.path.join(HERE, "%s_oracle_peaks.json" % name.lower()), "w") as fh:
            json.dump({"config": name, "written_by": "tests/golden/qualify_seeds.py (oracle/ and workloads/ only)",
                       "Nt": w.Nt, "Nf": w.Nf, "series": w.B,
                       "peak_idx": [int(i) for i in idx], "peak_val": [float("%.9g" % v) for v in val],
                       "rel_gap": [float("%.3g" % g) for g in gaps]}, fh, separators=(",", ":"))
        return {"config": name, "series": w.B, "min_rel_gap": float(gaps.min()), "ok": bool(gaps.min() >= GAP),
                "peak_mean": float(val.mean()), "peak_std": float(val.std()), "mean_power": float(P.mean()),
                "coverage": "full grid, every series"}
    if w.terms <= 2e9:
        P = oracle.periodogram(w.t, w.x, w.f_min, w.df, w.Nf)
        ks = np.arange(w.Nf)
        cov = "full grid"
    else:
        c = int(round(w.expected_peak_bin))
        ks = np.unique(np.concatenate([np.arange(0, w.Nf, max(1, w.Nf // STRIDED)), [w.Nf - 1],
                                       np.arange(max(0, c - 256), min(w.Nf, c + 257))]))
        P = oracle.periodogram(w.t, w.x, w.f_min, w.df, w.Nf, ks=ks)
        cov = "%d strided + last bin + dense window of +-256 bins around bin %d" % (STRIDED, c)
    i, pmax, gap = top_two_gap(P)
    return {"config": name, "series": 1, "peak_bin": int(ks[i]), "peak_power": pmax, "min_rel_gap": gap,
            "ok": bool(gap >= GAP), "expected_peak_bin": w.expected_peak_bin, "coverage": cov}


if __name__ == "__main__":
    names = sys.argv[1:] or ["C1", "C2", "C3", "C4", "C4S", "C5", "P0"]
    path = os.path.join(HERE, "seed_qualification.json")
    out = {}
    if os.path.exists(path):
        with open(path) as fh:
            out = json.load(fh)
    for n in names:
        out[n] = qualify(n)
        print(n, out[n], flush=True)
        with open(path, "w") as fh:
            json.dump(out, fh, indent=1, sort_keys=True)
