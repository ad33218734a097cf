#!/usr/bin/env python
"""Writes tests/golden/config5_gate.json -- the expected values of the config-5 gate (SURVEY.md
8(c), last pin row; Alg. 3).  Calls ONLY oracle/ and the seeded input generators;
nothing here comes from the CUDA path.

    python tests/golden/make_config5_gate.py [--threads T] [--skip-full] [--replica-n 32768]

Part "first_level" (full size, N = 262144, seed 4, dt_top = 2^-7): the oracle's time-steps of the
first hierarchy entry -- |S|, |F| and the histogram of time-step bins.  These are deterministic
functions of the input (one O(N^2) pass of Eq. 49-54: ~7e10 pair evaluations, minutes on 8 cores).

Part "replica" (N = 32768, same recipe, same seed, same dt_top; a full-size oracle step would take
~12 h on 8 cores): one whole oracle HHS-FSI step -- per-level entries / n_slow / n_fast, pair
counts, |dE/E|, |dP|, |dL|/|L| -- and the same step from inputs moved by +-1 ulp per component
(seeded), which shows down to which level the bookkeeping is a reproducible function of the input
(reading 23: eccentric hard binaries sweep their time-step across pivots thousands of
times per top step, and the deepest levels' entry counts then depend on the last bit).

Part "replica_split": the same replica, one whole oracle step with every level split into the connected
components of its fast pairs and the two-body components on their Kepler orbits (
oracle O6s + O6k), again from the inputs as they are and from inputs 1 ulp away.
"""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import frost_inputs as fi  # noqa: E402
import oracle  # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config5_gate.json")
SEED, DT_TOP, ETA = 4, 2.0 ** -7, 0.2


def first_level(n):
    pos, vel, mass, _ = fi.star_cluster(n, SEED)
    t0 = time.time()
    tau, bins = oracle.timesteps(pos, vel, mass, eta_ff=ETA, eta_fb=ETA, tau_pivot=DT_TOP)
    hist = np.bincount(bins[:n]).tolist()
    return {"n": n, "seed": SEED, "dt_top": DT_TOP, "eta": ETA,
            "n_slow": int((tau[:n] >= DT_TOP).sum()), "n_fast": int((tau[:n] < DT_TOP).sum()),
            "bin_histogram": hist, "tau_min": float(tau[:n].min()),
            "oracle_seconds": time.time() - t0}


def conserved(pos, vel, mass):
    d = oracle.diagnostics(pos, vel, mass)
    return d["E"], d["P"], d["L"]


def replica(n, **kw):
    pos, vel, mass, _ = fi.star_cluster(n, SEED)
    e0, p0, l0 = conserved(pos, vel, mass)
    out = {"n": n, "seed": SEED, "dt_top": DT_TOP, "eta": ETA}
    out.update(kw)
    rng = np.random.default_rng(0)
    for name in ("base", "ulp_perturbed"):
        p, v = pos.copy(), vel.copy()
        if name == "ulp_perturbed":
            p = np.ascontiguousarray(np.nextafter(p, rng.choice([-1.0, 1.0], size=p.shape) * np.inf))
            v = np.ascontiguousarray(np.nextafter(v, rng.choice([-1.0, 1.0], size=v.shape) * np.inf))
        t0 = time.time()
        st = oracle.hhs_step(p, v, mass, DT_TOP, eta_ff=ETA, eta_fb=ETA, **kw)
        e1, p1, l1 = conserved(p, v, mass)
        out[name] = {"stats": st, "dE_rel": float(e1 / e0 - 1.0),
                     "dP_max": float(np.abs(p1 - p0).max()),
                     "dL_rel": float(np.linalg.norm(l1 - l0) / np.linalg.norm(l0)),
                     "oracle_seconds": time.time() - t0}
    a, b = out["base"]["stats"], out["ulp_perturbed"]["stats"]
    k = 0
    while k <= min(a["depth"], b["depth"]) and all(a[q][k] == b[q][k] for q in ("entries", "n_slow", "n_fast", "n_comp")):
        k += 1
    out["levels_reproducible_under_1ulp"] = k
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--skip-full", action="store_true")
    ap.add_argument("--full-n", type=int, default=262144)
    ap.add_argument("--replica-n", type=int, default=32768)
    ap.add_argument("--only-split", action="store_true", help="(re)write only the replica_split part")
    args = ap.parse_args()
    if args.threads > 0:
        oracle.set_num_threads(args.threads)
    doc = json.load(open(OUT)) if os.path.exists(OUT) else {}
    doc["generated_by"] = "tests/golden/make_config5_gate.py (oracle/ only)"
    doc["cites"] = "SURVEY.md 8(c) last pin row; Alg. 3 PAPER.md:572-587; Eq. 49-54 PAPER.md:429-474"
    # Part "replica_split": the same replica with every level split into the components of its fast pairs
    # and the two-body components on their Kepler orbits (oracle O6s + O6k; readings 24-25)
    doc["replica_split"] = replica(args.replica_n, split_max=1 << 20, kepler=True)
    json.dump(doc, open(OUT, "w"), indent=1)
    if args.only_split:
        print("wrote", OUT)
        return
    doc["replica"] = replica(args.replica_n)
    json.dump(doc, open(OUT, "w"), indent=1)
    if not args.skip_full:
        doc["first_level"] = first_level(args.full_n)
        json.dump(doc, open(OUT, "w"), indent=1)
    print("wrote", OUT)


if __name__ == "__main__":
    main()
