#!/usr/bin/env python
"""Writes tests/golden/n2_oracle.json: the FULL oracle on the N2-shaped configurations of BASELINE.json that are too slow to
recompute inside a GPU test run (SURVEY.md 8(d) tiers 1 and 3): configs[2] (|S| = 1e5) and the points |S| = 1e4, 3e4 of the
scaling sweep configs[3] at eps2 = 1e-6, 1e-7, 1e-8 (the sweep stands in for the wall-time-versus-|V| chart of PAPER.md:454-456
and Table S7).

This script calls only `oracle/` and `synth_inputs/`; nothing here comes from the CUDA path.  Per case it stores what the GPU
test compares: nnz, a SHA-256 over the CSR structure and the bits of the off-diagonal values (they are bit-exact between the two
sides, reading Q7), E_S, and per eps2 the PT2 sum, the counts, the 16 per-class partial sums (reading Q14) and the conditioning
report.  PT2 runs over ranges of key classes so that the oracle's buckets stay within host memory.

    python tests/golden/make_golden_n2.py [case ...]      # default: every case; existing cases are kept, named ones recomputed

Hours of CPU time in total (the oracle visits every excitation of every source once per class range).
"""
import hashlib
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "n2_oracle.json")

# tag -> (config name, n_dets, eps2 values, key-class ranges per PT2 call)
CASES = {
    "n2sweep_1e4": ("n2sweep", 10_000, (1e-6, 1e-7, 1e-8), 1),
    "n2sweep_3e4": ("n2sweep", 30_000, (1e-6, 1e-7, 1e-8), 2),
    "n2_1e5": ("n2", 100_000, (1e-7,), 4),
}
N_PARTS = 16


def csr_digest(rp, col, val):
    """SHA-256 over row_ptr (int64), col (int32) and the off-diagonal values' bit patterns (little-endian, in CSR order)."""
    nd = len(rp) - 1
    rowid = np.repeat(np.arange(nd), np.diff(rp))
    off = col != rowid
    h = hashlib.sha256()
    h.update(np.ascontiguousarray(rp, dtype="<i8").tobytes())
    h.update(np.ascontiguousarray(col, dtype="<i4").tobytes())
    h.update(np.ascontiguousarray(val[off], dtype="<f8").tobytes())
    return h.hexdigest(), float(np.sum(val[~off]))


def compute(tag):
    import oracle
    from synth_inputs import make_problem
    name, n_dets, eps2s, chunks = CASES[tag]
    p = make_problem(name, n_dets=n_dets)
    t0 = time.time()
    rp, col, val = oracle.ham_build(p["n"], p["h1"], p["eri"], p["e_core"], p["dets"], p["eps"])
    e_s, n2 = oracle.energy(rp, col, val, p["psi"])
    digest, diag_sum = csr_digest(rp, col, val)
    rec = dict(config=name, n_dets=int(len(p["psi"])), eps=p["eps"], nnz=int(len(col)), csr_sha256=digest, diag_sum=diag_sum,
               e_s=e_s, norm2=n2, pt2={}, oracle_threads=oracle.num_threads())
    print(f"{tag}: ham_build + energy {time.time() - t0:.0f} s, nnz {len(col)}", flush=True)
    del rp, col, val
    for eps2 in eps2s:
        t0 = time.time()
        tot = dict(pt2=0.0, n_external=0, n_contrib=0, sum_abs=0.0, min_abs_den=float("inf"), part_sums=np.zeros(N_PARTS))
        for k in range(chunks):
            o = oracle.pt2(p["n"], p["h1"], p["eri"], p["e_core"], p["dets"], p["psi"], e_s, eps2, n_parts=N_PARTS,
                           part_begin=k * N_PARTS // chunks, part_end=(k + 1) * N_PARTS // chunks)
            tot["n_external"] += int(o["n_external"]); tot["n_contrib"] += int(o["n_contrib"])
            tot["sum_abs"] += o["sum_abs"]; tot["min_abs_den"] = min(tot["min_abs_den"], o["min_abs_den"])
            tot["part_sums"] += o["part_sums"]
        tot["part_sums"] = [float(x) for x in tot["part_sums"]]
        tot["pt2"] = float(np.sum(np.array(tot["part_sums"], dtype=np.longdouble)))  # class sums added in class order
        tot["seconds"] = time.time() - t0
        rec["pt2"][repr(eps2)] = tot
        print(f"{tag}: pt2 eps2={eps2:g}: {tot['n_contrib']} contributions, {tot['n_external']} externals, {tot['seconds']:.0f} s", flush=True)
    return rec


if __name__ == "__main__":
    want = sys.argv[1:] or list(CASES)
    for tag in want:
        out = json.load(open(PATH)) if os.path.exists(PATH) else {}
        out[tag] = compute(tag)
        with open(PATH, "w") as f:
            json.dump(out, f, indent=1, sort_keys=True)
            f.write("\n")
        print("wrote", tag, "to", PATH, flush=True)
