#!/usr/bin/env python
"""Writes tests/golden/tiny_oracle.json: regression values of the ORACLE on the Tiny config (BASELINE.json configs[0]).

The paper prints no worked example for this path (no matrix element, connection list or PT2 value; its energies need FCIDUMP
files and trained amplitudes that are not available), so there is no published value to store.  These numbers are written by
this script, which calls only `oracle/` and `synth_inputs/`; they guard the oracle against accidental change (a deliberate
change of its arithmetic must regenerate them and say why in the commit message).  Never produced by the CUDA path.

    python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)


def compute():
    import oracle
    from synth_inputs import make_problem
    out = {}
    for tag, n_dets, eps, eps2 in (("tiny_full", None, 0.0, 0.0), ("tiny_600_screened", 600, 1e-3, 1e-4)):
        p = make_problem("tiny", n_dets=n_dets)
        rp, col, val = oracle.ham_build(p["n"], p["h1"], p["eri"], p["e_core"], p["dets"], eps)
        e, n2 = oracle.energy(rp, col, val, p["psi"])
        r, t_int = oracle.residual(rp, col, val, p["psi"], e)
        pt = oracle.pt2(p["n"], p["h1"], p["eri"], p["e_core"], p["dets"], p["psi"], e, eps2, n_parts=4)
        keys, score, v, haa = oracle.expand(p["n"], p["h1"], p["eri"], p["e_core"], p["dets"], p["psi"], eps2)
        k0, h0, visited = oracle.connections(p["n"], p["h1"], p["eri"], p["e_core"], p["dets"][0], eps)
        out[tag] = dict(n_dets=int(len(p["psi"])), eps=eps, eps2=eps2, nnz=int(len(col)), e_s=e, norm2=n2, internal=t_int,
                        residual_norm=float(np.linalg.norm(r)), e_diag=oracle.ediag(rp, col, val), pt2=pt["pt2"],
                        n_external=int(pt["n_external"]), n_contrib=int(pt["n_contrib"]), part_sums=[float(x) for x in pt["part_sums"]],
                        sum_abs=pt["sum_abs"], expand_size=int(len(keys)), expand_score_sum=float(np.sum(score)),
                        first_key=[int(keys[0, 0]), int(keys[0, 1])], last_key=[int(keys[-1, 0]), int(keys[-1, 1])],
                        row0_connections=int(len(h0)), row0_abs_sum=float(np.sum(np.abs(h0))), row0_visited=int(visited))
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_oracle.json")
    with open(path, "w") as f:
        json.dump(compute(), f, indent=1, sort_keys=True)
        f.write("\n")
    print("wrote", path)
