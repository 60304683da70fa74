"""Writes tests/golden/trimul_n3.json: a tiny worked example (N=3, c_z=4, c=3, general pair
mask, both directions, with and without the output mask).

The paper (section 3.3) prints NO worked numerical example for this op,
so the stored values are written by this script, which calls only oracle/brute_force.py (the
scalar-loop restatement of Eq. 2-3 + the north_star op), never the CUDA path.
Run:  python tests/golden/make_trimul_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import brute_force  # noqa: E402


def main():
    rng = np.random.default_rng(20260314)
    N, c_z, c = 3, 4, 3
    r = lambda *s: np.round(rng.standard_normal(s), 3)       # 3 decimals: exactly re-readable
    p = {
        "ln_in_gamma": 1 + 0.1 * r(c_z), "ln_in_beta": 0.1 * r(c_z),
        "w_a": r(c, c_z) / 2, "b_a": 0.3 * r(c), "w_a_gate": r(c, c_z) / 2, "b_a_gate": 0.3 * r(c),
        "w_b": r(c, c_z) / 2, "b_b": 0.3 * r(c), "w_b_gate": r(c, c_z) / 2, "b_b_gate": 0.3 * r(c),
        "w_g": r(c_z, c_z) / 2, "b_g": 0.3 * r(c_z),
        "ln_out_gamma": 1 + 0.1 * r(c), "ln_out_beta": 0.1 * r(c),
        "w_o": r(c_z, c) / 2, "b_o": 0.3 * r(c_z),
    }
    z = r(N, N, c_z)
    M = np.array([[1, 1, 0], [1, 1, 1], [0, 1, 1.0]])
    pl = {k: np.asarray(v).tolist() for k, v in p.items()}
    doc = {"cite": "PAPER.md lines 117-130 (Eq. 2-3) + BASELINE.json north_star; values written by "
                   "tests/golden/make_trimul_golden.py from oracle/brute_force.py",
           "N": N, "c_z": c_z, "c_hidden": c, "eps": 1e-5,
           "z": z.tolist(), "mask": M.tolist(), "params": pl, "out": {}}
    for d in (0, 1):
        for mo in (True, False):
            out = brute_force.trimul_brute(z.tolist(), M.tolist(), pl, d, eps=1e-5, mask_output=mo)
            doc["out"][f"dir{d}_maskout{int(mo)}"] = out
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "trimul_n3.json")
    with open(path, "w") as f:
        json.dump(doc, f, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
