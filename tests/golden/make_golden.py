"""Writes tests/golden/oracle_small.json from oracle/ ONLY (never from the CUDA path).

Run from the repo root:  python tests/golden/make_golden.py
The inputs are the small integer matrices listed in SURVEY.md 8(c) ("TV1-TV4"); the stored values
are regression anchors for the oracle.  The closed-form / hand-derived pins that fix the oracle
itself live in tests/test_oracle_pins.py and cite the paper.
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402

A_TV1 = [[1.0, 2.0], [3.0, 4.0]]
A_TV2 = [[2.0, -1.0, 3.0], [1.0, 4.0, -2.0], [-3.0, 5.0, 1.0]]
A_TV3 = [[[1.0, 2.0], [3.0, 4.0]], [[2.0, -1.0], [1.0, 3.0]]]
S_TV3 = [0.5, -1.0 / 3.0]
A_TV4 = A_TV3 + [[[-1.0, 1.0], [2.0, 1.0]]]
S_TV4 = [0.5, 0.0, -0.5]


def main():
    cases = []
    for name, A, nf in (("TV1_nf2", A_TV1, 2), ("TV1_nf3", A_TV1, 3), ("TV2_nf2", A_TV2, 2), ("TV2_nf3", A_TV2, 3)):
        vals = oracle.o1_all_subsets(np.array([A]), nf, None, sb=False)
        cases.append({"name": name, "mode": "uniform", "n_flavors": nf, "A": [A], "sigma": None,
                      "values_by_bitmask": vals.tolist()})
    for name, A, s in (("TV3_sb2", A_TV3, S_TV3), ("TV4_sb3", A_TV4, S_TV4)):
        vals = oracle.o1_all_subsets(np.array(A), len(A), s, sb=True)
        cases.append({"name": name, "mode": "sb", "n_flavors": len(A), "A": A, "sigma": s,
                      "values_by_bitmask": vals.tolist()})
    out = {"source": "oracle.o1_all_subsets (brute-force definition, PAPER.md Eq. 58-63)",
           "index": "values_by_bitmask[k] is the connected value of subset with bitmask k+1",
           "cases": cases}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_small.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
