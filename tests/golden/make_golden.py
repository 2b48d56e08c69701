"""Writes tests/golden/tiny_oracle.txt: the fp64 oracle's outputs on a tiny seeded chunk.

Calls only oracle/ and numpy (the input is drawn here with numpy's seeded generator, not by the product
package).  Run from the repo root:  python -m tests.golden.make_golden
"""
from __future__ import annotations

import os

import numpy as np

from oracle import rfi_oracle as orc

PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_oracle.txt")
M, N_INT, N_TIME, N_CELLS = 4, 8, 16, 3
THRESHOLDS = [[1.0, 0.05, 1.2, 0.8], [0.5, 0.02, 2.0, 0.95]]


def make_input() -> np.ndarray:
    rng = np.random.default_rng(20241219)
    v = rng.normal(size=(N_TIME, N_CELLS, 4, 2)).round(3)
    v[5, 1] += np.array([[6, 0], [0, 6], [0, -6], [6, 0]])        # one strong polarised sample
    v[8:12, 2] = v[8, 2]                                          # one constant window
    return np.ascontiguousarray(v)


def compute() -> dict:
    res = orc.process(make_input(), M, N_INT, np.asarray(THRESHOLDS, np.float64))
    return {"tau": res.tau.reshape(-1), "r_re": res.r_re.reshape(-1), "r_im": res.r_im.reshape(-1),
            "flags": res.flags.astype(np.float64).reshape(-1),
            "avg": np.ascontiguousarray(res.avg).view(np.float64).reshape(-1),
            "weight": res.weight.astype(np.float64).reshape(-1)}


def read(path: str = PATH) -> dict:
    out = {}
    with open(path) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            key, vals = line.split(":", 1)
            out[key.strip()] = np.array([float.fromhex(x) if "0x" in x else float(x) for x in vals.split()])
    return out


def main():
    d = compute()
    with open(PATH, "w") as f:
        f.write("# Written by tests/golden/make_golden.py (calls only oracle/). fp64 oracle outputs, hex floats.\n")
        f.write(f"# input: numpy default_rng(20241219) normal rounded to 3 decimals, [{N_TIME}][{N_CELLS}][4][2]; "
                f"M={M}, n_int={N_INT}, thresholds={THRESHOLDS}\n")
        f.write("# layouts: tau [K][n_win][cells], r_re/r_im [n_win][cells], flags [K][n_win][cells], "
                "avg [K][n_out][cells][4][re,im], weight [K][n_out][cells]\n")
        for key, v in d.items():
            f.write(key + ": " + " ".join(float(x).hex() for x in v) + "\n")
    print("wrote", PATH)


if __name__ == "__main__":
    main()
