"""Writes tests/golden/oracle_small_cases.json from the FP64 oracle ONLY (never the CUDA path).

    python tests/golden/make_golden.py

The inputs are the seeded generators of paper_2101_06385_b200/workloads.py (which hold none of the method's
arithmetic).  The file freezes the oracle's per-layer decisions on tiny inputs so that an accidental change of the
oracle's arithmetic is caught by tests/test_oracle_pins.py::test_golden_small_cases."""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from oracle import sp2_oracle as O  # noqa: E402
from paper_2101_06385_b200 import workloads as W  # noqa: E402

CASES = [
    ("cfg1_seed0_N16_explicit", lambda: W.config1(0, n=16), "explicit"),
    ("cfg1_seed1_N24_auto", lambda: W.config1(1, n=24), "auto"),
    ("uniform10_nocc5_auto", None, "auto"),          # shape of the paper's Fig. 2 input
    ("uniform100_nocc10_auto", None, "auto"),        # shape of the paper's Fig. 5 input
]


def build():
    out = {}
    for name, mk, mode in CASES:
        if name.startswith("uniform10_"):
            H32, nocc = W.uniform_symmetric(2, 10), 5.0
        elif name.startswith("uniform100_"):
            H32, nocc = W.uniform_symmetric(5, 100), 10.0
        else:
            w = mk()
            H32, nocc = w.H32, w.N_occ
        bounds = (-1.0, 1.0) if mode == "explicit" else None
        D, st = O.sp2_ref(H32, nocc, bounds, tol=1e-9, max_layers=100)
        out[name] = {"n": int(H32.shape[0]), "n_occ": nocc, "bounds_mode": mode,
                     "bounds": [float(b) for b in st["bounds"]], "sigma": [int(s) for s in st["sigma"]],
                     "n_layers": int(st["n_layers"]), "stop_reason": int(st["stop_reason"]),
                     "trace_S": [float(f"{x:.12e}") for x in st["trace_S"]],
                     "trace_D": float(f"{np.trace(D):.12e}"), "D00": float(f"{D[0, 0]:.12e}")}
    return out


if __name__ == "__main__":
    path = os.path.join(HERE, "oracle_small_cases.json")
    with open(path, "w") as f:
        json.dump(build(), f, indent=1, sort_keys=True)
    print("wrote", path)
