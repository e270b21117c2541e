"""Writes tests/golden/c1_oracle.json: a few FP64 values of config 1 computed by `oracle/` ONLY
(never by the CUDA path).  A regression guard for the oracle's arithmetic, not a paper-printed
value: the paper (arXiv 2206.01580) prints no feature values, seeds or worked SORF example.

    python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import oracle  # noqa: E402
from workloads import make_workload  # noqa: E402


def main():
    w = make_workload("c1")
    Z = oracle.forward_w(w)
    G = oracle.force_rows_w(w)
    E, F = oracle.predict_w(w)
    A = np.concatenate([Z, G]).astype(np.float32)
    ZtZ, Zty = oracle.normal_equations(A, w.y)
    out = {
        "source": "oracle/sorf_oracle.c on workloads.make_workload('c1'); PAPER.md eq. 14-17, 20",
        "Z_0_first8": Z[0, :8].tolist(),
        "Z_fro": float(np.linalg.norm(Z)),
        "energy_first4": E[:4].tolist(),
        "forces_atom0": F[0].tolist(),
        "forces_fro": float(np.linalg.norm(F)),
        "G_fro": float(np.linalg.norm(G)),
        "ZtZ_0_first4": ZtZ[0, :4].tolist(),
        "ZtZ_trace": float(np.trace(ZtZ)),
        "Zty_first4": Zty[:4].tolist(),
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c1_oracle.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
