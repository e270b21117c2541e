"""Writes tests/golden/c1_oracle.json and tests/golden/fchl19_oracle.json: a few FP64 values of config 1 and of the
FCHL19 representation of a small seeded molecule computed by `oracle/` ONLY (never by the CUDA path).  A regression guard for the oracle's arithmetic, not a paper-printed
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

    # FCHL19 (eq. 23-33) with the paper's Table I (E + F) parameters on a seeded 7-atom molecule
    from workloads import FchlParams, molecules_geometry
    fp = FchlParams()
    g = molecules_geometry(99, [7])
    rho = oracle.fchl19(fp, g.r, g.elem, g.nbr_idx)
    J = oracle.fchl19_jacobian(fp, g.r, g.elem, g.nbr_idx, atoms=np.array([0]))
    nz = np.nonzero(rho[0])[0]
    out = {
        "source": "oracle/fchl19_oracle.c on workloads.molecules_geometry(99, [7]), Table I (E + F) parameters; PAPER.md eq. 23-33",
        "elements": g.elem.tolist(),
        "rep": int(rho.shape[1]),
        "rho_fro": float(np.linalg.norm(rho)),
        "rho_atom0_first_nonzero_index": int(nz[0]),
        "rho_atom0_first8_nonzero": rho[0, nz[:8]].tolist(),
        "rho_row_sums": rho.sum(1).tolist(),
        "jac_atom0_fro": float(np.linalg.norm(J)),
        "jac_atom0_self_first_nonzero_row": J[0, 0, nz[0]].tolist(),
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "fchl19_oracle.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
