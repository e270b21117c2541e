"""Moves a Workload-shaped object (attribute access only: model, x, elem, mol_off, alpha, y, grad) to the
GPU as the tensors the binding takes.  Marshalling only -- no arithmetic of the method."""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np
import torch

from . import Grad, SorfParams


@dataclass
class DeviceProblem:
    params: SorfParams
    x: torch.Tensor
    elem: torch.Tensor
    mol_off: torch.Tensor
    alpha: torch.Tensor
    y: Optional[torch.Tensor]
    grad: Optional[Grad]

    @property
    def n_atoms(self) -> int:
        return int(self.elem.shape[0])

    @property
    def n_mol(self) -> int:
        return int(self.mol_off.shape[0]) - 1


def _t(a, device, pin=False):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if pin:
        t = t.pin_memory()
    return t.to(device, non_blocking=pin)


def host_arrays(w) -> dict:
    """The per-step INPUT arrays of a workload as contiguous numpy arrays (what an end-to-end call uploads)."""
    out = {"x": w.x, "elem": w.elem, "mol_off": w.mol_off}
    if w.y is not None:
        out["y"] = w.y
    if w.grad is not None:
        if w.grad.layout == "dense":
            out["dense"] = w.grad.dense
            out["dense_off"] = w.grad.dense_off
        else:
            out["nbr_idx"] = w.grad.nbr_idx
            out["nbr_val"] = w.grad.nbr_val
    return {k: np.ascontiguousarray(v) for k, v in out.items()}


def device_params(model, device) -> SorfParams:
    return SorfParams(d=model.d, D=model.D, n_transform=model.T, n_elem=model.n_elem, sigma=model.sigma,
                      signs=_t(model.signs, device), bias=_t(model.bias, device))


def device_grad(arrs: dict, device) -> Optional[Grad]:
    if "dense" in arrs:
        return Grad.make_dense(arrs["dense"], arrs["dense_off"])
    if "nbr_idx" in arrs:
        return Grad.make_neighbor(arrs["nbr_idx"], arrs["nbr_val"])
    return None


def device_problem(w, device="cuda:0") -> DeviceProblem:
    arrs = {k: _t(v, device) for k, v in host_arrays(w).items()}
    return DeviceProblem(params=device_params(w.model, device), x=arrs["x"], elem=arrs["elem"],
                         mol_off=arrs["mol_off"], alpha=_t(w.alpha, device), y=arrs.get("y"),
                         grad=device_grad(arrs, device))
