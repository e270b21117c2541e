"""paper_2206_01580_b200 -- B200 (sm_100a) SORF hot path of QML-Lightning (arXiv 2206.01580).

Thin Python binding over the C-ABI library `libqmll.so` declared in include/qmll.h: argument marshalling
only (torch CUDA tensors -> device pointers, the current torch stream -> cudaStream_t).  Every step of the
path runs in the library's CUDA kernels; there is no CPU or PyTorch fallback, and importing the compute
functions fails loudly if the library is missing.  PyTorch is used for device memory and streams only.

    from paper_2206_01580_b200 import SorfParams, Grad, qmll_sorf_forward, qmll_sorf_backward_forces, \
        qmll_normal_equations, qmll_predict
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqmll.so")

QMLL_GRAD_DENSE, QMLL_GRAD_NEIGHBOR = 1, 2
CALL_FORWARD, CALL_FORWARD_GRAD, CALL_BACKWARD_FORCES, CALL_NORMAL_EQUATIONS, CALL_PREDICT, CALL_SOLVE = range(6)

NE_SPLIT_F16, NE_SPLIT_TF32, NE_SPLIT_F16_PAIRS = 0, 1, 2
ROWS_AUTO, ROWS_FWHT, ROWS_MMA, ROWS_MMA2 = 0, 1, 2, 3

EXPORTS = ("qmll_solve", "qmll_sorf_forward", "qmll_sorf_forward_mode", "qmll_sorf_backward_forces", "qmll_normal_equations",
           "qmll_normal_equations_mode", "qmll_predict", "qmll_workspace_bytes", "qmll_normal_equations_min_workspace",
           "qmll_normal_equations_workspace", "qmll_normal_equations_min_workspace_mode", "qmll_status_string",
           "qmll_launch_count", "qmll_reset_launch_count", "qmll_time_normal_equations_kernel",
           "qmll_collect_normal_equations_kernel_ms", "qmll_microbench", "qmll_microbench_mma", "qmll_pack_lower", "qmll_unpack_lower", "qmll_project",
           "qmll_project_neighbor", "qmll_fchl19", "qmll_fchl19_rep_size", "qmll_sorf_forward_mma", "qmll_rff_forward",
           "qmll_featmap_workspace_bytes", "qmll_sorf_backward_g", "qmll_project_back", "qmll_fchl19_backward",
           "qmll_predict_static", "qmll_predict_static_max_bytes", "qmll_energies")


class _CParams(ctypes.Structure):
    _fields_ = [("d", ctypes.c_int32), ("D", ctypes.c_int32), ("n_transform", ctypes.c_int32),
                ("n_elem", ctypes.c_int32), ("sigma", ctypes.c_float), ("signs", ctypes.c_void_p),
                ("bias", ctypes.c_void_p)]


class _CGrad(ctypes.Structure):
    _fields_ = [("layout", ctypes.c_int32), ("dense", ctypes.c_void_p), ("dense_off", ctypes.c_void_p),
                ("nbr_idx", ctypes.c_void_p), ("nbr_val", ctypes.c_void_p), ("K", ctypes.c_int32),
                ("dense_floats", ctypes.c_int64)]


class _CFchl(ctypes.Structure):
    _fields_ = [("n_elem", ctypes.c_int32), ("n2", ctypes.c_int32), ("n3", ctypes.c_int32), ("eta2", ctypes.c_float),
                ("eta3", ctypes.c_float), ("two_body_decay", ctypes.c_float), ("three_body_decay", ctypes.c_float),
                ("three_body_weight", ctypes.c_float), ("zeta", ctypes.c_float), ("r_cut", ctypes.c_float)]


class QmllError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"qmll status {status}: {text}")
        self.status = status


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libqmll.so (built by paper_2206_01580_b200.build / __graft_entry__.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2206_01580_b200.build` "
                          "(there is no fallback path)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
    pp, gp = ctypes.POINTER(_CParams), ctypes.POINTER(_CGrad)
    lib.qmll_sorf_forward.argtypes = [pp, vp, vp, vp, i64, i32, gp, vp, vp, vp, sz, vp]
    lib.qmll_sorf_forward_mode.argtypes = [pp, vp, vp, vp, i64, i32, gp, vp, vp, vp, sz, i32, vp]
    lib.qmll_sorf_forward_mode.restype = ctypes.c_int
    lib.qmll_sorf_backward_forces.argtypes = [pp, vp, vp, vp, i64, i32, vp, gp, vp, vp, sz, vp]
    lib.qmll_normal_equations.argtypes = [vp, vp, i64, i32, i32, vp, vp, vp, sz, vp]
    lib.qmll_normal_equations_mode.argtypes = [vp, vp, i64, i32, i32, vp, vp, vp, sz, i32, vp]
    lib.qmll_normal_equations_mode.restype = ctypes.c_int
    lib.qmll_normal_equations_workspace.argtypes = [i64, i32, i32]
    lib.qmll_normal_equations_workspace.restype = sz
    lib.qmll_normal_equations_min_workspace_mode.argtypes = [i32, i32]
    lib.qmll_normal_equations_min_workspace_mode.restype = sz
    lib.qmll_predict.argtypes = [pp, vp, vp, vp, i64, i32, vp, gp, vp, vp, vp, sz, vp]
    lib.qmll_predict_static.argtypes = [pp, vp, vp, vp, i64, i32, vp, gp, vp, vp, vp]
    lib.qmll_predict_static.restype = ctypes.c_int
    lib.qmll_energies.argtypes = [vp, vp, i64, i32, vp, vp]
    lib.qmll_energies.restype = ctypes.c_int
    lib.qmll_predict_static_max_bytes.argtypes = []
    lib.qmll_predict_static_max_bytes.restype = sz
    lib.qmll_project.argtypes = [vp, vp, vp, i64, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.qmll_project.restype = ctypes.c_int
    lib.qmll_project_neighbor.argtypes = [vp, vp, vp, i64, i32, i32, i32, i32, vp, vp, vp]
    lib.qmll_project_neighbor.restype = ctypes.c_int
    lib.qmll_fchl19.argtypes = [ctypes.POINTER(_CFchl), vp, vp, i64, vp, vp, i32, vp, vp, vp, vp, vp]
    lib.qmll_fchl19.restype = ctypes.c_int
    lib.qmll_fchl19_rep_size.argtypes = [ctypes.POINTER(_CFchl)]
    lib.qmll_fchl19_rep_size.restype = i32
    lib.qmll_sorf_backward_g.argtypes = [pp, vp, vp, vp, i64, i32, vp, vp, vp, vp, sz, vp]
    lib.qmll_sorf_backward_g.restype = ctypes.c_int
    lib.qmll_project_back.argtypes = [vp, vp, i64, i32, i32, i32, vp, vp, vp]
    lib.qmll_project_back.restype = ctypes.c_int
    lib.qmll_fchl19_backward.argtypes = [ctypes.POINTER(_CFchl), vp, vp, i64, vp, vp, i32, vp, vp, vp, vp]
    lib.qmll_fchl19_backward.restype = ctypes.c_int
    lib.qmll_sorf_forward_mma.argtypes = [pp, vp, vp, vp, i64, i32, vp, vp, sz, vp]
    lib.qmll_sorf_forward_mma.restype = ctypes.c_int
    lib.qmll_rff_forward.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp, i64, i32, vp, vp, sz, vp]
    lib.qmll_rff_forward.restype = ctypes.c_int
    lib.qmll_featmap_workspace_bytes.argtypes = [i32, i32, i32, i64, i32]
    lib.qmll_featmap_workspace_bytes.restype = sz
    lib.qmll_pack_lower.argtypes = [vp, i32, vp, vp]
    lib.qmll_pack_lower.restype = ctypes.c_int
    lib.qmll_unpack_lower.argtypes = [vp, i32, vp, vp]
    lib.qmll_unpack_lower.restype = ctypes.c_int
    for name in ("qmll_sorf_forward", "qmll_sorf_backward_forces", "qmll_normal_equations", "qmll_predict"):
        getattr(lib, name).restype = ctypes.c_int
    lib.qmll_solve.argtypes = [vp, vp, i32, ctypes.c_double, vp, vp, vp, sz, vp]
    lib.qmll_solve.restype = ctypes.c_int
    lib.qmll_workspace_bytes.argtypes = [ctypes.c_int, pp, i64, i32, i64]
    lib.qmll_workspace_bytes.restype = sz
    lib.qmll_normal_equations_min_workspace.argtypes = [i32]
    lib.qmll_normal_equations_min_workspace.restype = sz
    lib.qmll_status_string.argtypes = [ctypes.c_int]
    lib.qmll_status_string.restype = ctypes.c_char_p
    lib.qmll_launch_count.restype = i64
    lib.qmll_reset_launch_count.restype = None
    lib.qmll_time_normal_equations_kernel.argtypes = [ctypes.c_int]
    lib.qmll_time_normal_equations_kernel.restype = None
    lib.qmll_collect_normal_equations_kernel_ms.argtypes = [ctypes.POINTER(ctypes.c_double),
                                                            ctypes.POINTER(ctypes.c_int)]
    lib.qmll_collect_normal_equations_kernel_ms.restype = ctypes.c_int
    _lib = lib
    return lib


def _check(status: int) -> None:
    if status != 0:
        raise QmllError(status, load_library().qmll_status_string(status).decode())


def _dev(t: Optional[torch.Tensor], dtype, name: str):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of dtype {dtype}")
    return ctypes.c_void_p(t.data_ptr())


def _stream() -> ctypes.c_void_p:
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


@dataclass
class SorfParams:
    """qmll_sorf_params: signs int8 [E, D/d, T, d] and bias fp32 [E, D] are CUDA tensors."""
    d: int
    D: int
    n_transform: int
    n_elem: int
    sigma: float
    signs: torch.Tensor
    bias: torch.Tensor

    def c(self) -> _CParams:
        return _CParams(self.d, self.D, self.n_transform, self.n_elem, float(self.sigma),
                        _dev(self.signs, torch.int8, "signs"), _dev(self.bias, torch.float32, "bias"))


@dataclass
class Grad:
    """qmll_grad: dense (flat fp32 + int64 offsets [n_mol+1]) or neighbour (int32 [n,K] + fp32 [n,K,d,3])."""
    layout: int
    dense: Optional[torch.Tensor] = None
    dense_off: Optional[torch.Tensor] = None
    nbr_idx: Optional[torch.Tensor] = None
    nbr_val: Optional[torch.Tensor] = None
    K: int = 0

    @staticmethod
    def make_dense(dense: torch.Tensor, dense_off: torch.Tensor) -> "Grad":
        return Grad(QMLL_GRAD_DENSE, dense=dense, dense_off=dense_off)

    @staticmethod
    def make_neighbor(nbr_idx: torch.Tensor, nbr_val: torch.Tensor) -> "Grad":
        return Grad(QMLL_GRAD_NEIGHBOR, nbr_idx=nbr_idx, nbr_val=nbr_val, K=int(nbr_idx.shape[1]))

    def c(self) -> _CGrad:
        return _CGrad(self.layout, _dev(self.dense, torch.float32, "dense"),
                      _dev(self.dense_off, torch.int64, "dense_off"), _dev(self.nbr_idx, torch.int32, "nbr_idx"),
                      _dev(self.nbr_val, torch.float32, "nbr_val"), int(self.K),
                      int(self.dense.numel()) if self.dense is not None else 0)


_workspaces: dict = {}


def workspace(nbytes: int, device) -> torch.Tensor:
    """A cached, grow-only scratch tensor per (device, stream): the C-ABI is stateless but this cache is not, so
    calls issued on different streams never share scratch.  A replaced tensor is handed back to torch's caching
    allocator, which is keyed to the stream it was allocated on -- the only stream that ever used it."""
    dev = torch.device(device)
    index = dev.index if dev.index is not None else torch.cuda.current_device()
    with torch.cuda.device(index):
        key = (index, torch.cuda.current_stream().cuda_stream)
        ws = _workspaces.get(key)
        if ws is None or ws.numel() < nbytes:
            _workspaces.pop(key, None)
            ws = None
            ws = torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=torch.device("cuda", index))
            _workspaces[key] = ws
    return ws


def release_workspaces() -> None:
    _workspaces.clear()


def workspace_bytes(which: int, p: SorfParams, n_atoms: int = 0, n_mol: int = 0, rows: int = 0) -> int:
    cp = p.c()
    return int(load_library().qmll_workspace_bytes(which, ctypes.byref(cp), n_atoms, n_mol, rows))


def _problem(x, elem, mol_off):
    n_atoms, n_mol = int(elem.shape[0]), int(mol_off.shape[0]) - 1
    return (_dev(x, torch.float32, "x"), _dev(elem, torch.int32, "elem"), _dev(mol_off, torch.int32, "mol_off"),
            n_atoms, n_mol)


def qmll_sorf_forward(p: SorfParams, x, elem, mol_off, grad: Optional[Grad] = None, Z=None, G=None,
                      want_Z: bool = True, force_rows_mode: int = ROWS_AUTO):
    """Z [n_mol, D] (and G [3 n_atoms, D] when `grad` is given): include/qmll.h qmll_sorf_forward."""
    lib = load_library()
    xp, ep, mp, n_atoms, n_mol = _problem(x, elem, mol_off)
    if Z is None and want_Z:
        Z = torch.empty((n_mol, p.D), dtype=torch.float32, device=x.device)
    if grad is not None and G is None:
        G = torch.empty((3 * n_atoms, p.D), dtype=torch.float32, device=x.device)
    cp = p.c()
    cg = grad.c() if grad is not None else None
    dense_floats = int(grad.dense.numel()) if (grad is not None and grad.dense is not None) else 0
    nb = lib.qmll_workspace_bytes(CALL_FORWARD_GRAD if grad is not None else CALL_FORWARD, ctypes.byref(cp),
                                  n_atoms, n_mol, dense_floats)
    ws = workspace(nb, x.device)
    _check(lib.qmll_sorf_forward_mode(ctypes.byref(cp), xp, ep, mp, n_atoms, n_mol,
                                      ctypes.byref(cg) if cg is not None else None, _dev(Z, torch.float32, "Z"),
                                      _dev(G, torch.float32, "G"), ctypes.c_void_p(ws.data_ptr()), ws.numel(),
                                      force_rows_mode, _stream()))
    return (Z, G) if grad is not None else Z


def qmll_sorf_backward_forces(p: SorfParams, x, elem, mol_off, alpha, grad: Grad, forces=None):
    """forces [n_atoms, 3] = -dE/dr: include/qmll.h qmll_sorf_backward_forces."""
    lib = load_library()
    xp, ep, mp, n_atoms, n_mol = _problem(x, elem, mol_off)
    if forces is None:
        forces = torch.empty((n_atoms, 3), dtype=torch.float32, device=x.device)
    cp, cg = p.c(), grad.c()
    nb = lib.qmll_workspace_bytes(CALL_BACKWARD_FORCES, ctypes.byref(cp), n_atoms, n_mol, 0)
    ws = workspace(nb, x.device)
    _check(lib.qmll_sorf_backward_forces(ctypes.byref(cp), xp, ep, mp, n_atoms, n_mol,
                                         _dev(alpha, torch.float32, "alpha"), ctypes.byref(cg),
                                         _dev(forces, torch.float32, "forces"), ctypes.c_void_p(ws.data_ptr()),
                                         ws.numel(), _stream()))
    return forces


def qmll_predict(p: SorfParams, x, elem, mol_off, alpha, grad: Optional[Grad] = None, energies=None, forces=None):
    """(energies [n_mol], forces [n_atoms, 3] or None): include/qmll.h qmll_predict."""
    lib = load_library()
    xp, ep, mp, n_atoms, n_mol = _problem(x, elem, mol_off)
    if energies is None:
        energies = torch.empty((n_mol,), dtype=torch.float32, device=x.device)
    if grad is not None and forces is None:
        forces = torch.empty((n_atoms, 3), dtype=torch.float32, device=x.device)
    cp = p.c()
    cg = grad.c() if grad is not None else None
    nb = lib.qmll_workspace_bytes(CALL_PREDICT, ctypes.byref(cp), n_atoms, n_mol, 0)
    ws = workspace(nb, x.device)
    _check(lib.qmll_predict(ctypes.byref(cp), xp, ep, mp, n_atoms, n_mol, _dev(alpha, torch.float32, "alpha"),
                            ctypes.byref(cg) if cg is not None else None, _dev(energies, torch.float32, "energies"),
                            _dev(forces, torch.float32, "forces"), ctypes.c_void_p(ws.data_ptr()), ws.numel(),
                            _stream()))
    return energies, forces


def qmll_energies(Z, alpha, energies=None):
    """energies [n_mol] = Z @ alpha: include/qmll.h qmll_energies (step a4 for a caller that holds Z)."""
    lib = load_library()
    n_mol, D = int(Z.shape[0]), int(Z.shape[1])
    if energies is None:
        energies = torch.empty((n_mol,), dtype=torch.float32, device=Z.device)
    _check(lib.qmll_energies(_dev(Z, torch.float32, "Z"), _dev(alpha, torch.float32, "alpha"), n_mol, D,
                             _dev(energies, torch.float32, "energies"), _stream()))
    return energies


def qmll_predict_static(p: SorfParams, x, elem, mol_off, alpha, energies, grad: Optional[Grad] = None, forces=None):
    """include/qmll.h qmll_predict_static: qmll_predict on the library's static scratch.  The call allocates nothing,
    so the outputs are the caller's: energies [n_mol] and, with grad, forces [n_atoms, 3].  Calls that overlap on the
    GPU race on the shared scratch; problems beyond qmll_predict_static_max_bytes() raise QmllError (status -3)."""
    lib = load_library()
    xp, ep, mp, n_atoms, n_mol = _problem(x, elem, mol_off)
    if energies is None or (grad is not None and forces is None):
        raise ValueError("qmll_predict_static allocates nothing: pass energies (and forces with grad)")
    cp = p.c()
    cg = grad.c() if grad is not None else None
    status = lib.qmll_predict_static(ctypes.byref(cp), xp, ep, mp, n_atoms, n_mol, _dev(alpha, torch.float32, "alpha"),
                                     ctypes.byref(cg) if cg is not None else None,
                                     _dev(energies, torch.float32, "energies"), _dev(forces, torch.float32, "forces"),
                                     _stream())
    if status == -3:
        need = int(lib.qmll_workspace_bytes(CALL_PREDICT, ctypes.byref(cp), n_atoms, n_mol, 0))
        raise QmllError(status, f"qmll_predict_static: this problem needs {need} bytes of scratch, the static array "
                                f"holds {int(lib.qmll_predict_static_max_bytes())}; use qmll_predict with a workspace")
    _check(status)
    return energies, forces


def qmll_normal_equations(A, y=None, ZtZ=None, Zty=None, accumulate: bool = False,
                          workspace_limit: Optional[int] = None, mode: int = NE_SPLIT_F16):
    """(ZtZ [D, D], Zty [D] or None) (+)= (A^T A, A^T y): include/qmll.h qmll_normal_equations(_mode)."""
    lib = load_library()
    rows, D = int(A.shape[0]), int(A.shape[1])
    if ZtZ is None:
        if accumulate:
            raise ValueError("accumulate=True needs ZtZ")
        ZtZ = torch.empty((D, D), dtype=torch.float32, device=A.device)
    if y is not None and Zty is None:
        if accumulate:
            raise ValueError("accumulate=True needs Zty")
        Zty = torch.empty((D,), dtype=torch.float32, device=A.device)
    nb = int(lib.qmll_normal_equations_workspace(rows, D, mode))
    if workspace_limit is not None:
        nb = max(min(nb, int(workspace_limit)), int(lib.qmll_normal_equations_min_workspace_mode(D, mode)))
    ws = workspace(nb, A.device)
    _check(lib.qmll_normal_equations_mode(_dev(A, torch.float32, "A") if rows > 0 else None,
                                          _dev(y, torch.float32, "y"), rows, D, 1 if accumulate else 0,
                                          _dev(ZtZ, torch.float32, "ZtZ"), _dev(Zty, torch.float32, "Zty"),
                                          ctypes.c_void_p(ws.data_ptr()), min(ws.numel(), nb), mode, _stream()))
    return ZtZ, Zty


def qmll_project(rho, elem, U, mol_off=None, grad_in=None, grad_in_off=None, grad_out_off=None, want_x: bool = True):
    """(x [n_atoms, d], projected dense gradient or None): include/qmll.h qmll_project (eq. 21-22)."""
    n_elem, rep, d = (int(v) for v in U.shape)
    n_atoms = int(elem.shape[0])
    x = torch.empty((n_atoms, d), dtype=torch.float32, device=U.device) if want_x else None
    gout = None
    n_mol = 0
    if grad_in is not None:
        n_mol = int(mol_off.shape[0]) - 1
        total = int(grad_out_off[-1].item()) if grad_out_off.numel() else 0
        gout = torch.empty((total,), dtype=torch.float32, device=U.device)
    _check(load_library().qmll_project(_dev(rho, torch.float32, "rho"), _dev(elem, torch.int32, "elem"),
                                       _dev(mol_off, torch.int32, "mol_off"), n_atoms, n_mol, rep, d, n_elem,
                                       _dev(U, torch.float32, "U"), _dev(x, torch.float32, "x"),
                                       _dev(grad_in, torch.float32, "grad_in"), _dev(grad_in_off, torch.int64, "grad_in_off"),
                                       _dev(gout, torch.float32, "grad_out"), _dev(grad_out_off, torch.int64, "grad_out_off"),
                                       _stream()))
    return x, gout


def qmll_sorf_forward_mma(p: SorfParams, x, elem, mol_off, Z=None):
    """Z [n_mol, D] of steps a1-a3 on the tensor cores (expanded W, d = 128 / 256): include/qmll.h."""
    lib = load_library()
    xp, ep, mp, n_atoms, n_mol = _problem(x, elem, mol_off)
    if Z is None:
        Z = torch.empty((n_mol, p.D), dtype=torch.float32, device=x.device)
    nbytes = int(lib.qmll_featmap_workspace_bytes(p.d, p.D, p.n_elem, n_atoms, 0))
    ws = workspace(nbytes, x.device)
    cp = p.c()
    _check(lib.qmll_sorf_forward_mma(ctypes.byref(cp), xp, ep, mp, n_atoms, n_mol, _dev(Z, torch.float32, "Z"),
                                     ctypes.c_void_p(ws.data_ptr()), ws.numel(), _stream()))
    return Z


def qmll_rff_forward(W, bias, x, elem, mol_off, Z=None):
    """Z [n_mol, D] of the dense-matrix random Fourier feature map (eq. 12-14, 18): W [n_elem, D, d], bias [n_elem, D]."""
    lib = load_library()
    n_elem, D, d = (int(v) for v in W.shape)
    xp, ep, mp, n_atoms, n_mol = _problem(x, elem, mol_off)
    if Z is None:
        Z = torch.empty((n_mol, D), dtype=torch.float32, device=x.device)
    nbytes = int(lib.qmll_featmap_workspace_bytes(d, D, n_elem, n_atoms, 1))
    ws = workspace(nbytes, x.device)
    _check(lib.qmll_rff_forward(_dev(W, torch.float32, "W"), _dev(bias, torch.float32, "bias"), d, D, n_elem, xp, ep, mp,
                                n_atoms, n_mol, _dev(Z, torch.float32, "Z"), ctypes.c_void_p(ws.data_ptr()), ws.numel(),
                                _stream()))
    return Z


@dataclass
class Fchl19Params:
    """qmll_fchl19_params (Table I; defaults = column E + F)."""
    n_elem: int = 5
    n2: int = 24
    n3: int = 20
    eta2: float = 0.32
    eta3: float = 2.7
    two_body_decay: float = 1.8
    three_body_decay: float = 0.57
    three_body_weight: float = 13.4
    zeta: float = 3.141592653589793
    r_cut: float = 6.0

    def c(self) -> _CFchl:
        return _CFchl(self.n_elem, self.n2, self.n3, self.eta2, self.eta3, self.two_body_decay, self.three_body_decay,
                      self.three_body_weight, self.zeta, self.r_cut)

    @property
    def rep(self) -> int:
        cp = self.c()
        return int(load_library().qmll_fchl19_rep_size(ctypes.byref(cp)))


def qmll_fchl19(fp: Fchl19Params, r, elem, nbr_idx, nbr_shift=None, jacobian: bool = False, want_rho: bool = True):
    """(rho [n_atoms, rep], jac_idx [n_atoms, K + 1] | None, jac_val [n_atoms, K + 1, rep, 3] | None, info int32[1]):
    include/qmll.h qmll_fchl19 (eq. 23-33).  (jac_idx, jac_val) is a NEIGHBOR-layout gradient of length rep."""
    n_atoms, K = int(nbr_idx.shape[0]), int(nbr_idx.shape[1])
    rep = fp.rep
    if rep < 0:
        raise QmllError(-1, "qmll_fchl19_params invalid or outside the supported range (include/qmll.h)")
    dev = r.device
    rho = torch.empty((n_atoms, rep), dtype=torch.float32, device=dev) if want_rho else None
    jac_idx = torch.empty((n_atoms, K + 1), dtype=torch.int32, device=dev) if jacobian else None
    jac_val = torch.empty((n_atoms, K + 1, rep, 3), dtype=torch.float32, device=dev) if jacobian else None
    info = torch.zeros((1,), dtype=torch.int32, device=dev)
    cp = fp.c()
    _check(load_library().qmll_fchl19(ctypes.byref(cp), _dev(r, torch.float32, "r"), _dev(elem, torch.int32, "elem"),
                                      n_atoms, _dev(nbr_idx, torch.int32, "nbr_idx"),
                                      _dev(nbr_shift, torch.float32, "nbr_shift"), K, _dev(rho, torch.float32, "rho"),
                                      _dev(jac_idx, torch.int32, "jac_idx"), _dev(jac_val, torch.float32, "jac_val"),
                                      _dev(info, torch.int32, "info"), _stream()))
    return rho, jac_idx, jac_val, info


def qmll_sorf_backward_g(p: SorfParams, x, elem, mol_off, alpha, want_energies: bool = True):
    """(energies [n_mol] | None, g [n_atoms, d] = dE/dx): include/qmll.h qmll_sorf_backward_g (step a5 alone)."""
    lib = load_library()
    xp, ep, mp, n_atoms, n_mol = _problem(x, elem, mol_off)
    g = torch.empty((n_atoms, p.d), dtype=torch.float32, device=x.device)
    E = torch.empty((n_mol,), dtype=torch.float32, device=x.device) if want_energies else None
    ws = workspace(workspace_bytes(CALL_PREDICT, p, n_atoms, n_mol), x.device)
    cp = p.c()
    _check(lib.qmll_sorf_backward_g(ctypes.byref(cp), xp, ep, mp, n_atoms, n_mol, _dev(alpha, torch.float32, "alpha"),
                                    _dev(E, torch.float32, "energies"), _dev(g, torch.float32, "g"),
                                    ctypes.c_void_p(ws.data_ptr()), ws.numel(), _stream()))
    return E, g


def qmll_project_back(g, elem, U):
    """w [n_atoms, rep] = U_e g (dE / d rho from dE / dx): include/qmll.h qmll_project_back."""
    n_elem, rep, d = (int(v) for v in U.shape)
    n_atoms = int(elem.shape[0])
    w = torch.empty((n_atoms, rep), dtype=torch.float32, device=U.device)
    _check(load_library().qmll_project_back(_dev(g, torch.float32, "g"), _dev(elem, torch.int32, "elem"), n_atoms, rep, d,
                                            n_elem, _dev(U, torch.float32, "U"), _dev(w, torch.float32, "w"), _stream()))
    return w


def qmll_fchl19_backward(fp: "Fchl19Params", r, elem, nbr_idx, w, nbr_shift=None, forces=None):
    """(forces [n_atoms, 3], info): F = -sum_I w_I . d rho_I / d r without a Jacobian: include/qmll.h."""
    n_atoms, K = int(nbr_idx.shape[0]), int(nbr_idx.shape[1])
    if fp.rep < 0:
        raise QmllError(-1, "qmll_fchl19_params invalid or outside the supported range (include/qmll.h)")
    if forces is None:
        forces = torch.empty((n_atoms, 3), dtype=torch.float32, device=r.device)
    info = torch.zeros((1,), dtype=torch.int32, device=r.device)
    cp = fp.c()
    _check(load_library().qmll_fchl19_backward(ctypes.byref(cp), _dev(r, torch.float32, "r"), _dev(elem, torch.int32, "elem"),
                                               n_atoms, _dev(nbr_idx, torch.int32, "nbr_idx"),
                                               _dev(nbr_shift, torch.float32, "nbr_shift"), K, _dev(w, torch.float32, "w"),
                                               _dev(forces, torch.float32, "forces"), _dev(info, torch.int32, "info"),
                                               _stream()))
    return forces, info


def qmll_project_neighbor(grad_in, elem, U, idx=None, grad_out=None):
    """[n_atoms, S, rep, 3] -> [n_atoms, S, d, 3] with every atom's own U_e: include/qmll.h qmll_project_neighbor."""
    n_elem, rep, d = (int(v) for v in U.shape)
    n_atoms, S = int(grad_in.shape[0]), int(grad_in.shape[1])
    if grad_out is None:
        grad_out = torch.empty((n_atoms, S, d, 3), dtype=torch.float32, device=U.device)
    _check(load_library().qmll_project_neighbor(_dev(grad_in, torch.float32, "grad_in"), _dev(idx, torch.int32, "idx"),
                                                _dev(elem, torch.int32, "elem"), n_atoms, S, rep, d, n_elem,
                                                _dev(U, torch.float32, "U"), _dev(grad_out, torch.float32, "grad_out"),
                                                _stream()))
    return grad_out


def qmll_pack_lower(ZtZ, packed=None):
    """Row-packed lower triangle of ZtZ [D (D + 1) / 2]: include/qmll.h qmll_pack_lower."""
    D = int(ZtZ.shape[0])
    if packed is None:
        packed = torch.empty((D * (D + 1) // 2,), dtype=torch.float32, device=ZtZ.device)
    _check(load_library().qmll_pack_lower(_dev(ZtZ, torch.float32, "ZtZ"), D, _dev(packed, torch.float32, "packed"),
                                          _stream()))
    return packed


def qmll_unpack_lower(packed, ZtZ):
    """ZtZ (both triangles) from its row-packed lower triangle: include/qmll.h qmll_unpack_lower."""
    D = int(ZtZ.shape[0])
    _check(load_library().qmll_unpack_lower(_dev(packed, torch.float32, "packed"), D, _dev(ZtZ, torch.float32, "ZtZ"),
                                            _stream()))
    return ZtZ


def qmll_solve(ZtZ, Zty, lam: float, alpha=None):
    """(alpha [D], info int32[1]) with (ZtZ + lam I) alpha = Zty: include/qmll.h qmll_solve (FP64 Cholesky)."""
    lib = load_library()
    D = int(ZtZ.shape[0])
    if alpha is None:
        alpha = torch.empty((D,), dtype=torch.float32, device=ZtZ.device)
    info = torch.zeros((1,), dtype=torch.int32, device=ZtZ.device)
    cp = _CParams(0, D, 0, 0, 0.0, None, None)
    nb = int(lib.qmll_workspace_bytes(CALL_SOLVE, ctypes.byref(cp), 0, 0, 0))
    ws = workspace(nb, ZtZ.device)
    _check(lib.qmll_solve(_dev(ZtZ, torch.float32, "ZtZ"), _dev(Zty, torch.float32, "Zty"), D, float(lam),
                          _dev(alpha, torch.float32, "alpha"), _dev(info, torch.int32, "info"),
                          ctypes.c_void_p(ws.data_ptr()), ws.numel(), _stream()))
    return alpha, info


def launch_count() -> int:
    return int(load_library().qmll_launch_count())


def reset_launch_count() -> None:
    load_library().qmll_reset_launch_count()


def time_normal_equations_kernel(enable: bool) -> None:
    load_library().qmll_time_normal_equations_kernel(1 if enable else 0)


def collect_normal_equations_kernel_ms():
    """(summed ms, launches) of the tcgen05 kernel since the last collect (waits for the events)."""
    ms, n = ctypes.c_double(0.0), ctypes.c_int(0)
    _check(load_library().qmll_collect_normal_equations_kernel_ms(ctypes.byref(ms), ctypes.byref(n)))
    return float(ms.value), int(n.value)
