"""oracle/ -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

numpy/ctypes front end of `sorf_oracle.c`, the plain FP64 CPU statement of the SORF hot path
(eq. 14-17, 20; see the C file's header for readings and pins).  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may import
this package; the product (`paper_2206_01580_b200/`) never does, and this package never
imports the product.  Arguments are plain numpy arrays and scalars (the same fp32/int8/int32
arrays the GPU library is given); results are float64.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sorf_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "fchl19_oracle.c")]
_LIB = os.path.join(_HERE, "libsorf_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile sorf_oracle.c and fchl19_oracle.c with gcc (-O2, no fast-math, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(s) for s in _SRCS):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared"] + _SRCS + ["-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.qo_scale.restype = ctypes.c_double
        _lib.qo_scale.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double]
        _lib.qo_num_threads.restype = ctypes.c_int
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _i8(a):
    return np.ascontiguousarray(a, dtype=np.int8)


_I, _L, _D = ctypes.c_int, ctypes.c_int64, ctypes.c_double


def num_threads() -> int:
    return int(_load().qo_num_threads())


def fwht(v: np.ndarray) -> np.ndarray:
    """Unnormalised natural-order Walsh-Hadamard transform of a length-2^n vector (L163-167)."""
    out = np.array(v, dtype=np.float64, copy=True)
    _load().qo_fwht(_p(out), _I(out.shape[0]))
    return out


def scale(d: int, T: int, sigma: float) -> float:
    return float(_load().qo_scale(d, T, float(sigma)))


def sorf_u(x_I, e: int, d: int, D: int, T: int, sigma: float, signs) -> np.ndarray:
    """u = W_e x_I (eq. 20), length D, stack-major."""
    x_I, signs = _f32(x_I), _i8(signs)
    u = np.empty(D, dtype=np.float64)
    _load().qo_sorf_u(_p(x_I), _I(e), _I(d), _I(D), _I(T), _D(sigma), _p(signs), _p(u))
    return u


def forward(x, elem, mol_off, d, D, T, sigma, signs, bias) -> np.ndarray:
    """Z[n_mol, D] (eq. 14 + eq. 15)."""
    x, elem, mol_off, signs, bias = _f32(x), _i32(elem), _i32(mol_off), _i8(signs), _f32(bias)
    n_mol = mol_off.shape[0] - 1
    Z = np.empty((n_mol, D), dtype=np.float64)
    _load().qo_forward(_p(x), _p(elem), _p(mol_off), _L(elem.shape[0]), _I(n_mol), _I(d), _I(D), _I(T),
                       _D(sigma), _p(signs), _p(bias), _p(Z))
    return Z


def rff_forward(W, bias, x, elem, mol_off) -> np.ndarray:
    """Z[n_mol, D] of the dense-matrix random Fourier feature map (eq. 12-14, 18): W [n_elem, D, d], bias [n_elem, D]."""
    W, bias, x, elem, mol_off = _f32(W), _f32(bias), _f32(x), _i32(elem), _i32(mol_off)
    n_elem, D, d = W.shape
    n_mol = mol_off.shape[0] - 1
    Z = np.empty((n_mol, D), dtype=np.float64)
    _load().qo_rff_forward(_p(W), _p(bias), _I(d), _I(D), _p(x), _p(elem), _p(mol_off), _I(n_mol), _p(Z))
    return Z


def energy(Z, alpha) -> np.ndarray:
    Z = np.ascontiguousarray(Z, dtype=np.float64)
    alpha = _f32(alpha)
    out = np.empty(Z.shape[0], dtype=np.float64)
    _load().qo_energy(_p(Z), _p(alpha), _I(Z.shape[0]), _I(Z.shape[1]), _p(out))
    return out


def backward_g(x, elem, d, D, T, sigma, signs, bias, alpha) -> np.ndarray:
    """g[n_atoms, d] = dE/dx (chain rule through eq. 14 and the transposed eq. 20)."""
    x, elem, signs, bias, alpha = _f32(x), _i32(elem), _i8(signs), _f32(bias), _f32(alpha)
    g = np.empty((elem.shape[0], d), dtype=np.float64)
    _load().qo_backward_g(_p(x), _p(elem), _L(elem.shape[0]), _I(d), _I(D), _I(T), _D(sigma), _p(signs),
                          _p(bias), _p(alpha), _p(g))
    return g


def forces_dense(g, mol_off, d, dense, dense_off) -> np.ndarray:
    g = np.ascontiguousarray(g, dtype=np.float64)
    mol_off, dense = _i32(mol_off), _f32(dense)
    dense_off = np.ascontiguousarray(dense_off, dtype=np.int64)
    F = np.zeros((g.shape[0], 3), dtype=np.float64)
    _load().qo_forces_dense(_p(g), _p(mol_off), _I(mol_off.shape[0] - 1), _I(d), _p(dense), _p(dense_off), _p(F))
    return F


def forces_neighbor(g, d, nbr_idx, nbr_val) -> np.ndarray:
    g = np.ascontiguousarray(g, dtype=np.float64)
    nbr_idx, nbr_val = _i32(nbr_idx), _f32(nbr_val)
    F = np.zeros((g.shape[0], 3), dtype=np.float64)
    _load().qo_forces_neighbor(_p(g), _L(g.shape[0]), _I(d), _I(nbr_idx.shape[1]), _p(nbr_idx), _p(nbr_val), _p(F))
    return F


def force_rows_dense(x, elem, mol_off, d, D, T, sigma, signs, bias, dense, dense_off) -> np.ndarray:
    """G[3 n_atoms, D] = -dZ/dr, rows (M, j, k) (L137, reading A8)."""
    x, elem, mol_off, signs, bias, dense = _f32(x), _i32(elem), _i32(mol_off), _i8(signs), _f32(bias), _f32(dense)
    dense_off = np.ascontiguousarray(dense_off, dtype=np.int64)
    G = np.zeros((3 * elem.shape[0], D), dtype=np.float64)
    _load().qo_force_rows_dense(_p(x), _p(elem), _p(mol_off), _I(mol_off.shape[0] - 1), _I(d), _I(D), _I(T),
                                _D(sigma), _p(signs), _p(bias), _p(dense), _p(dense_off), _p(G))
    return G


def force_rows_neighbor(x, elem, d, D, T, sigma, signs, bias, nbr_idx, nbr_val) -> np.ndarray:
    x, elem, signs, bias = _f32(x), _i32(elem), _i8(signs), _f32(bias)
    nbr_idx, nbr_val = _i32(nbr_idx), _f32(nbr_val)
    G = np.zeros((3 * elem.shape[0], D), dtype=np.float64)
    _load().qo_force_rows_neighbor(_p(x), _p(elem), _L(elem.shape[0]), _I(d), _I(D), _I(T), _D(sigma), _p(signs),
                                   _p(bias), _I(nbr_idx.shape[1]), _p(nbr_idx), _p(nbr_val), _p(G))
    return G


def normal_equations(A, y):
    """(ZtZ, Zty) = (A^T A, A^T y) in FP64 from the fp32 rows the GPU is given (eq. 16-17)."""
    A, y = _f32(A), _f32(y)
    rows, D = A.shape
    ZtZ = np.empty((D, D), dtype=np.float64)
    Zty = np.empty(D, dtype=np.float64)
    _load().qo_normal_equations(_p(A), _p(y), _L(rows), _I(D), _p(ZtZ), _p(Zty))
    return ZtZ, Zty


def solve(ZtZ, Zty, lam: float):
    """(alpha[D] float64, info): (ZtZ + lam I) alpha = Zty by FP64 Cholesky (eq. 16-17)."""
    ZtZ, Zty = _f32(ZtZ), _f32(Zty)
    D = ZtZ.shape[0]
    alpha = np.zeros(D, dtype=np.float64)
    lib = _load()
    lib.qo_solve.restype = ctypes.c_int
    info = lib.qo_solve(_p(ZtZ), _p(Zty), _I(D), _D(lam), _p(alpha))
    return alpha, int(info)


def gram_entries(A, ii, jj) -> np.ndarray:
    A, ii, jj = _f32(A), _i32(ii), _i32(jj)
    out = np.empty(ii.shape[0], dtype=np.float64)
    _load().qo_gram_entries(_p(A), _L(A.shape[0]), _I(A.shape[1]), _p(ii), _p(jj), _L(ii.shape[0]), _p(out))
    return out


def gram_rows(A, y, ii):
    A, ii = _f32(A), _i32(ii)
    y = None if y is None else _f32(y)
    out = np.empty((ii.shape[0], A.shape[1]), dtype=np.float64)
    out_y = np.empty(ii.shape[0], dtype=np.float64)
    _load().qo_gram_rows(_p(A), _p(y), _L(A.shape[0]), _I(A.shape[1]), _p(ii), _I(ii.shape[0]), _p(out), _p(out_y))
    return out, out_y


def project(rho, elem, U) -> np.ndarray:
    """x [n_atoms, d] = rho_I^T U_e (eq. 22): rho [n_atoms, rep] fp32, U [n_elem, rep, d] fp32."""
    rho, elem, U = _f32(rho), _i32(elem), _f32(U)
    n_atoms, rep = rho.shape
    d = U.shape[2]
    x = np.empty((n_atoms, d), dtype=np.float64)
    _load().qo_project(_p(rho), _p(elem), _L(n_atoms), _I(rep), _I(d), _p(U), _p(x))
    return x


def project_gradient(gin, in_off, elem, mol_off, U, out_off) -> np.ndarray:
    """Dense gradient [n, rep, n, 3] per molecule -> [n, d, n, 3] per molecule (flat float64, offsets out_off)."""
    gin, elem, mol_off, U = _f32(gin), _i32(elem), _i32(mol_off), _f32(U)
    in_off = np.ascontiguousarray(in_off, dtype=np.int64)
    out_off = np.ascontiguousarray(out_off, dtype=np.int64)
    rep, d = U.shape[1], U.shape[2]
    gout = np.zeros(int(out_off[-1]), dtype=np.float64)
    _load().qo_project_gradient(_p(gin), _p(in_off), _p(elem), _p(mol_off), _I(mol_off.shape[0] - 1), _I(rep), _I(d),
                                _p(U), _p(out_off), _p(gout))
    return gout


# ---- FCHL19 representation and its Jacobian (fchl19_oracle.c; eq. 23-33) ----

def _fchl_args(fp):
    """fp: any object with n_elem, n2, n3, eta2, eta3, N2, N3, c3, zeta, r_cut (attribute access only)."""
    return [_I(fp.n_elem), _I(fp.n2), _I(fp.n3), _D(fp.eta2), _D(fp.eta3), _D(fp.N2), _D(fp.N3), _D(fp.c3),
            _D(fp.zeta), _D(fp.r_cut)]


def fchl19_rep_size(fp) -> int:
    return int(_load().qo_fchl19_rep_size(_I(fp.n_elem), _I(fp.n2), _I(fp.n3)))


def fchl19(fp, r, elem, nbr_idx, nbr_shift=None) -> np.ndarray:
    """rho [n_atoms, rep]: the FCHL19 representation of every atom from its neighbour images (readings B1-B8)."""
    r, elem, nbr_idx = _f32(r), _i32(elem), _i32(nbr_idx)
    nbr_shift = None if nbr_shift is None else _f32(nbr_shift)
    n_atoms, K = nbr_idx.shape
    rho = np.empty((n_atoms, fchl19_rep_size(fp)), dtype=np.float64)
    _load().qo_fchl19(_p(r), _p(elem), _L(n_atoms), _p(nbr_idx), _p(nbr_shift), _I(K), *_fchl_args(fp), _p(rho))
    return rho


def fchl19_jacobian(fp, r, elem, nbr_idx, nbr_shift=None, atoms=None) -> np.ndarray:
    """jac [n_sel, K + 1, rep, 3] for the atoms in `atoms` (default: all): slot 0 = the atom itself, slot 1 + q =
    neighbour slot q (reading B9); complex-step derivative of the representation."""
    r, elem, nbr_idx = _f32(r), _i32(elem), _i32(nbr_idx)
    nbr_shift = None if nbr_shift is None else _f32(nbr_shift)
    n_atoms, K = nbr_idx.shape
    atoms = np.arange(n_atoms, dtype=np.int64) if atoms is None else np.ascontiguousarray(atoms, dtype=np.int64)
    jac = np.empty((atoms.shape[0], K + 1, fchl19_rep_size(fp), 3), dtype=np.float64)
    _load().qo_fchl19_jacobian(_p(r), _p(elem), _p(nbr_idx), _p(nbr_shift), _I(K), _p(atoms), _L(atoms.shape[0]),
                               *_fchl_args(fp), _p(jac))
    return jac


def fchl19_atom(fp, centre, img, img_elem, jacobian: bool = False):
    """rho [rep] (and jac [nn + 1, rep, 3]) of one atom from FP64 positions: centre [3], img [nn, 3]."""
    centre = np.ascontiguousarray(centre, dtype=np.float64)
    img = np.ascontiguousarray(img, dtype=np.float64).reshape(-1, 3)
    img_elem = _i32(img_elem)
    nn, rep = img.shape[0], fchl19_rep_size(fp)
    rho = np.empty(rep, dtype=np.float64)
    jac = np.empty((nn + 1, rep, 3), dtype=np.float64) if jacobian else None
    _load().qo_fchl19_atom_f64(_p(centre), _p(img), _p(img_elem), _I(nn), *_fchl_args(fp), _p(rho), _p(jac))
    return (rho, jac) if jacobian else rho


def project_back(g, elem, U) -> np.ndarray:
    """w [n_atoms, rep] = U_e g: dE / d rho from g = dE / dx (backward pass of eq. 22)."""
    g = np.ascontiguousarray(g, dtype=np.float64)
    elem, U = _i32(elem), _f32(U)
    n_atoms, d = g.shape
    rep = U.shape[1]
    w = np.empty((n_atoms, rep), dtype=np.float64)
    _load().qo_project_back(_p(g), _p(elem), _L(n_atoms), _I(rep), _I(d), _p(U), _p(w))
    return w


def fchl19_backward(fp, r, elem, nbr_idx, w, nbr_shift=None) -> np.ndarray:
    """F [n_atoms, 3] = -sum_i w_i . d rho_i / d r: contraction of the oracle's Jacobian with w = dE / d rho."""
    r, elem, nbr_idx = _f32(r), _i32(elem), _i32(nbr_idx)
    nbr_shift = None if nbr_shift is None else _f32(nbr_shift)
    w = np.ascontiguousarray(w, dtype=np.float64)
    n_atoms, K = nbr_idx.shape
    F = np.empty((n_atoms, 3), dtype=np.float64)
    _load().qo_fchl19_backward(_p(r), _p(elem), _L(n_atoms), _p(nbr_idx), _p(nbr_shift), _I(K), _p(w), *_fchl_args(fp),
                               _p(F))
    return F


def project_neighbor_gradient(gin, elem, U) -> np.ndarray:
    """[n_atoms, S, rep, 3] fp32 -> [n_atoms, S, d, 3] float64 with every atom's own U_e (eq. 21-22)."""
    gin, elem, U = _f32(gin), _i32(elem), _f32(U)
    n_atoms, S, rep, _ = gin.shape
    d = U.shape[2]
    out = np.empty((n_atoms, S, d, 3), dtype=np.float64)
    _load().qo_project_neighbor_gradient(_p(gin), _p(elem), _L(n_atoms), _I(S), _I(rep), _I(d), _p(U), _p(out))
    return out


# ---- conveniences over a workloads.Workload-shaped object (attribute access only; no import) ----

def _m(w):
    m = w.model
    return m.d, m.D, m.T, m.sigma, m.signs, m.bias


def forward_w(w) -> np.ndarray:
    return forward(w.x, w.elem, w.mol_off, *_m(w))


def backward_g_w(w, alpha=None) -> np.ndarray:
    return backward_g(w.x, w.elem, *_m(w), w.alpha if alpha is None else alpha)


def forces_w(w, alpha=None) -> np.ndarray:
    """F[n_atoms, 3] = -dE/dr through the supplied descriptor gradient (a5 + a6)."""
    g = backward_g_w(w, alpha)
    if w.grad.layout == "dense":
        return forces_dense(g, w.mol_off, w.model.d, w.grad.dense, w.grad.dense_off)
    return forces_neighbor(g, w.model.d, w.grad.nbr_idx, w.grad.nbr_val)


def force_rows_w(w) -> np.ndarray:
    if w.grad.layout == "dense":
        return force_rows_dense(w.x, w.elem, w.mol_off, *_m(w), w.grad.dense, w.grad.dense_off)
    return force_rows_neighbor(w.x, w.elem, *_m(w), w.grad.nbr_idx, w.grad.nbr_val)


def predict_w(w, alpha=None):
    """(energies[n_mol], forces[n_atoms, 3] or None): eq. 15 and F = -dE/dr."""
    a = w.alpha if alpha is None else alpha
    E = energy(forward_w(w), a)
    F = forces_w(w, a) if w.grad is not None else None
    return E, F
