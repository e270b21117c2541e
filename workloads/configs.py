"""Seeded generators for the five synthetic workloads of BASELINE.json:configs.

The paper measures on QM9, MD17/rMD17, 3BPA and periodic cells (PAPER.md L282-302,
L332-347, Table V).  None of those datasets is available, so these inputs
stand in for them: only shapes, sizes, element mixes and value distributions are
taken (BASELINE.json:configs[0..4]); no dataset record is reproduced.

Recipe (also stated in DESIGN.md "Input recipe"):
  * every array has its own stream  Generator(PCG64(SeedSequence([seed, tag, block])))
    with seed = 20220600 + config number, tag = one of the TAG_* constants below and
    block = index of a block of rows of the array (BLOCK_ROWS rows per block), so a big
    array can be filled by several threads and still be reproducible;
  * normal draws are float32 `standard_normal`, scaled by the stated STANDARD DEVIATION;
    `alpha ~ N(0, 1/D)` is read as variance 1/D;
  * element ids: H=0, C=1, N=2, O=3, F=4 (n_elem = 5 for every config);
  * element mean vectors mu[e, :] ~ N(0, 1) i.i.d. (BASELINE.json leaves them open).

Nothing in this file performs any step of the method (no transform, no cos, no Gram
product): it only draws and lays out inputs.
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

ELEMENTS = ("H", "C", "N", "O", "F")
N_ELEM = len(ELEMENTS)
H_, C_, N_, O_, F_ = range(5)

CONFIG_NAMES = ("c1", "c2", "c3", "c4", "c5")

TAG_MU, TAG_TOPO, TAG_X, TAG_SIGNS, TAG_BIAS, TAG_ALPHA, TAG_Y, TAG_GRAD, TAG_NBR = range(1, 10)
BLOCK_ROWS = 4096          # rows of the leading axis per independent stream
_BASE_SEED = 20220600


def _rng(seed: int, tag: int, block: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([seed, tag, block])))


def _normal_f32(seed: int, tag: int, shape, std: float, block_rows: int = BLOCK_ROWS) -> np.ndarray:
    """float32 N(0, std) array of `shape`, filled block-of-rows by block-of-rows."""
    shape = tuple(int(s) for s in shape)
    out = np.empty(shape, dtype=np.float32)
    n = shape[0] if shape else 0
    if out.size == 0:
        return out
    blocks = [(b, lo, min(lo + block_rows, n)) for b, lo in enumerate(range(0, n, block_rows))]

    def fill(args):
        b, lo, hi = args
        view = out[lo:hi]
        _rng(seed, tag, b).standard_normal(view.shape, dtype=np.float32, out=view)
        if std != 1.0:
            view *= np.float32(std)

    if len(blocks) == 1:
        fill(blocks[0])
    else:
        with ThreadPoolExecutor(max_workers=8) as pool:
            list(pool.map(fill, blocks))
    return out


@dataclass
class SorfModel:
    """The SORF 'model' minus alpha (eq. 20, eq. 14)."""
    d: int                    # descriptor length (power of two)
    D: int                    # number of features N_F (multiple of d)
    T: int                    # N_transform
    sigma: float
    n_elem: int
    signs: np.ndarray         # int8 [n_elem, D/d, T, d], entries +1/-1; t=0 is D_1 (applied first)
    bias: np.ndarray          # float32 [n_elem, D], b in [0, 2pi)

    @property
    def n_stacks(self) -> int:
        return self.D // self.d


@dataclass
class DescriptorGradient:
    """d x_I[m] / d r_{j,k}, in one of the two layouts of include/qmll.h."""
    layout: str                                # "dense" | "neighbor"
    dense: Optional[np.ndarray] = None         # float32 flat; molecule M (n atoms) holds [n, d, n, 3]
    dense_off: Optional[np.ndarray] = None     # int64 [n_mol+1] offsets (in floats) into `dense`
    nbr_idx: Optional[np.ndarray] = None       # int32 [n_atoms, K], global atom index or -1
    nbr_val: Optional[np.ndarray] = None       # float32 [n_atoms, K, d, 3]
    K: int = 0

    def dense_block(self, M: int, n: int, d: int) -> np.ndarray:
        lo, hi = int(self.dense_off[M]), int(self.dense_off[M + 1])
        return self.dense[lo:hi].reshape(n, d, n, 3)


@dataclass
class Workload:
    name: str
    model: SorfModel
    elem: np.ndarray                  # int32 [n_atoms]
    mol_off: np.ndarray               # int32 [n_mol+1]; atoms of a molecule are contiguous
    x: np.ndarray                     # float32 [n_atoms, d]
    alpha: np.ndarray                 # float32 [D]
    y: Optional[np.ndarray] = None    # float32 [n_mol (+ 3 n_atoms)]: energies then forces (M, j, k)
    grad: Optional[DescriptorGradient] = None
    meta: dict = field(default_factory=dict)

    @property
    def n_atoms(self) -> int:
        return int(self.elem.shape[0])

    @property
    def n_mol(self) -> int:
        return int(self.mol_off.shape[0] - 1)


def make_model(seed: int, d: int, D: int, T: int, sigma: float, n_elem: int = N_ELEM) -> SorfModel:
    """Rademacher sign diagonals and b ~ U[0, 2pi) per element (BASELINE.json:configs[0])."""
    assert d & (d - 1) == 0 and D % d == 0
    n_s = D // d
    bits = _rng(seed, TAG_SIGNS).integers(0, 2, size=(n_elem, n_s, T, d), dtype=np.int8)
    signs = (2 * bits - 1).astype(np.int8)
    bias = (_rng(seed, TAG_BIAS).random(size=(n_elem, D), dtype=np.float32) * np.float32(2.0 * np.pi))
    bias = np.minimum(bias, np.nextafter(np.float32(2.0 * np.pi), np.float32(0.0))).astype(np.float32)
    return SorfModel(d=d, D=D, T=T, sigma=float(sigma), n_elem=n_elem, signs=signs, bias=bias)


def _alpha(seed: int, D: int) -> np.ndarray:
    return _normal_f32(seed, TAG_ALPHA, (D,), std=float(1.0 / np.sqrt(D)))


def _mu(seed: int, d: int) -> np.ndarray:
    return _normal_f32(seed, TAG_MU, (N_ELEM, d), std=1.0)


def _x_around_mu(seed: int, elem: np.ndarray, mu: Optional[np.ndarray], d: int, std: float) -> np.ndarray:
    x = _normal_f32(seed, TAG_X, (elem.shape[0], d), std=std)
    if mu is not None:
        step = 1 << 16
        for lo in range(0, elem.shape[0], step):
            x[lo:lo + step] += mu[elem[lo:lo + step]]
    return x


def _dense_grad(seed: int, counts: np.ndarray, d: int, std: float) -> DescriptorGradient:
    sizes = (counts.astype(np.int64) ** 2) * (3 * d)
    off = np.zeros(counts.shape[0] + 1, dtype=np.int64)
    np.cumsum(sizes, out=off[1:])
    total = int(off[-1])
    # one stream per block of 2^22 floats of the flat array
    blk = 1 << 22
    flat = _normal_f32(seed, TAG_GRAD, (-(-total // blk), blk), std=std, block_rows=1).reshape(-1)[:total]
    return DescriptorGradient(layout="dense", dense=flat, dense_off=off)


def _fixed_topology(n_mol: int, composition) -> tuple[np.ndarray, np.ndarray]:
    comp = np.asarray(composition, dtype=np.int32)
    elem = np.tile(comp, n_mol)
    mol_off = (np.arange(n_mol + 1, dtype=np.int64) * comp.shape[0]).astype(np.int32)
    return elem, mol_off


def _y(seed: int, rows: int) -> np.ndarray:
    return _normal_f32(seed, TAG_Y, (rows,), std=1.0)


def make_workload(name: str, n_mol: Optional[int] = None, D: Optional[int] = None,
                  part: str = "train", with_grad: bool = True, T: int = 3,
                  n_atoms: Optional[int] = None, K: Optional[int] = None) -> Workload:
    """Build config `name` in ("c1".."c5").  `n_mol`, `D`, `n_atoms` (c5) and `K` (c5) shrink the
    case for parity tests; defaults are BASELINE.json's full sizes.  `part` selects c4's
    500-configuration training set or its 2000-configuration inference set (same model)."""
    name = name.lower()
    cfg = CONFIG_NAMES.index(name) + 1
    seed = _BASE_SEED + cfg
    part_id = {"train": 0, "infer": 1}[part]
    dseed = seed + 1000 * part_id          # data streams differ per part, model streams do not

    if name == "c1":
        d, DD, sigma = 64, D or 256, 2.0
        nm = n_mol or 16
        elem, mol_off = _fixed_topology(nm, [C_, C_, O_] + [H_] * 6)
        model = make_model(seed, d, DD, T, sigma)
        x = _x_around_mu(dseed, elem, None, d, 1.0)
        grad = _dense_grad(dseed, np.full(nm, 9), d, 0.1) if with_grad else None
        rows = nm + (3 * elem.shape[0] if with_grad else 0)
    elif name == "c2":
        d, DD, sigma = 128, D or 8192, 8.0
        nm = n_mol or 1000
        elem, mol_off = _fixed_topology(nm, [C_] * 9 + [O_] * 4 + [H_] * 8)
        model = make_model(seed, d, DD, T, sigma)
        x = _x_around_mu(dseed, elem, _mu(seed, d), d, 0.3)
        grad = _dense_grad(dseed, np.full(nm, 21), d, 0.05) if with_grad else None
        rows = nm + (3 * elem.shape[0] if with_grad else 0)
    elif name == "c3":
        d, DD, sigma = 128, D or 16384, 4.0
        nm = n_mol or 100_000
        rt = _rng(dseed, TAG_TOPO)
        counts = rt.integers(3, 30, size=nm).astype(np.int32)          # uniform 3..29
        mol_off = np.zeros(nm + 1, dtype=np.int32)
        np.cumsum(counts, out=mol_off[1:])
        elem = rt.choice(N_ELEM, size=int(mol_off[-1]), p=[0.51, 0.35, 0.06, 0.07, 0.01]).astype(np.int32)
        model = make_model(seed, d, DD, T, sigma)
        x = _x_around_mu(dseed, elem, _mu(seed, d), d, 1.0)
        grad = None
        rows = nm
    elif name == "c4":
        d, DD, sigma = 256, D or 16384, 16.0
        nm = n_mol or (500 if part == "train" else 2000)
        elem, mol_off = _fixed_topology(nm, [C_] * 12 + [N_] * 2 + [O_] + [H_] * 12)
        model = make_model(seed, d, DD, T, sigma)
        x = _x_around_mu(dseed, elem, _mu(seed, d), d, 0.5)
        grad = _dense_grad(dseed, np.full(nm, 27), d, 0.05) if with_grad else None
        rows = nm + (3 * elem.shape[0] if with_grad else 0)
    elif name == "c5":
        d, DD, sigma = 256, D or 32768, 8.0
        na = n_atoms or 16384
        KK = K or 48
        elem = np.where(np.arange(na) % 3 == 0, O_, H_).astype(np.int32)
        mol_off = np.array([0, na], dtype=np.int32)
        model = make_model(seed, d, DD, T, sigma)
        x = _x_around_mu(dseed, elem, _mu(seed, d), d, 1.0)
        grad = None
        if with_grad:
            nbr_idx = _rng(dseed, TAG_NBR).integers(0, na, size=(na, KK)).astype(np.int32)
            nbr_val = _normal_f32(dseed, TAG_GRAD, (na, KK, d, 3), std=0.05, block_rows=256)
            grad = DescriptorGradient(layout="neighbor", nbr_idx=nbr_idx, nbr_val=nbr_val, K=KK)
        rows = 1
    else:  # pragma: no cover
        raise ValueError(name)

    return Workload(name=name if part == "train" else f"{name}-{part}", model=model, elem=elem,
                    mol_off=mol_off, x=x, alpha=_alpha(seed, DD), y=_y(dseed, rows), grad=grad,
                    meta={"config": cfg, "seed": seed, "part": part})


def tiny_workload(seed: int, d: int, D: int, T: int, sigma: float, counts, n_elem: int = 3,
                  grad: Optional[str] = "dense", K: int = 4, x_std: float = 1.0, pad_fraction: float = 0.25) -> Workload:
    """Small free-form case for pins and edge-case parity: ragged molecules (counts may hold 0),
    random elements, dense or neighbour gradients (with -1 padding, self and duplicate indices)."""
    counts = np.asarray(counts, dtype=np.int32)
    mol_off = np.zeros(counts.shape[0] + 1, dtype=np.int32)
    np.cumsum(counts, out=mol_off[1:])
    na = int(mol_off[-1])
    elem = _rng(seed, TAG_TOPO).integers(0, n_elem, size=na).astype(np.int32)
    model = make_model(seed, d, D, T, sigma, n_elem=n_elem)
    x = _normal_f32(seed, TAG_X, (na, d), std=x_std)
    g = None
    if grad == "dense":
        g = _dense_grad(seed, counts, d, 0.1)
    elif grad == "neighbor":
        r = _rng(seed, TAG_NBR)
        idx = r.integers(0, max(na, 1), size=(na, K)).astype(np.int32)
        idx[r.random(size=(na, K)) < pad_fraction] = -1
        val = _normal_f32(seed, TAG_GRAD, (na, K, d, 3), std=0.1)
        g = DescriptorGradient(layout="neighbor", nbr_idx=idx, nbr_val=val, K=K)
    rows = counts.shape[0] + (3 * na if g is not None else 0)
    return Workload(name=f"tiny-{seed}", model=model, elem=elem, mol_off=mol_off, x=x,
                    alpha=_normal_f32(seed, TAG_ALPHA, (D,), std=float(1.0 / np.sqrt(D))),
                    y=_y(seed, rows), grad=g, meta={"seed": seed})


TAG_RHO, TAG_U, TAG_DRHO = 10, 11, 12


@dataclass
class ProjectionInputs:
    """Inputs of the per-element PCA projection (eq. 21-22): raw representations rho, the kept
    columns of every element's U_e, and (optionally) the dense gradient of rho.  Synthetic stand-ins for FCHL19
    vectors (rep of a few hundred, L179-230); U_e has orthonormal columns, as the left singular vectors of eq. 21."""
    rep: int
    d: int
    elem: np.ndarray                 # int32 [n_atoms]
    mol_off: np.ndarray              # int32 [n_mol + 1]
    rho: np.ndarray                  # float32 [n_atoms, rep]
    U: np.ndarray                    # float32 [n_elem, rep, d]
    drho: Optional[np.ndarray] = None        # float32 flat: molecule M holds [n, rep, n, 3]
    drho_off: Optional[np.ndarray] = None    # int64 [n_mol + 1]
    dx_off: Optional[np.ndarray] = None      # int64 [n_mol + 1]: offsets of the projected gradient [n, d, n, 3]


def projection_inputs(seed: int, counts, rep: int, d: int, n_elem: int = N_ELEM, with_grad: bool = False,
                      rho_std: float = 1.0, grad_std: float = 0.05) -> ProjectionInputs:
    counts = np.asarray(counts, dtype=np.int32)
    mol_off = np.zeros(counts.shape[0] + 1, dtype=np.int32)
    np.cumsum(counts, out=mol_off[1:])
    na = int(mol_off[-1])
    elem = _rng(seed, TAG_TOPO).integers(0, n_elem, size=na).astype(np.int32)
    rho = _normal_f32(seed, TAG_RHO, (na, rep), std=rho_std)
    U = np.empty((n_elem, rep, d), dtype=np.float32)
    for e in range(n_elem):        # orthonormal columns: QR of a Gaussian matrix (input generation, not the method)
        q, _ = np.linalg.qr(_rng(seed, TAG_U, e).standard_normal((rep, d)))
        U[e] = q.astype(np.float32)
    out = ProjectionInputs(rep=rep, d=d, elem=elem, mol_off=mol_off, rho=rho, U=U)
    if with_grad:
        c2 = counts.astype(np.int64) ** 2
        out.drho_off = np.zeros(counts.shape[0] + 1, dtype=np.int64)
        np.cumsum(3 * rep * c2, out=out.drho_off[1:])
        out.dx_off = np.zeros(counts.shape[0] + 1, dtype=np.int64)
        np.cumsum(3 * d * c2, out=out.dx_off[1:])
        out.drho = _normal_f32(seed, TAG_DRHO, (int(out.drho_off[-1]),), std=grad_std)
    return out
