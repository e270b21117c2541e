"""Seeded synthetic geometries for the FCHL19 representation (PAPER.md section E; Table I).

The paper evaluates on molecules (MD17, QM9) and on periodic cells (liquid water, a MOF; Table V); none of
those structures is available, so these stand in for them: atoms on a jittered cubic lattice at a liquid-like number
density, elements drawn with stated probabilities (or a fixed water-like pattern), and the neighbour list inside
r_cut.  The neighbour list (and, for periodic cells, the image shifts) is INPUT to both the oracle and the GPU library
-- building it is the caller's job on both sides (tiled neighbour list / minimum image are out
of scope).  Nothing here evaluates any term of the representation.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np

from .configs import _rng

TAG_POS, TAG_GELEM = 20, 21


@dataclass
class FchlParams:
    """Table I (L248-260), column E + F, with r_cut as an argument (the paper uses 6.0)."""
    n_elem: int = 5
    n2: int = 24
    n3: int = 20
    eta2: float = 0.32
    eta3: float = 2.7
    N2: float = 1.8
    N3: float = 0.57
    c3: float = 13.4
    zeta: float = float(np.pi)
    r_cut: float = 6.0

    @property
    def rep(self) -> int:
        return self.n_elem * self.n2 + self.n_elem * (self.n_elem + 1) * self.n3


FCHL_E = dict(n2=23, n3=22, eta2=0.27, eta3=5.6, N2=2.78, N3=2.1, c3=60.1)      # Table I, column E


@dataclass
class Geometry:
    r: np.ndarray                      # float32 [n_atoms, 3]
    elem: np.ndarray                   # int32 [n_atoms]
    mol_off: np.ndarray                # int32 [n_mol + 1]
    nbr_idx: np.ndarray                # int32 [n_atoms, K], -1 = padding
    nbr_shift: Optional[np.ndarray]    # float32 [n_atoms, K, 3] (periodic image offset) or None
    box: Optional[float] = None


def _lattice(seed: int, n_side: int, spacing: float, jitter: float) -> np.ndarray:
    g = np.stack(np.meshgrid(*([np.arange(n_side)] * 3), indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float64)
    g = g * spacing + _rng(seed, TAG_POS).uniform(-jitter, jitter, size=g.shape)
    return g


def _neighbours(pos: np.ndarray, groups: np.ndarray, r_list: float, K: Optional[int], box: Optional[float]):
    """All pairs closer than r_list: same group only (isolated molecules, brute force per group) when box is None, else
    every periodic image (one per pair since box > 2 r_list; k-d tree with periodic boundaries).  Neighbours of an atom
    are listed by increasing index j.  Returns idx [n, K] (-1 = padding) and the image shifts [n, K, 3] (or None)."""
    n = pos.shape[0]
    rows = [[] for _ in range(n)]
    if box is None:
        for gid in np.unique(groups):
            members = np.nonzero(groups == gid)[0]
            p = pos[members]
            d2 = ((p[:, None, :] - p[None, :, :]) ** 2).sum(-1)
            for a, row in zip(members, d2):
                rows[a] = [int(members[b]) for b in np.nonzero(row < r_list * r_list)[0] if members[b] != a]
    else:
        from scipy.spatial import cKDTree
        wrapped = np.mod(pos, box)
        tree = cKDTree(wrapped, boxsize=box)
        for a, lst in enumerate(tree.query_ball_point(wrapped, r_list)):
            rows[a] = sorted(int(b) for b in lst if b != a)
    kmax = max((len(x) for x in rows), default=0)
    K = kmax if K is None else K
    if kmax > K:
        raise ValueError(f"an atom has {kmax} neighbours inside the list radius, more than K = {K}")
    idx = np.full((n, K), -1, dtype=np.int32)
    for a in range(n):
        idx[a, :len(rows[a])] = rows[a]
    if box is None:
        return idx, None
    sh = np.zeros((n, K, 3), dtype=np.float32)
    valid = idx >= 0
    delta = pos[np.where(valid, idx, 0)] - pos[:, None, :]            # r_j - r_i without images
    sh[valid] = (-np.round(delta / box) * box)[valid].astype(np.float32)
    return idx, sh


def molecules_geometry(seed: int, counts, n_elem: int = 5, spacing: float = 1.45, jitter: float = 0.25,
                       r_list: float = 6.0, K: Optional[int] = None, probs=None) -> Geometry:
    """Isolated molecules: molecule M is a compact jittered-lattice cluster of counts[M] atoms; the neighbour list
    holds every other atom of the same molecule closer than r_list."""
    counts = np.asarray(counts, dtype=np.int32)
    mol_off = np.zeros(counts.shape[0] + 1, dtype=np.int32)
    np.cumsum(counts, out=mol_off[1:])
    na = int(mol_off[-1])
    pos = np.zeros((na, 3))
    groups = np.zeros(na, dtype=np.int64)
    for M, n in enumerate(counts):
        side = int(np.ceil(n ** (1.0 / 3.0)))
        g = _lattice(seed * 1000 + M, side, spacing, jitter)
        order = np.argsort(((g - g.mean(0)) ** 2).sum(1), kind="stable")[:n]     # the n sites nearest the centre
        pos[mol_off[M]:mol_off[M + 1]] = g[order] + 20.0 * M                      # molecules far apart
        groups[mol_off[M]:mol_off[M + 1]] = M
    probs = np.full(n_elem, 1.0 / n_elem) if probs is None else np.asarray(probs, dtype=np.float64)
    elem = _rng(seed, TAG_GELEM).choice(n_elem, size=na, p=probs / probs.sum()).astype(np.int32)
    r32 = pos.astype(np.float32)
    idx, _ = _neighbours(r32.astype(np.float64), groups, r_list, K, None)
    return Geometry(r=r32, elem=elem, mol_off=mol_off, nbr_idx=idx, nbr_shift=None)


def cell_geometry(seed: int, n_side: int, spacing: float = 2.15, jitter: float = 0.35, r_list: float = 4.4,
                  K: Optional[int] = None, water_like: bool = True, n_elem: int = 5) -> Geometry:
    """One periodic cubic cell of n_side^3 atoms (box = n_side * spacing; ~0.1 atoms / A^3 like liquid water);
    elements O (3) if I % 3 == 0 else H (0) when water_like.  Neighbours: every periodic image closer than r_list
    (requires box > 2 r_list)."""
    box = n_side * spacing
    if box <= 2 * r_list:
        raise ValueError("box must exceed 2 r_list (one image per pair)")
    pos = _lattice(seed, n_side, spacing, jitter)
    na = pos.shape[0]
    if water_like:
        elem = np.where(np.arange(na) % 3 == 0, 3, 0).astype(np.int32)
    else:
        elem = _rng(seed, TAG_GELEM).integers(0, n_elem, size=na).astype(np.int32)
    r32 = pos.astype(np.float32)
    idx, sh = _neighbours(r32.astype(np.float64), np.zeros(na, dtype=np.int64), r_list, K, box)
    return Geometry(r=r32, elem=elem, mol_off=np.array([0, na], dtype=np.int32), nbr_idx=idx, nbr_shift=sh, box=box)
