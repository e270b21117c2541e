"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times: the CUDA path runs the
whole config; the FP64 oracle recomputes SAMPLED outputs one by one (selected molecules / atoms / matrix rows) and
properties that hold at any size.  Tolerances as in test_gpu_parity.py (north_star)."""
import numpy as np
import pytest

import oracle
from workloads import make_workload, Workload, DescriptorGradient

pytestmark = pytest.mark.gpu
TOL, TOL_F = 1e-5, 1e-4


def rel(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def q():
    import torch
    import paper_2206_01580_b200 as pkg
    from paper_2206_01580_b200 import workload_io
    pkg.load_library()
    yield pkg, workload_io, torch
    pkg.release_workspaces()
    torch.cuda.empty_cache()


def sub_molecules(w, mols):
    """The workload restricted to the molecules `mols` (inputs only: slicing, no arithmetic)."""
    mols = list(mols)
    atoms = np.concatenate([np.arange(w.mol_off[M], w.mol_off[M + 1]) for M in mols]).astype(np.int64)
    counts = np.array([w.mol_off[M + 1] - w.mol_off[M] for M in mols], dtype=np.int32)
    mol_off = np.zeros(len(mols) + 1, dtype=np.int32); np.cumsum(counts, out=mol_off[1:])
    grad = None
    if w.grad is not None and w.grad.layout == "dense":
        blocks = [w.grad.dense[w.grad.dense_off[M]:w.grad.dense_off[M + 1]] for M in mols]
        off = np.zeros(len(mols) + 1, dtype=np.int64); np.cumsum([b.size for b in blocks], out=off[1:])
        grad = DescriptorGradient(layout="dense", dense=np.concatenate(blocks), dense_off=off)
    return Workload(name=w.name + "-sub", model=w.model, elem=w.elem[atoms], mol_off=mol_off, x=w.x[atoms],
                    alpha=w.alpha, y=None, grad=grad), atoms


def check_gram_samples(A_host, y_host, ZtZ, Zty, rng, n_rows=4, n_cols=256, n_vec=2, all_diagonal=False):
    """Sampled parity of a full-size Gram matrix against the FP64 oracle, plus properties that hold at any size:
      * exact symmetry;
      * `n_rows` full rows (oracle.gram_rows) and Zty on those rows;
      * every entry among `n_cols` sampled columns (n_cols^2 entries: oracle.normal_equations on the column slice);
      * all D diagonal entries if asked (oracle.gram_entries);
      * ZtZ v = A^T (A v) for `n_vec` random vectors and tr ZtZ = |A|_F^2 (fp64 on the host)."""
    D = A_host.shape[1]
    ZtZn = ZtZ.cpu().numpy()
    for lo in range(0, D, 2048):                                         # exactly symmetric (blockwise: no D^2 temporaries)
        assert np.array_equal(ZtZn[lo:lo + 2048], ZtZn[:, lo:lo + 2048].T)
    rows = np.sort(rng.choice(D, size=n_rows, replace=False)).astype(np.int32)
    ref_rows, ref_y = oracle.gram_rows(A_host, y_host, rows)               # FP64 definition, row by row
    assert rel(ZtZn[rows], ref_rows) <= TOL
    if Zty is not None:
        assert rel(Zty.cpu().numpy()[rows], ref_y) <= TOL
    cols = np.sort(rng.choice(D, size=min(n_cols, D), replace=False))
    Asub = np.ascontiguousarray(A_host[:, cols])                           # slicing only
    ref_sub, ref_sub_y = oracle.normal_equations(Asub, y_host if y_host is not None else np.zeros(len(Asub), np.float32))
    assert rel(ZtZn[np.ix_(cols, cols)], ref_sub) <= TOL
    if Zty is not None:
        assert rel(Zty.cpu().numpy()[cols], ref_sub_y) <= TOL
    if all_diagonal:
        ii = np.arange(D, dtype=np.int32)
        assert rel(np.diagonal(ZtZn), oracle.gram_entries(A_host, ii, ii)) <= TOL
    # whole-matrix properties: ZtZ V = A^T (A V), trace = |A|_F^2 (fp64 on the host, row blocks)
    V = rng.standard_normal((D, n_vec))
    lhs = np.zeros((D, n_vec)); rhs = np.zeros((D, n_vec)); fro2 = 0.0
    for lo in range(0, D, 1024):
        lhs[lo:lo + 1024] = ZtZn[lo:lo + 1024].astype(np.float64) @ V
    for lo in range(0, A_host.shape[0], 4096):
        blk = A_host[lo:lo + 4096].astype(np.float64)
        rhs += blk.T @ (blk @ V)
        fro2 += float(np.sum(blk * blk))
    for k in range(n_vec):
        assert rel(lhs[:, k], rhs[:, k]) <= TOL
    assert abs(float(np.trace(ZtZn.astype(np.float64))) / fro2 - 1.0) <= TOL


def test_c2_full_step(q):
    """The step on config 2 at full size (1000 x 21 atoms, D = 8192, 64 000 rows), both operand containers."""
    pkg, wio, torch = q
    w = make_workload("c2")
    dp = wio.device_problem(w)
    n_mol, n_atoms, D = w.n_mol, w.n_atoms, w.model.D
    A = torch.empty((n_mol + 3 * n_atoms, D), dtype=torch.float32, device="cuda")
    Z, G = A[:n_mol], A[n_mol:]
    pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off, dp.grad, Z=Z, G=G)
    ZtZ, Zty = pkg.qmll_normal_equations(A, dp.y)
    E, F = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, dp.grad)
    torch.cuda.synchronize()
    rng = np.random.default_rng(2)
    mols = sorted(rng.choice(n_mol, size=8, replace=False).tolist())
    ws, atoms = sub_molecules(w, mols)
    assert rel(Z.cpu().numpy()[mols], oracle.forward_w(ws)) <= TOL
    rows = np.concatenate([3 * atoms + k for k in range(3)])
    rows.sort()
    assert rel(G.cpu().numpy()[rows], oracle.force_rows_w(ws)) <= TOL
    Eo, Fo = oracle.predict_w(ws)
    assert rel(E.cpu().numpy()[mols], Eo) <= TOL
    assert rel(F.cpu().numpy()[atoms], Fo) <= TOL_F
    Ah = A.cpu().numpy()
    check_gram_samples(Ah, w.y, ZtZ, Zty, rng, n_rows=8, n_cols=512, all_diagonal=True)
    ZtZ2, Zty2 = pkg.qmll_normal_equations(A, dp.y, mode=pkg.NE_SPLIT_TF32)
    torch.cuda.synchronize()
    check_gram_samples(Ah, w.y, ZtZ2, Zty2, rng, n_rows=2, n_cols=128)


def test_c3_full_100000_molecules(q):
    """Config 3 at full size (QM9-like: 100 000 ragged molecules of 3-29 atoms, D = 16384): forward on all of them,
    the 100 000-row normal equations (the longest accumulation on the path), energies-only predict.
    Oracle: 64 sampled molecules (Z, E); Gram: all 16 384 diagonal entries, 64 full rows, the 2^20 entries among
    1024 sampled columns, ZtZ V = A^T (A V) for 8 vectors."""
    pkg, wio, torch = q
    w = make_workload("c3")
    assert w.n_mol == 100000
    dp = wio.device_problem(w)
    Z = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off)
    E, _ = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha)
    ZtZ, Zty = pkg.qmll_normal_equations(Z, dp.y)
    torch.cuda.synchronize()
    rng = np.random.default_rng(3)
    mols = sorted(rng.choice(w.n_mol, size=64, replace=False).tolist())
    ws, _ = sub_molecules(w, mols)
    Zh = Z.cpu().numpy()
    Zo = oracle.forward_w(ws)
    assert rel(Zh[mols], Zo) <= TOL
    assert rel(E.cpu().numpy()[mols], oracle.energy(Zo, w.alpha)) <= TOL
    del Z
    pkg.release_workspaces()
    torch.cuda.empty_cache()
    check_gram_samples(Zh, w.y, ZtZ, Zty, rng, n_rows=64, n_cols=1024, n_vec=8, all_diagonal=True)


def test_c4_infer_predict_full(q):
    """Config 4 inference set at full size (2000 x 27 atoms, d = 256, D = 16384): 16 sampled molecules."""
    pkg, wio, torch = q
    w = make_workload("c4", part="infer")
    dp = wio.device_problem(w)
    E, F = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, dp.grad)
    torch.cuda.synchronize()
    rng = np.random.default_rng(4)
    mols = sorted(rng.choice(w.n_mol, size=16, replace=False).tolist())
    ws, atoms = sub_molecules(w, mols)
    Eo, Fo = oracle.predict_w(ws)
    assert rel(E.cpu().numpy()[mols], Eo) <= TOL
    assert rel(F.cpu().numpy()[atoms], Fo) <= TOL_F


def test_c4_train_full_step(q):
    """Config 4 training set at full size (500 x 27 atoms, d = 256, D = 16384, 41 000 rows): Z, G on sampled
    molecules against the oracle, and the normal equations of all 41 000 rows on sampled rows / columns."""
    pkg, wio, torch = q
    w = make_workload("c4")
    dp = wio.device_problem(w)
    n_mol, n_atoms, D = w.n_mol, w.n_atoms, w.model.D
    A = torch.empty((n_mol + 3 * n_atoms, D), dtype=torch.float32, device="cuda")
    Z, G = A[:n_mol], A[n_mol:]
    pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off, dp.grad, Z=Z, G=G)
    ZtZ, Zty = pkg.qmll_normal_equations(A, dp.y)
    torch.cuda.synchronize()
    mols = [7, 311, 402]
    ws, atoms = sub_molecules(w, mols)
    assert rel(Z.cpu().numpy()[mols], oracle.forward_w(ws)) <= TOL
    rows = np.sort(np.concatenate([3 * atoms + k for k in range(3)]))
    assert rel(G[torch.from_numpy(rows).cuda()].cpu().numpy(), oracle.force_rows_w(ws)) <= TOL
    check_gram_samples(A.cpu().numpy(), w.y, ZtZ, Zty, np.random.default_rng(44), n_rows=4, n_cols=256)


def test_c5_full_cell_against_oracle(q):
    """Config 5 at full size (one 16 384-atom cell, D = 32768, 48 neighbours per atom): Z (1 x 32768), the energy and
    ALL forces [16384, 3] element by element against the FP64 oracle run on the whole cell."""
    pkg, wio, torch = q
    w = make_workload("c5")
    assert w.n_atoms == 16384 and w.n_mol == 1
    dp = wio.device_problem(w)
    E, F = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, dp.grad)
    Z = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off)
    F2 = pkg.qmll_sorf_backward_forces(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, dp.grad)
    torch.cuda.synchronize()
    Zo = oracle.forward_w(w)
    assert rel(Z.cpu().numpy(), Zo) <= TOL
    assert rel(E.cpu().numpy(), oracle.energy(Zo, w.alpha)) <= TOL
    Fo = oracle.forces_w(w)
    assert rel(F.cpu().numpy(), Fo) <= TOL_F
    assert rel(F2.cpu().numpy(), Fo) <= TOL_F


def test_solve_at_the_bench_size(q):
    """qmll_solve at D = 16384 (the step's normal equations; the oracle's unblocked Cholesky would need ~1e12 flops on
    the host).  Properties that hold at any size: the FP64 residual of the fp32 alpha is at the fp32 rounding level,
    and alpha agrees with a library FP64 solve (torch.linalg, cuSOLVER) of the same system."""
    pkg, wio, torch = q
    D = 16384
    g = torch.Generator(device="cuda").manual_seed(7)
    A = torch.randn((D + 512, D), device="cuda", generator=g) / D ** 0.5
    ZtZ = A.T @ A
    del A
    Zty = torch.randn((D,), device="cuda", generator=g)
    lam = 1e-3
    alpha, info = pkg.qmll_solve(ZtZ, Zty, lam)
    assert int(info.item()) == 0
    M = torch.tril(ZtZ.double())
    M = M + torch.tril(M, -1).T                         # the symmetric matrix the solve reads (lower triangle)
    M.diagonal().add_(lam)
    res = (M @ alpha.double() - Zty.double()).norm() / Zty.double().norm()
    assert float(res) <= 1e-5
    ref = torch.linalg.solve(M, Zty.double())
    assert float((alpha.double() - ref).norm() / ref.norm()) <= 1e-6
