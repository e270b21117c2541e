"""GPU parity of SURVEY.md section 8(f) #4 (variants): the feature map on the tensor cores -- qmll_sorf_forward_mma
(SORF with the chain of every stack expanded into its integer matrix) and qmll_rff_forward (dense-matrix random Fourier
features, eq. 12-14, 18) -- against the FP64 oracle.  Tolerance: relative Frobenius error <= 1e-5 for Z."""
import numpy as np
import pytest

import oracle
from workloads import make_workload, tiny_workload

pytestmark = pytest.mark.gpu

TOL = 1e-5


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / den) if den > 0 else float(np.linalg.norm(a))


@pytest.fixture(scope="module")
def q():
    import torch
    import paper_2206_01580_b200 as pkg
    from paper_2206_01580_b200 import workload_io
    pkg.load_library()
    assert torch.cuda.is_available()
    return pkg, workload_io, torch


@pytest.mark.parametrize("d,D,T,counts,n_elem", [
    (128, 512, 3, [5, 3, 0, 7], 3),              # one feature group, an empty molecule
    (128, 1280, 3, [21] * 9 + [1, 2], 5),        # 10 stacks: feature-group tail (4 + 4 + 2), several atom tiles
    (128, 640, 2, [29, 3, 17, 40, 11], 4),       # T = 2
    (128, 384, 1, [70, 90], 2),                  # molecules longer than an atom tile (runs cross tile borders)
    (256, 1024, 3, [27] * 8, 4),                 # d = 256: 96-atom tiles
    (256, 768, 3, [100, 5, 130], 1),             # one element, odd number of stacks
    (128, 256, 3, [3] * 50, 16),                 # 16 elements: mostly padded tiles
])
def test_sorf_forward_mma_matches_oracle(q, d, D, T, counts, n_elem):
    pkg, wio, torch = q
    w = tiny_workload(seed=100 + d + D, d=d, D=D, T=T, sigma=4.0, counts=counts, n_elem=n_elem, grad=None)
    dp = wio.device_problem(w)
    Z = pkg.qmll_sorf_forward_mma(dp.params, dp.x, dp.elem, dp.mol_off)
    torch.cuda.synchronize()
    Zo = oracle.forward_w(w)
    assert rel(Z.cpu().numpy(), Zo) <= TOL
    # and the register-FWHT path gives the same Z
    Z2 = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off)
    assert rel(Z.cpu().numpy(), Z2.cpu().numpy()) <= TOL


def test_sorf_forward_mma_large_inputs_and_unsupported_shapes(q):
    pkg, wio, torch = q
    # descriptor values far outside fp16's range: the per-tile power-of-two scale keeps the split exact enough
    w = tiny_workload(seed=7, d=128, D=512, T=3, sigma=3.0e5, counts=[9, 12], n_elem=2, grad=None)
    w.x *= np.float32(1.0e5)
    dp = wio.device_problem(w)
    Z = pkg.qmll_sorf_forward_mma(dp.params, dp.x, dp.elem, dp.mol_off)
    assert rel(Z.cpu().numpy(), oracle.forward_w(w)) <= TOL
    w64 = tiny_workload(seed=8, d=64, D=256, T=3, sigma=2.0, counts=[4], n_elem=2, grad=None)
    dp = wio.device_problem(w64)
    with pytest.raises(pkg.QmllError):
        pkg.qmll_sorf_forward_mma(dp.params, dp.x, dp.elem, dp.mol_off)
    # no atoms: Z is zero
    w0 = tiny_workload(seed=9, d=128, D=256, T=3, sigma=2.0, counts=[0, 0], n_elem=2, grad=None)
    dp = wio.device_problem(w0)
    Z = pkg.qmll_sorf_forward_mma(dp.params, dp.x, dp.elem, dp.mol_off)
    assert Z.shape == (2, 256) and float(Z.abs().max()) == 0.0


@pytest.mark.parametrize("d,D,counts,n_elem,sigma", [
    (128, 512, [5, 3, 0, 7], 3, 4.0),
    (128, 1000, [21] * 7, 5, 8.0),               # D not a multiple of 128: masked tail rows
    (256, 640, [27] * 5 + [1], 4, 16.0),
    (256, 128, [200], 1, 6.0),
])
def test_rff_forward_matches_oracle(q, d, D, counts, n_elem, sigma):
    pkg, wio, torch = q
    rng = np.random.default_rng(d + D)
    w = tiny_workload(seed=200 + d + D, d=d, D=d * ((D + d - 1) // d), T=1, sigma=sigma, counts=counts, n_elem=n_elem,
                      grad=None)
    W = (rng.standard_normal((n_elem, D, d)) / sigma).astype(np.float32)
    b = rng.uniform(0, 2 * np.pi, size=(n_elem, D)).astype(np.float32)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Z = pkg.qmll_rff_forward(t(W), t(b), t(w.x), t(w.elem), t(w.mol_off))
    torch.cuda.synchronize()
    Zo = oracle.rff_forward(W, b, w.x, w.elem, w.mol_off)
    assert rel(Z.cpu().numpy(), Zo) <= TOL


def test_rff_with_the_dense_sorf_matrix_reproduces_sorf(q):
    """The chain tying the variants together on the GPU: W built from the oracle's u on unit vectors (the explicit SORF
    matrix) through qmll_rff_forward == qmll_sorf_forward == qmll_sorf_forward_mma."""
    pkg, wio, torch = q
    w = tiny_workload(seed=31, d=128, D=256, T=3, sigma=2.5, counts=[6, 9], n_elem=2, grad=None)
    m = w.model
    eye = np.eye(128, dtype=np.float32)
    W = np.stack([np.stack([oracle.sorf_u(eye[j], e, m.d, m.D, m.T, m.sigma, m.signs) for j in range(128)], axis=1)
                  for e in range(2)]).astype(np.float32)                     # [n_elem, D, d]
    dp = wio.device_problem(w)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    Zr = pkg.qmll_rff_forward(t(W), dp.params.bias, dp.x, dp.elem, dp.mol_off).cpu().numpy()
    Zo = oracle.forward_w(w)
    assert rel(Zr, Zo) <= TOL
    assert rel(pkg.qmll_sorf_forward_mma(dp.params, dp.x, dp.elem, dp.mol_off).cpu().numpy(), Zo) <= TOL


@pytest.mark.parametrize("n_mol,D", [(1, 4), (7, 130), (33, 1024), (300, 8192), (5, 3)])
def test_energies_from_z_matches_oracle(q, n_mol, D):
    """qmll_energies (step a4 on a given Z, eq. 15) against the oracle's FP64 product; odd D takes the scalar path."""
    pkg, wio, torch = q
    rng = np.random.default_rng(n_mol + D)
    Z = rng.standard_normal((n_mol, D)).astype(np.float32)
    alpha = (rng.standard_normal(D) / np.sqrt(D)).astype(np.float32)
    E = pkg.qmll_energies(torch.from_numpy(Z).cuda(), torch.from_numpy(alpha).cuda())
    torch.cuda.synchronize()
    assert rel(E.cpu().numpy(), oracle.energy(Z, alpha)) <= TOL
    assert pkg.qmll_energies(torch.empty((0, D), device="cuda"), torch.from_numpy(alpha).cuda()).shape == (0,)


def test_feature_map_plus_energies_is_the_energy_only_prediction(q):
    """Tensor-core feature map + qmll_energies = energies of qmll_predict, against the oracle (config 2 shape, 200
    molecules) -- the energies-only prediction of the f4 variants."""
    pkg, wio, torch = q
    w = make_workload("c2", n_mol=200, with_grad=False)
    dp = wio.device_problem(w)
    E = pkg.qmll_energies(pkg.qmll_sorf_forward_mma(dp.params, dp.x, dp.elem, dp.mol_off), dp.alpha)
    E_fwht, _ = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha)
    torch.cuda.synchronize()
    Eo = oracle.energy(oracle.forward_w(w), w.alpha)
    assert rel(E.cpu().numpy(), Eo) <= TOL and rel(E_fwht.cpu().numpy(), Eo) <= TOL


def test_sorf_forward_mma_fullsize_c3(q):
    """Config 3 at full size (100 000 molecules, 1.6 M atoms, D = 16384) in the launch configuration bench.py times
    (configs.c3.forward_mma_ms): 64 sampled molecules against the oracle, all of Z against the register-FWHT path."""
    pkg, wio, torch = q
    w = make_workload("c3")
    dp = wio.device_problem(w)
    Z = pkg.qmll_sorf_forward_mma(dp.params, dp.x, dp.elem, dp.mol_off)
    torch.cuda.synchronize()
    rng = np.random.default_rng(11)
    mols = np.sort(rng.choice(w.n_mol, size=64, replace=False))
    m = w.model
    for M in mols:
        a0, a1 = int(w.mol_off[M]), int(w.mol_off[M + 1])
        Zo = oracle.forward(w.x[a0:a1], w.elem[a0:a1], np.array([0, a1 - a0], dtype=np.int32), m.d, m.D, m.T, m.sigma,
                            m.signs, m.bias)
        assert rel(Z[int(M)].cpu().numpy(), Zo[0]) <= TOL
    Z2 = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off)
    num = float((Z - Z2).double().norm())
    den = float(Z2.double().norm())
    assert num / den <= TOL
    # energies of all 100 000 molecules from this Z: the sampled ones against the oracle, all against qmll_predict
    E = pkg.qmll_energies(Z, dp.alpha)
    E_fwht, _ = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha)
    torch.cuda.synchronize()
    Eo = oracle.energy(Z[torch.from_numpy(mols).cuda()].cpu().numpy(), w.alpha)
    assert rel(E.cpu().numpy()[mols], Eo) <= TOL
    assert float((E - E_fwht).double().norm() / E_fwht.double().norm()) <= TOL


def test_sorf_forward_mma_offsets_beyond_31_bits(q):
    """n_mol * D > 2^31: the per-run table then holds molecule indices instead of Z offsets (64-bit addressing in the
    epilogue).  131 073 one- and two-atom molecules, D = 16384; all of Z against the FWHT path, samples against the oracle."""
    pkg, wio, torch = q
    n_mol = 131073
    counts = [1 + (i % 2) for i in range(n_mol)]
    w = tiny_workload(seed=77, d=128, D=16384, T=3, sigma=5.0, counts=counts, n_elem=3, grad=None)
    assert n_mol * 16384 > 2 ** 31
    dp = wio.device_problem(w)
    Z = pkg.qmll_sorf_forward_mma(dp.params, dp.x, dp.elem, dp.mol_off)
    Z2 = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off)
    torch.cuda.synchronize()
    assert float((Z - Z2).double().norm() / Z2.double().norm()) <= TOL
    m = w.model
    for M in (0, 1, 65536, 131071, 131072):
        a0, a1 = int(w.mol_off[M]), int(w.mol_off[M + 1])
        Zo = oracle.forward(w.x[a0:a1], w.elem[a0:a1], np.array([0, a1 - a0], dtype=np.int32), m.d, m.D, m.T, m.sigma,
                            m.signs, m.bias)
        assert rel(Z[M].cpu().numpy(), Zo[0]) <= TOL
