"""GPU parity of SURVEY.md section 8(f) #3: qmll_fchl19 (representation + Jacobian, eq. 23-33) and
qmll_project_neighbor against the FP64 oracle on the same seeded geometries, and the chain
coordinates -> qmll_fchl19 -> qmll_project / qmll_project_neighbor -> qmll_predict against the oracle's chain.

Tolerances: relative Frobenius error <= 1e-5 for rho and the projected descriptor, <= 1e-4 for
the Jacobian and the forces (fp32 kernels against FP64); jac_idx is integer work and must match exactly.
"""
from dataclasses import replace

import numpy as np
import pytest

import oracle
from workloads import FCHL_E, FchlParams, cell_geometry, make_model, molecules_geometry, projection_inputs

pytestmark = pytest.mark.gpu

TOL, TOL_J = 1e-5, 1e-4


def rel(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    den = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / den) if den > 0 else float(np.linalg.norm(a))


@pytest.fixture(scope="module")
def q():
    import torch
    import paper_2206_01580_b200 as pkg
    pkg.load_library()
    assert torch.cuda.is_available()
    return pkg, torch


def dev_params(pkg, fp):
    return pkg.Fchl19Params(n_elem=fp.n_elem, n2=fp.n2, n3=fp.n3, eta2=fp.eta2, eta3=fp.eta3, two_body_decay=fp.N2,
                            three_body_decay=fp.N3, three_body_weight=fp.c3, zeta=fp.zeta, r_cut=fp.r_cut)


def run_gpu(q, fp, g, jacobian=True):
    pkg, torch = q
    t = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()
    out = pkg.qmll_fchl19(dev_params(pkg, fp), t(g.r), t(g.elem), t(g.nbr_idx), t(g.nbr_shift), jacobian=jacobian)
    torch.cuda.synchronize()
    return out


def expected_jac_idx(fp, g):
    """slot 0 = the atom; slot 1 + q = nbr_idx[i, q] if that image is inside r_cut, else -1 (fp32 distances, as the
    kernel decides; atoms within 1e-4 of r_cut are excluded from the exact comparison by the caller)."""
    n, K = g.nbr_idx.shape
    ri = g.r.astype(np.float64)
    img = ri[np.where(g.nbr_idx >= 0, g.nbr_idx, 0)] + (0 if g.nbr_shift is None else g.nbr_shift.astype(np.float64))
    dist = np.linalg.norm(img - ri[:, None, :], axis=2)
    inside = (g.nbr_idx >= 0) & (dist < fp.r_cut)
    edge = (g.nbr_idx >= 0) & (np.abs(dist - fp.r_cut) < 1e-4)
    idx = np.concatenate([np.arange(n, dtype=np.int32)[:, None], np.where(inside, g.nbr_idx, -1)], axis=1)
    return idx, np.concatenate([np.zeros((n, 1), bool), edge], axis=1)


def check_against_oracle(q, fp, g, atoms=None):
    rho, jac_idx, jac_val, info = run_gpu(q, fp, g)
    assert int(info.item()) == 0
    rho_o = oracle.fchl19(fp, g.r, g.elem, g.nbr_idx, g.nbr_shift)
    assert rel(rho.cpu().numpy(), rho_o) <= TOL
    idx_o, edge = expected_jac_idx(fp, g)
    got = jac_idx.cpu().numpy()
    assert np.array_equal(got[~edge], idx_o[~edge])
    atoms = np.arange(g.r.shape[0]) if atoms is None else np.asarray(atoms)
    J_o = oracle.fchl19_jacobian(fp, g.r, g.elem, g.nbr_idx, g.nbr_shift, atoms=atoms)
    J = jac_val[torch_index(q, atoms)].cpu().numpy()
    assert rel(J, J_o) <= TOL_J
    # blocks of slots without a neighbour are exactly zero
    dead = got[atoms] < 0
    assert np.all(J[dead] == 0)
    # representation only (no Jacobian) gives the same rho
    rho2, a, b, _ = run_gpu(q, fp, g, jacobian=False)
    assert a is None and b is None
    assert rel(rho2.cpu().numpy(), rho_o) <= TOL
    return rel(rho.cpu().numpy(), rho_o), rel(J, J_o)


def torch_index(q, atoms):
    return q[1].from_numpy(np.asarray(atoms, dtype=np.int64)).cuda()


@pytest.mark.parametrize("which", ["E+F", "E"])
def test_fchl19_molecules(q, which):
    fp = FchlParams() if which == "E+F" else replace(FchlParams(), **FCHL_E)
    g = molecules_geometry(11, [1, 2, 3, 5, 9, 21, 27, 40], probs=[0.45, 0.35, 0.07, 0.1, 0.03])
    e_rho, e_jac = check_against_oracle(q, fp, g)
    print(f"fchl19 molecules ({which}): rho {e_rho:.2e} jacobian {e_jac:.2e}")


def test_fchl19_periodic_cell_with_image_shifts(q):
    fp = replace(FchlParams(), r_cut=3.6)
    g = cell_geometry(12, 6, spacing=2.0, jitter=0.35, r_list=3.9)       # list radius > r_cut: some slots are outside
    assert (np.abs(g.nbr_shift) > 0).any()
    e_rho, e_jac = check_against_oracle(q, fp, g)
    print(f"fchl19 cell 216 atoms: rho {e_rho:.2e} jacobian {e_jac:.2e}")


def test_fchl19_small_element_sets_and_grids(q):
    for n_elem, n2, n3 in ((1, 5, 3), (2, 32, 32), (7, 9, 11)):
        fp = replace(FchlParams(), n_elem=n_elem, n2=n2, n3=n3, r_cut=4.5)
        g = molecules_geometry(13 + n_elem, [4, 11, 18], n_elem=n_elem)
        check_against_oracle(q, fp, g)


def test_fchl19_edge_cases(q):
    pkg, torch = q
    fp = FchlParams()
    # no neighbour columns at all; an empty system
    g = molecules_geometry(5, [1, 1, 1])
    assert g.nbr_idx.shape[1] == 0
    rho, jac_idx, jac_val, info = run_gpu(q, fp, g)
    assert np.all(rho.cpu().numpy() == 0) and jac_val.shape == (3, 1, fp.rep, 3) and np.all(jac_val.cpu().numpy() == 0)
    assert jac_idx.cpu().numpy().ravel().tolist() == [0, 1, 2]
    g0 = replace(g, r=g.r[:0], elem=g.elem[:0], nbr_idx=g.nbr_idx[:0])
    rho, _, _, _ = run_gpu(q, fp, g0)
    assert rho.shape == (0, fp.rep)
    # more neighbours inside r_cut than the kernel holds: reported through info
    dense = cell_geometry(3, 8, spacing=1.0, jitter=0.1, r_list=3.6)
    assert (dense.nbr_idx >= 0).sum(1).max() > 160
    _, _, _, info = run_gpu(q, replace(fp, r_cut=3.6), dense, jacobian=False)
    assert int(info.item()) > 0
    # host-side argument checks
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    with pytest.raises(pkg.QmllError):
        pkg.qmll_fchl19(dev_params(pkg, replace(fp, n3=40)), t(g.r), t(g.elem), t(g.nbr_idx))
    with pytest.raises(pkg.QmllError):
        pkg.qmll_fchl19(dev_params(pkg, replace(fp, r_cut=0.0)), t(g.r), t(g.elem), t(g.nbr_idx))


def test_project_neighbor_matches_oracle(q):
    pkg, torch = q
    rng = np.random.default_rng(3)
    for n_atoms, S, rep, d, E in ((7, 4, 37, 16, 3), (33, 13, 720, 128, 5), (5, 23, 496, 256, 4)):
        gin = rng.normal(size=(n_atoms, S, rep, 3)).astype(np.float32)
        U = rng.normal(size=(E, rep, d)).astype(np.float32)
        elem = rng.integers(0, E, size=n_atoms).astype(np.int32)
        idx = rng.integers(-1, 5, size=(n_atoms, S)).astype(np.int32)
        ref = oracle.project_neighbor_gradient(gin, elem, U)
        out = pkg.qmll_project_neighbor(torch.from_numpy(gin).cuda(), torch.from_numpy(elem).cuda(), torch.from_numpy(U).cuda())
        assert rel(out.cpu().numpy(), ref) <= TOL
        out = pkg.qmll_project_neighbor(torch.from_numpy(gin).cuda(), torch.from_numpy(elem).cuda(), torch.from_numpy(U).cuda(),
                                        idx=torch.from_numpy(idx).cuda()).cpu().numpy()
        ref[idx < 0] = 0
        assert rel(out, ref) <= TOL and np.all(out[idx < 0] == 0)


def test_chain_coordinates_to_forces(q):
    """r -> FCHL19 (+ Jacobian) -> per-element projection -> SORF energy and forces, every step on the GPU, against
    the oracle's chain (whose force is pinned by finite differences of E(r) in tests/test_fchl19_pins.py)."""
    pkg, torch = q
    fp = FchlParams()
    g = molecules_geometry(21, [9, 21, 27], probs=[0.5, 0.35, 0.05, 0.1, 0.0])
    d, D = 128, 1024
    model = make_model(77, d=d, D=D, T=3, sigma=3.0)
    pi = projection_inputs(seed=78, counts=[1], rep=fp.rep, d=d)
    alpha = (np.random.default_rng(79).normal(size=D) / np.sqrt(D)).astype(np.float32)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    # GPU chain
    rho, jac_idx, jac_val, info = pkg.qmll_fchl19(dev_params(pkg, fp), t(g.r), t(g.elem), t(g.nbr_idx), jacobian=True)
    x, _ = pkg.qmll_project(rho, t(g.elem), t(pi.U))
    dx = pkg.qmll_project_neighbor(jac_val, t(g.elem), t(pi.U), idx=jac_idx)
    params = pkg.SorfParams(d=d, D=D, n_transform=3, n_elem=5, sigma=3.0, signs=t(model.signs), bias=t(model.bias))
    E, F = pkg.qmll_predict(params, x, t(g.elem), t(g.mol_off), t(alpha), pkg.Grad.make_neighbor(jac_idx, dx))
    torch.cuda.synchronize()
    # oracle chain (its own FP64 intermediates, rounded to fp32 where its interfaces take fp32)
    rho_o = oracle.fchl19(fp, g.r, g.elem, g.nbr_idx)
    J_o = oracle.fchl19_jacobian(fp, g.r, g.elem, g.nbr_idx)
    x_o = oracle.project(rho_o.astype(np.float32), g.elem, pi.U)
    dx_o = oracle.project_neighbor_gradient(J_o.astype(np.float32), g.elem, pi.U)
    idx_o, _ = expected_jac_idx(fp, g)
    Z_o = oracle.forward(x_o.astype(np.float32), g.elem, g.mol_off, d, D, 3, 3.0, model.signs, model.bias)
    E_o = oracle.energy(Z_o, alpha)
    g_o = oracle.backward_g(x_o.astype(np.float32), g.elem, d, D, 3, 3.0, model.signs, model.bias, alpha)
    F_o = oracle.forces_neighbor(g_o, d, idx_o, dx_o.astype(np.float32))
    assert rel(x.cpu().numpy(), x_o) <= TOL
    assert rel(E.cpu().numpy(), E_o) <= TOL
    assert rel(F.cpu().numpy(), F_o) <= TOL_J


def test_fchl19_fullsize_periodic_cell_15625_atoms(q):
    """The launch configuration bench.py times (configs.fchl19_cell): 25^3-atom water-like periodic cell, r_cut 4.8,
    K = 64, Table I parameters.  Sampled atoms against the oracle; properties that hold at any size on all atoms:
    translation sum rule of the Jacobian, zero blocks exactly where jac_idx is negative, jac_idx itself."""
    pkg, torch = q
    fp = replace(FchlParams(), r_cut=4.8)
    g = cell_geometry(2, 25, r_list=4.8, K=64)
    rho, jac_idx, jac_val, info = run_gpu(q, fp, g)
    assert int(info.item()) == 0 and rho.shape == (15625, 720) and jac_val.shape == (15625, 65, 720, 3)
    rng = np.random.default_rng(17)
    atoms = np.sort(rng.choice(15625, size=48, replace=False))
    sub_idx = g.nbr_idx[atoms]
    # oracle on the sampled atoms only: a reduced problem with the same images (positions of all atoms are needed)
    ro = np.stack([oracle.fchl19_atom(fp, g.r[i].astype(np.float64),
                                      g.r[sub_idx[t][sub_idx[t] >= 0]].astype(np.float64) + g.nbr_shift[i][sub_idx[t] >= 0],
                                      g.elem[sub_idx[t][sub_idx[t] >= 0]]) for t, i in enumerate(atoms)])
    assert rel(rho[torch_index(q, atoms)].cpu().numpy(), ro) <= TOL
    J_o = oracle.fchl19_jacobian(fp, g.r, g.elem, g.nbr_idx, g.nbr_shift, atoms=atoms[:12])
    assert rel(jac_val[torch_index(q, atoms[:12])].cpu().numpy(), J_o) <= TOL_J
    idx_o, edge = expected_jac_idx(fp, g)
    got = jac_idx.cpu().numpy()
    assert np.array_equal(got[~edge], idx_o[~edge])
    # whole-output properties (device-side reductions; no oracle needed)
    tot = jac_val.sum(dim=1)                                         # [n, rep, 3]: translation invariance
    scale = jac_val.abs().amax(dim=(1, 2, 3))                        # per atom
    assert float((tot.abs().amax(dim=(1, 2)) / scale).max()) < 2e-5
    dead = jac_idx < 0
    assert float(jac_val[dead].abs().max()) == 0.0
    assert bool(torch.isfinite(rho).all()) and bool(torch.isfinite(jac_val).all())


def _backward_chain_gpu(q, fp, g, model, U, alpha):
    """coordinates -> forces without a Jacobian: fchl19 -> project -> backward_g -> project_back -> fchl19_backward."""
    pkg, torch = q
    t = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()
    dfp = dev_params(pkg, fp)
    r, e, idx, sh = t(g.r), t(g.elem), t(g.nbr_idx), t(g.nbr_shift)
    rho, _, _, info = pkg.qmll_fchl19(dfp, r, e, idx, sh)
    x, _ = pkg.qmll_project(rho, e, t(U))
    params = pkg.SorfParams(d=model.d, D=model.D, n_transform=model.T, n_elem=model.n_elem, sigma=model.sigma,
                            signs=t(model.signs), bias=t(model.bias))
    E, gx = pkg.qmll_sorf_backward_g(params, x, e, t(g.mol_off), t(alpha))
    w = pkg.qmll_project_back(gx, e, t(U))
    F, info2 = pkg.qmll_fchl19_backward(dfp, r, e, idx, w, nbr_shift=sh)
    torch.cuda.synchronize()
    assert int(info.item()) == 0 and int(info2.item()) == 0
    return x, E, gx, w, F


def _backward_chain_oracle(fp, g, model, U, alpha):
    rho = oracle.fchl19(fp, g.r, g.elem, g.nbr_idx, g.nbr_shift)
    x = oracle.project(rho.astype(np.float32), g.elem, U)
    x32 = x.astype(np.float32)
    Z = oracle.forward(x32, g.elem, g.mol_off, model.d, model.D, model.T, model.sigma, model.signs, model.bias)
    E = oracle.energy(Z, alpha)
    gx = oracle.backward_g(x32, g.elem, model.d, model.D, model.T, model.sigma, model.signs, model.bias, alpha)
    w = oracle.project_back(gx, g.elem, U)
    F = oracle.fchl19_backward(fp, g.r, g.elem, g.nbr_idx, w, g.nbr_shift)
    return x, E, gx, w, F


@pytest.mark.parametrize("kind", ["molecules", "cell"])
def test_backward_chain_without_jacobian(q, kind):
    """qmll_sorf_backward_g, qmll_project_back and qmll_fchl19_backward against the oracle, step by step and as a chain;
    and the same forces as the Jacobian route (qmll_fchl19 + qmll_project_neighbor + qmll_predict)."""
    pkg, torch = q
    if kind == "molecules":
        fp = FchlParams()
        g = molecules_geometry(23, [9, 21, 27, 2, 1], probs=[0.5, 0.3, 0.06, 0.12, 0.02])
    else:
        fp = replace(FchlParams(), r_cut=3.6)
        g = cell_geometry(14, 6, spacing=2.0, jitter=0.35, r_list=3.9)
    d, D = 128, 1024
    model = make_model(81, d=d, D=D, T=3, sigma=3.0)
    U = projection_inputs(seed=82, counts=[1], rep=fp.rep, d=d).U
    alpha = (np.random.default_rng(83).normal(size=D) / np.sqrt(D)).astype(np.float32)
    x, E, gx, w, F = _backward_chain_gpu(q, fp, g, model, U, alpha)
    xo, Eo, gxo, wo, Fo = _backward_chain_oracle(fp, g, model, U, alpha)
    assert rel(x.cpu().numpy(), xo) <= TOL
    assert rel(E.cpu().numpy(), Eo) <= TOL
    assert rel(gx.cpu().numpy(), gxo) <= TOL_J
    assert rel(w.cpu().numpy(), wo) <= TOL_J
    assert rel(F.cpu().numpy(), Fo) <= TOL_J
    # each backward kernel alone on the oracle's own inputs
    t = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()
    w1 = pkg.qmll_project_back(t(gxo.astype(np.float32)), t(g.elem), t(U))
    assert rel(w1.cpu().numpy(), oracle.project_back(gxo.astype(np.float32), g.elem, U)) <= TOL
    F1, _ = pkg.qmll_fchl19_backward(dev_params(pkg, fp), t(g.r), t(g.elem), t(g.nbr_idx), t(wo.astype(np.float32)),
                                     nbr_shift=t(g.nbr_shift))
    assert rel(F1.cpu().numpy(), oracle.fchl19_backward(fp, g.r, g.elem, g.nbr_idx, wo.astype(np.float32), g.nbr_shift)) <= TOL_J
    # the Jacobian route gives the same forces
    dfp = dev_params(pkg, fp)
    rho, jidx, jval, _ = pkg.qmll_fchl19(dfp, t(g.r), t(g.elem), t(g.nbr_idx), t(g.nbr_shift), jacobian=True)
    dx = pkg.qmll_project_neighbor(jval, t(g.elem), t(U), idx=jidx)
    params = pkg.SorfParams(d=d, D=D, n_transform=3, n_elem=5, sigma=3.0, signs=t(model.signs), bias=t(model.bias))
    E2, F2 = pkg.qmll_predict(params, x, t(g.elem), t(g.mol_off), t(alpha), pkg.Grad.make_neighbor(jidx, dx))
    assert rel(F2.cpu().numpy(), Fo) <= TOL_J
    assert rel(F.cpu().numpy(), F2.cpu().numpy()) <= TOL_J


def test_backward_chain_fullsize_cell_properties(q):
    """15 625-atom cell (the configuration bench.py times): forces of the Jacobian-free chain equal those of the
    Jacobian route on ALL atoms, sum to zero, and match the oracle's contraction on sampled source atoms."""
    pkg, torch = q
    fp = replace(FchlParams(), r_cut=4.8)
    g = cell_geometry(2, 25, r_list=4.8, K=64)
    d, D = 256, 4096
    model = make_model(91, d=d, D=D, T=3, sigma=8.0)
    U = projection_inputs(seed=78, counts=[1], rep=fp.rep, d=d).U
    alpha = (np.random.default_rng(93).normal(size=D) / np.sqrt(D)).astype(np.float32)
    x, E, gx, w, F = _backward_chain_gpu(q, fp, g, model, U, alpha)
    t = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()
    dfp = dev_params(pkg, fp)
    rho, jidx, jval, _ = pkg.qmll_fchl19(dfp, t(g.r), t(g.elem), t(g.nbr_idx), t(g.nbr_shift), jacobian=True)
    dx = pkg.qmll_project_neighbor(jval, t(g.elem), t(U), idx=jidx)
    del jval
    params = pkg.SorfParams(d=d, D=D, n_transform=3, n_elem=5, sigma=8.0, signs=t(model.signs), bias=t(model.bias))
    E2, F2 = pkg.qmll_predict(params, x, t(g.elem), t(g.mol_off), t(alpha), pkg.Grad.make_neighbor(jidx, dx))
    torch.cuda.synchronize()
    Fn, F2n = F.cpu().numpy().astype(np.float64), F2.cpu().numpy().astype(np.float64)
    assert rel(Fn, F2n) <= TOL_J
    assert rel(E.cpu().numpy(), E2.cpu().numpy()) <= TOL
    assert np.abs(Fn.sum(0)).max() <= 1e-4 * np.abs(Fn).sum(0).max()
    # oracle on sampled source atoms: contributions of atom i alone (w zero elsewhere) scattered to its neighbours
    rng = np.random.default_rng(5)
    wn = w.cpu().numpy()
    for i in rng.choice(g.r.shape[0], size=6, replace=False):
        w1 = np.zeros_like(wn)
        w1[i] = wn[i]
        Fg, _ = pkg.qmll_fchl19_backward(dfp, t(g.r), t(g.elem), t(g.nbr_idx), t(w1), nbr_shift=t(g.nbr_shift))
        J = oracle.fchl19_jacobian(fp, g.r, g.elem, g.nbr_idx, g.nbr_shift, atoms=np.array([i]))[0]
        Fo = np.zeros((g.r.shape[0], 3))
        slots = np.concatenate([[i], g.nbr_idx[i]])
        for s, j in enumerate(slots):
            if j >= 0:
                Fo[j] -= wn[i].astype(np.float64) @ J[s]
        assert rel(Fg.cpu().numpy(), Fo) <= TOL_J
