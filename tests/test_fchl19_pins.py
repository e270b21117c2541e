"""Pins of the FCHL19 oracle (oracle/fchl19_oracle.c) against what the paper and the mathematics fix
(PAPER.md section E, eqs. 23-33; readings B1-B9 in DESIGN.md).  CPU only.

The paper prints no representation values, so the pins are: a library density (scipy.stats.lognorm) and the moments
eq. 25-26 are built to have, normalisation / centre / width of eq. 29, closed forms on triangles whose angles are
known (equilateral, right angle at the centre, right angle at a neighbour, 120-30-30), invariances, the cut-off, pair
additivity, and for the Jacobian Richardson finite differences plus its sum rules.
"""
from dataclasses import replace

import numpy as np
import pytest
from scipy import stats

import oracle
from workloads import FchlParams, molecules_geometry, cell_geometry

FP = FchlParams()            # Table I, column E + F (L248-260), r_cut = 6
O3 = np.zeros(3)


def off3(fp):
    return fp.n_elem * fp.n2


def pair_bin(fp, X, Y):
    X, Y = min(X, Y), max(X, Y)
    return X * fp.n_elem - X * (X - 1) // 2 + (Y - X)


def three_body(fp, rho, X, Y):
    """[n3, 2] block of element pair (X, Y)."""
    p = pair_bin(fp, X, Y)
    return rho[off3(fp) + p * fp.n3 * 2: off3(fp) + (p + 1) * fp.n3 * 2].reshape(fp.n3, 2)


def f_cut(r, rc):
    return 0.5 * (np.cos(np.pi * r / rc) + 1.0)


# ------------------------------------------------------------------------------------------------ two-body

def test_two_body_is_a_lognormal_density_with_mean_r_and_variance_eta2():
    """eq. 24-26: as a function of R_s the term is f_cut(r) r^-N2 times a log-normal density whose parameters
    mu(r), sigma(r) give it mean r and variance eta_2.  Fine grid => Riemann sums of the oracle's output."""
    fp = replace(FP, n2=6000, n3=1, eta2=0.02, N2=1.8)
    dR = fp.r_cut / fp.n2
    Rs = fp.r_cut * (np.arange(fp.n2) + 1) / fp.n2
    for r, X in ((1.1, 1), (2.0, 3), (3.0, 0)):           # r_cut / 3 and r_cut / 2: f_cut = 3/4 and 1/2 exactly
        rho = oracle.fchl19_atom(fp, O3, [[r, 0, 0]], [X])
        g = rho[X * fp.n2:(X + 1) * fp.n2]
        mass = g.sum() * dR
        mean = (Rs * g).sum() * dR / mass
        var = ((Rs - mean) ** 2 * g).sum() * dR / mass
        assert abs(mean - r) < 1e-6 * r
        assert abs(var - fp.eta2) < 1e-5 * fp.eta2
        fc = {2.0: 0.75, 3.0: 0.5}.get(r, f_cut(r, fp.r_cut))
        assert abs(mass - fc * r ** -fp.N2) < 1e-7 * mass
        # only the bin of the neighbour's element is populated
        others = np.delete(rho[:off3(fp)].reshape(fp.n_elem, fp.n2), X, axis=0)
        assert np.all(others == 0) and np.all(rho[off3(fp):] == 0)
        # point-wise against the library density with the shape / scale that have these two moments
        s2 = np.log1p(var / mean ** 2)
        ref = fc * r ** -fp.N2 * stats.lognorm.pdf(Rs, s=np.sqrt(s2), scale=mean / np.sqrt(1 + var / mean ** 2))
        assert np.linalg.norm(g - ref) < 1e-4 * np.linalg.norm(ref)     # moments are measured, hence 1e-4


def test_two_body_lognormal_pointwise_table_parameters():
    """Same check at the paper's parameters (Table I), point-wise against scipy.stats.lognorm.pdf."""
    for fp in (FP, replace(FP, n2=23, eta2=0.27, N2=2.78)):
        Rs = fp.r_cut * (np.arange(fp.n2) + 1) / fp.n2
        for r in (0.9, 1.5, 4.2, 5.9):
            g = oracle.fchl19_atom(fp, O3, [[0, r, 0]], [2])[2 * fp.n2:3 * fp.n2]
            s2 = np.log1p(fp.eta2 / r ** 2)                       # variance eta2, mean r
            ref = f_cut(r, fp.r_cut) * r ** -fp.N2 * stats.lognorm.pdf(Rs, s=np.sqrt(s2), scale=r / np.sqrt(1 + fp.eta2 / r ** 2))
            np.testing.assert_allclose(g, ref, rtol=1e-10, atol=1e-14 * ref.max())


def test_two_body_decay_exponent_and_cutoff_values():
    fp0 = replace(FP, N2=0.0)
    for r in (1.3, 2.7):
        a = oracle.fchl19_atom(FP, O3, [[r, 0, 0]], [0])[:FP.n2]
        b = oracle.fchl19_atom(fp0, O3, [[r, 0, 0]], [0])[:FP.n2]
        np.testing.assert_allclose(a, b * r ** -FP.N2, rtol=1e-13)
    # cut-off: zero at and beyond r_cut, continuous approach (f ~ (pi (rc - r) / (2 rc))^2)
    assert np.all(oracle.fchl19_atom(FP, O3, [[FP.r_cut, 0, 0]], [0]) == 0)
    assert np.all(oracle.fchl19_atom(FP, O3, [[FP.r_cut + 1.0, 0, 0]], [0]) == 0)
    near = oracle.fchl19_atom(FP, O3, [[FP.r_cut - 1e-4, 0, 0]], [0])
    mid = oracle.fchl19_atom(FP, O3, [[FP.r_cut - 1.0, 0, 0]], [0])
    assert 0 < np.abs(near).max() < 1e-8 * np.abs(mid).max()


# ------------------------------------------------------------------------------------------------ three-body

def _integrated(fp, centre, img, elems, X, Y):
    """(sum_s G3 dR [cos, sin], centre of mass in R_s, variance in R_s) of the pair block."""
    rho = oracle.fchl19_atom(fp, centre, img, elems)
    g = three_body(fp, rho, X, Y)
    dR = fp.r_cut / fp.n3
    Rs = fp.r_cut * (np.arange(fp.n3) + 1) / fp.n3
    tot = g.sum(0) * dR
    w = np.abs(g[:, 1])
    mean = (Rs * w).sum() / w.sum()
    var = ((Rs - mean) ** 2 * w).sum() / w.sum()
    return tot, mean, var


def test_three_body_equilateral_closed_form():
    """All angles 60 degrees: xi_3 = c3 (1 + 3/8) / L^(3 N3), cos theta = 1/2, sin theta = sqrt(3)/2, L = r_cut / 3 so
    that every f_cut is exactly 3/4; eq. 29 integrates to 1 over R_s, is centred at (r_ij + r_ik) / 2 = L and has
    variance 1 / (2 eta_3)."""
    fp = replace(FP, n2=1, n3=3000, eta3=6.0)
    L = fp.r_cut / 3
    img = [[L, 0, 0], [L / 2, L * np.sqrt(3) / 2, 0]]
    tot, mean, var = _integrated(fp, O3, img, [1, 3], 1, 3)
    pref = fp.c3 * (1 + 3 / 8) / L ** (3 * fp.N3) * 0.75 ** 3 * 2 * np.exp(-fp.zeta ** 2 / 2)
    np.testing.assert_allclose(tot, [pref * 0.5, pref * np.sqrt(3) / 2], rtol=1e-9)
    assert abs(mean - L) < 1e-9 and abs(var - 1 / (2 * fp.eta3)) < 1e-9


def test_three_body_right_angle_at_centre_and_at_neighbour():
    fp = replace(FP, n2=1, n3=3000, eta3=6.0, r_cut=4.8)
    damp2 = 2 * np.exp(-fp.zeta ** 2 / 2)
    # right angle at the central atom: cos theta_kij = 0 kills the Axilrod-Teller product and the cos channel
    ra, rb = 1.6, 2.4                                 # r_cut / 3, r_cut / 2: f = 3/4, 1/2
    rc = np.hypot(ra, rb)
    tot, mean, _ = _integrated(fp, O3, [[ra, 0, 0], [0, 0, rb]], [0, 0], 0, 0)
    want = fp.c3 / (ra * rb * rc) ** fp.N3 * damp2 * 0.75 * 0.5 * f_cut(rc, fp.r_cut)
    assert abs(tot[0]) < 1e-12 * want
    np.testing.assert_allclose(tot[1], want, rtol=1e-9)
    assert abs(mean - (ra + rb) / 2) < 1e-9
    # right angle at neighbour j: the product is again zero, but the Fourier term uses the angle AT THE CENTRE
    # (cos = 3/5, sin = 4/5 for the 3-4-5 triangle)
    j, k = np.array([1.2, 0, 0]), np.array([1.2, 1.6, 0])
    tot, mean, _ = _integrated(fp, O3, [j, k], [2, 4], 2, 4)
    want = fp.c3 / (1.2 * 2.0 * 1.6) ** fp.N3 * damp2 * f_cut(1.2, 4.8) * f_cut(2.0, 4.8) * 0.75
    np.testing.assert_allclose(tot, [want * 0.6, want * 0.8], rtol=1e-7)   # 2e-8 of the Gaussian lies below R = 0
    assert abs(mean - 1.6) < 1e-6


def test_three_body_obtuse_triangle_numerator():
    """Angles 120 (centre), 30, 30: 1 + 3 cos cos cos = 1 - 9/8 = -1/8; cos theta = -1/2 => the cos channel is
    POSITIVE (two negatives), the sin channel negative."""
    fp = replace(FP, n2=1, n3=3000, eta3=6.0)
    r = 2.5
    img = [[r, 0, 0], [r * np.cos(2 * np.pi / 3), r * np.sin(2 * np.pi / 3), 0]]
    rc = r * np.sqrt(3)
    tot, _, _ = _integrated(fp, O3, img, [0, 1], 0, 1)
    pref = fp.c3 * (-1 / 8) / (r * r * rc) ** fp.N3 * f_cut(r, 6.0) ** 2 * f_cut(rc, 6.0) * 2 * np.exp(-fp.zeta ** 2 / 2)
    np.testing.assert_allclose(tot, [pref * -0.5, pref * np.sqrt(3) / 2], rtol=1e-9)


def test_three_body_third_cutoff_and_each_triangle_once():
    # j and k both inside r_cut of the centre but further than r_cut from each other: no contribution (B3)
    rho = oracle.fchl19_atom(FP, O3, [[4.0, 0, 0], [-4.0, 0, 0.1]], [0, 0])
    assert np.all(rho[off3(FP):] == 0) and np.any(rho[:off3(FP)] != 0)
    # additivity: three neighbours = the three pairs taken separately (each unordered pair once, B6); the closed-form
    # tests above fix the absolute factor
    rng = np.random.default_rng(5)
    img = rng.normal(size=(3, 3)) * 1.3
    el = [1, 1, 1]
    full = oracle.fchl19_atom(FP, O3, img, el)[off3(FP):]
    parts = sum(oracle.fchl19_atom(FP, O3, img[[a, b]], [1, 1])[off3(FP):] for a, b in ((0, 1), (0, 2), (1, 2)))
    np.testing.assert_allclose(full, parts, rtol=1e-12, atol=1e-300)


# ------------------------------------------------------------------------------------------------ invariances

def _random_env(seed, nn=9, n_elem=5):
    rng = np.random.default_rng(seed)
    img = rng.normal(size=(nn, 3)) * 1.8
    img += np.sign(img) * 0.4
    return rng.normal(size=3), img, rng.integers(0, n_elem, size=nn).astype(np.int32)


def test_rotation_translation_permutation_invariance():
    c, img, el = _random_env(11)
    base = oracle.fchl19_atom(FP, c, img + c, el)
    Q, _ = np.linalg.qr(np.random.default_rng(12).normal(size=(3, 3)))
    t = np.array([3.0, -2.0, 0.7])
    moved = oracle.fchl19_atom(FP, c @ Q.T + t, (img + c) @ Q.T + t, el)
    np.testing.assert_allclose(moved, base, rtol=1e-10, atol=1e-14)
    perm = np.random.default_rng(13).permutation(len(el))
    np.testing.assert_allclose(oracle.fchl19_atom(FP, c, (img + c)[perm], el[perm]), base, rtol=1e-12, atol=1e-300)


def test_element_relabelling_permutes_blocks():
    c, img, el = _random_env(21)
    base = oracle.fchl19_atom(FP, c, img + c, el)
    relabel = np.array([2, 0, 4, 1, 3], dtype=np.int32)
    other = oracle.fchl19_atom(FP, c, img + c, relabel[el])
    E = FP.n_elem
    for X in range(E):
        np.testing.assert_array_equal(other[relabel[X] * FP.n2:(relabel[X] + 1) * FP.n2], base[X * FP.n2:(X + 1) * FP.n2])
        for Y in range(X, E):
            np.testing.assert_allclose(three_body(FP, other, relabel[X], relabel[Y]), three_body(FP, base, X, Y),
                                       rtol=1e-12, atol=1e-300)
    assert FP.rep == E * FP.n2 + E * (E + 1) * FP.n3 == base.shape[0]


def test_array_api_matches_single_atom_api_and_periodic_images():
    g = molecules_geometry(3, [4, 7, 12])
    rho = oracle.fchl19(FP, g.r, g.elem, g.nbr_idx)
    for i in (0, 5, 17):
        q = g.nbr_idx[i][g.nbr_idx[i] >= 0]
        one = oracle.fchl19_atom(FP, g.r[i].astype(np.float64), g.r[q].astype(np.float64), g.elem[q])
        np.testing.assert_allclose(rho[i], one, rtol=1e-13, atol=1e-300)
    # a periodic cell: translating every atom by a lattice vector's worth of "wrap" changes nothing, and the shifts
    # are what is added to r_j
    c = cell_geometry(4, 5, spacing=2.0, jitter=0.3, r_list=3.6)
    fp = replace(FP, r_cut=3.6)
    rho = oracle.fchl19(fp, c.r, c.elem, c.nbr_idx, c.nbr_shift)
    i = 7
    sel = c.nbr_idx[i] >= 0
    img = c.r[c.nbr_idx[i][sel]].astype(np.float64) + c.nbr_shift[i][sel]
    np.testing.assert_allclose(rho[i], oracle.fchl19_atom(fp, c.r[i].astype(np.float64), img, c.elem[c.nbr_idx[i][sel]]),
                               rtol=1e-13, atol=1e-300)
    assert np.all(np.linalg.norm(img - c.r[i], axis=1) < 3.6 + 1e-5)
    assert (np.abs(c.nbr_shift) > 0).any()


# ------------------------------------------------------------------------------------------------ Jacobian

def _richardson(f, x, h):
    d1 = (f(x + h) - f(x - h)) / (2 * h)
    d2 = (f(x + 2 * h) - f(x - 2 * h)) / (4 * h)
    return (4 * d1 - d2) / 3


@pytest.mark.parametrize("fp", [FP, replace(FP, n2=23, n3=22, eta2=0.27, eta3=5.6, N2=2.78, N3=2.1, c3=60.1)])
def test_jacobian_matches_finite_differences(fp):
    c, img, el = _random_env(31, nn=7)
    img = img + c
    rho, jac = oracle.fchl19_atom(fp, c, img, el, jacobian=True)
    assert jac.shape == (8, fp.rep, 3)
    scale = np.abs(jac).max()
    for slot in range(8):
        for ax in range(3):
            def f(t):
                cc, ii = c.copy(), img.copy()
                if slot == 0:
                    cc[ax] = t
                else:
                    ii[slot - 1, ax] = t
                return oracle.fchl19_atom(fp, cc, ii, el)
            x0 = c[ax] if slot == 0 else img[slot - 1, ax]
            fd = _richardson(f, x0, 1e-3)
            assert np.abs(fd - jac[slot, :, ax]).max() < 2e-8 * scale


def test_jacobian_sum_rules():
    c, img, el = _random_env(41, nn=10)
    img = img + c
    _, jac = oracle.fchl19_atom(FP, c, img, el, jacobian=True)
    scale = np.abs(jac).max()
    # translation invariance: sum over all slots vanishes
    assert np.abs(jac.sum(0)).max() < 1e-12 * scale
    # rotation invariance: sum_slots (r_slot x d rho / d r_slot) = 0 for every component of rho
    pos = np.vstack([c[None], img])
    torque = np.cross(pos[:, None, :], jac).sum(0)
    assert np.abs(torque).max() < 1e-11 * scale * np.abs(pos).max()
    # a neighbour outside the cut-off has a zero block and changes nothing else
    far = np.vstack([img, c + [0, 0, FP.r_cut + 0.5]])
    _, jac2 = oracle.fchl19_atom(FP, c, far, np.append(el, 0).astype(np.int32), jacobian=True)
    assert np.all(jac2[-1] == 0)
    np.testing.assert_array_equal(jac2[:-1], jac)


def test_array_jacobian_layout_padding_and_selection():
    g = molecules_geometry(6, [5, 9], K=12)
    atoms = np.array([1, 6, 13], dtype=np.int64)
    J = oracle.fchl19_jacobian(FP, g.r, g.elem, g.nbr_idx, atoms=atoms)
    assert J.shape == (3, 13, FP.rep, 3)
    for t, i in enumerate(atoms):
        sel = np.nonzero(g.nbr_idx[i] >= 0)[0]
        q = g.nbr_idx[i][sel]
        _, one = oracle.fchl19_atom(FP, g.r[i].astype(np.float64), g.r[q].astype(np.float64), g.elem[q], jacobian=True)
        np.testing.assert_allclose(J[t, 0], one[0], rtol=1e-12, atol=1e-300)
        for m, s in enumerate(sel):
            np.testing.assert_allclose(J[t, 1 + s], one[1 + m], rtol=1e-12, atol=1e-300)
        pad = np.nonzero(g.nbr_idx[i] < 0)[0]
        assert len(pad) > 0 and np.all(J[t, 1 + pad] == 0)


def test_project_neighbor_gradient_is_the_per_element_matrix_product():
    rng = np.random.default_rng(7)
    n_atoms, S, rep, d, E = 6, 4, 37, 16, 3
    gin = rng.normal(size=(n_atoms, S, rep, 3)).astype(np.float32)
    U = rng.normal(size=(E, rep, d)).astype(np.float32)
    elem = rng.integers(0, E, size=n_atoms).astype(np.int32)
    out = oracle.project_neighbor_gradient(gin, elem, U)
    for a in range(n_atoms):
        ref = np.einsum("skc,km->smc", gin[a].astype(np.float64), U[elem[a]].astype(np.float64))
        np.testing.assert_allclose(out[a], ref, rtol=1e-12, atol=1e-14)


def test_chain_forces_match_finite_differences_of_the_energy():
    """Whole chain in the oracle: r -> rho (FCHL19) -> x = rho^T U_e -> E = sum_I alpha . z(x_I); the force assembled
    from the Jacobian (slot 0 = the atom, slot 1 + q = neighbour q), the projected gradient and the SORF backward
    pass must be -dE/dr.  Coordinates lie on a 2^-10 grid and the step is 2^-6, so every displaced geometry is exact
    in the fp32 arrays the oracle's interfaces take; the fp32 hand-over of rho limits the agreement to ~1e-5."""
    from workloads import make_model
    fp = replace(FP, n_elem=2, n2=6, n3=4, r_cut=4.0)
    g = molecules_geometry(51, [5], n_elem=2)
    r0 = (np.round(g.r.astype(np.float64) * 1024) / 1024).astype(np.float32)
    d, D, T, sigma = 16, 256, 3, 2.5
    model = make_model(52, d=d, D=D, T=T, sigma=sigma, n_elem=2)
    rng = np.random.default_rng(53)
    U = rng.normal(size=(2, fp.rep, d)).astype(np.float32) * 0.5
    alpha = rng.normal(size=D).astype(np.float32)

    def energy(r):
        rho = oracle.fchl19(fp, r, g.elem, g.nbr_idx)
        x = oracle.project(rho.astype(np.float32), g.elem, U)
        Z = oracle.forward(x.astype(np.float32), g.elem, g.mol_off, d, D, T, sigma, model.signs, model.bias)
        return float(oracle.energy(Z, alpha)[0])

    rho = oracle.fchl19(fp, r0, g.elem, g.nbr_idx)
    J = oracle.fchl19_jacobian(fp, r0, g.elem, g.nbr_idx)
    x = oracle.project(rho.astype(np.float32), g.elem, U).astype(np.float32)
    dx = oracle.project_neighbor_gradient(J.astype(np.float32), g.elem, U)
    idx = np.concatenate([np.arange(5, dtype=np.int32)[:, None], g.nbr_idx], axis=1)
    gx = oracle.backward_g(x, g.elem, d, D, T, sigma, model.signs, model.bias, alpha)
    F = oracle.forces_neighbor(gx, d, idx, dx.astype(np.float32))
    h = 2.0 ** -6
    F_fd = np.zeros_like(F)
    for a in range(5):
        for c in range(3):
            def e(step):
                r = r0.copy()
                r[a, c] += np.float32(step)
                return energy(r)
            F_fd[a, c] = -(8 * (e(h) - e(-h)) - (e(2 * h) - e(-2 * h))) / (12 * h)
    assert np.linalg.norm(F) > 0
    assert np.linalg.norm(F - F_fd) <= 1e-4 * np.linalg.norm(F_fd)


def test_backward_chain_equals_jacobian_chain_and_finite_differences():
    """The Jacobian-free backward pass in the oracle (dE/dx -> dE/d rho -> forces) is the same contraction in another
    order: it must equal the force assembled through the projected Jacobian (pinned above by finite differences of
    E(r)), to rounding; project_back is the plain transposed matrix product."""
    from workloads import make_model
    fp = replace(FP, n_elem=3, n2=7, n3=5, r_cut=4.5)
    g = molecules_geometry(61, [6, 4], n_elem=3)
    d, D, T, sigma = 16, 128, 3, 2.0
    model = make_model(62, d=d, D=D, T=T, sigma=sigma, n_elem=3)
    rng = np.random.default_rng(63)
    U = rng.normal(size=(3, fp.rep, d)).astype(np.float32) * 0.4
    alpha = rng.normal(size=D).astype(np.float32)
    rho = oracle.fchl19(fp, g.r, g.elem, g.nbr_idx)
    J = oracle.fchl19_jacobian(fp, g.r, g.elem, g.nbr_idx)
    x = oracle.project(rho.astype(np.float32), g.elem, U).astype(np.float32)
    gx = oracle.backward_g(x, g.elem, d, D, T, sigma, model.signs, model.bias, alpha)
    w = oracle.project_back(gx, g.elem, U)
    for a in range(10):
        np.testing.assert_allclose(w[a], U[g.elem[a]].astype(np.float64) @ gx[a], rtol=1e-12, atol=1e-14)
    F_back = oracle.fchl19_backward(fp, g.r, g.elem, g.nbr_idx, w)
    # the same force through the (exact, FP64) projected Jacobian: einsum written out in the test
    idx = np.concatenate([np.arange(10, dtype=np.int32)[:, None], g.nbr_idx], axis=1)
    F_jac = np.zeros((10, 3))
    for a in range(10):
        dx = np.einsum("skc,km->smc", J[a], U[g.elem[a]].astype(np.float64))
        for s, j in enumerate(idx[a]):
            if j >= 0:
                F_jac[j] -= gx[a] @ dx[s]
    np.testing.assert_allclose(F_back, F_jac, rtol=1e-10, atol=1e-12 * np.abs(F_jac).max())
    assert np.abs(F_back.sum(0)).max() < 1e-10 * np.abs(F_back).max()       # no net force (translation invariance)


def test_table_1_parameters_are_the_papers():
    """tests/golden/fchl19_table1.json holds Table I as the paper prints it (L248-260); the generator's defaults, its
    energy-only set and the binding's defaults must be those numbers."""
    import json
    import os
    with open(os.path.join(os.path.dirname(__file__), "golden", "fchl19_table1.json")) as f:
        tab = json.load(f)
    from workloads import FCHL_E
    ef, e = FchlParams(), replace(FchlParams(), **FCHL_E)
    for got, want in ((ef, tab["E+F"]), (e, tab["E"])):
        for k, v in want.items():
            assert getattr(got, k) == pytest.approx(v, rel=0, abs=1e-15), k
    import paper_2206_01580_b200 as pkg
    b = pkg.Fchl19Params()
    w = tab["E+F"]
    assert (b.n2, b.n3, b.eta2, b.eta3, b.two_body_decay, b.three_body_decay, b.three_body_weight, b.r_cut) == \
        (w["n2"], w["n3"], w["eta2"], w["eta3"], w["N2"], w["N3"], w["c3"], w["r_cut"])
    assert b.zeta == pytest.approx(np.pi)


def test_fchl19_golden_regression():
    """tests/golden/fchl19_oracle.json was written by tests/golden/make_golden.py (oracle only): a guard against
    accidental changes of the oracle's arithmetic, not a pin."""
    import json
    import os
    with open(os.path.join(os.path.dirname(__file__), "golden", "fchl19_oracle.json")) as f:
        gold = json.load(f)
    g = molecules_geometry(99, [7])
    assert g.elem.tolist() == gold["elements"]
    rho = oracle.fchl19(FP, g.r, g.elem, g.nbr_idx)
    J = oracle.fchl19_jacobian(FP, g.r, g.elem, g.nbr_idx, atoms=np.array([0]))
    i0 = gold["rho_atom0_first_nonzero_index"]
    nz = np.nonzero(rho[0])[0]
    assert rho.shape[1] == gold["rep"] and nz[0] == i0
    np.testing.assert_allclose(np.linalg.norm(rho), gold["rho_fro"], rtol=1e-12)
    np.testing.assert_allclose(rho[0, nz[:8]], gold["rho_atom0_first8_nonzero"], rtol=1e-11)
    np.testing.assert_allclose(rho.sum(1), gold["rho_row_sums"], rtol=1e-11)
    np.testing.assert_allclose(np.linalg.norm(J), gold["jac_atom0_fro"], rtol=1e-11)
    np.testing.assert_allclose(J[0, 0, i0], gold["jac_atom0_self_first_nonzero_row"], rtol=1e-9, atol=1e-14)
