"""Pins for the FP64 oracle: each test checks `oracle/` against something the paper or the
mathematics fixes, never against the oracle itself (and never against the CUDA path).

Citations are PAPER.md lines; readings A1-A16 are SURVEY.md section 8(c) / DESIGN.md.
"""
import numpy as np
import pytest

import oracle
from workloads import make_workload, make_model, tiny_workload, Workload, DescriptorGradient


# ----------------------------------------------------------------------------- helpers (test-local)
def dense_H(d: int) -> np.ndarray:
    """Explicit Sylvester matrix from the recursion H_{2n} = [[H, H], [H, -H]], H_1 = 1 (L163-165)."""
    H = np.array([[1.0]])
    while H.shape[0] < d:
        H = np.block([[H, H], [H, -H]])
    return H


def dense_W(model, e: int) -> np.ndarray:
    """Explicit D x d matrix of eq. 20 for element e: rows s*d..(s+1)*d = c * H D_T ... H D_1."""
    d, D, T = model.d, model.D, model.T
    H = dense_H(d)
    c = np.sqrt(d) / model.sigma * d ** (-T / 2.0)
    blocks = []
    for s in range(D // d):
        W = np.eye(d)
        for t in range(T):
            W = H @ (np.diag(model.signs[e, s, t].astype(np.float64)) @ W)
        blocks.append(c * W)
    return np.concatenate(blocks, axis=0)


# ----------------------------------------------------------------------------- FWHT (a1)
@pytest.mark.parametrize("d", [1, 2, 4, 8, 16, 32, 64])
def test_fwht_equals_dense_hadamard(d):
    rng = np.random.default_rng(d)
    H = dense_H(d)
    for _ in range(3):
        v = rng.standard_normal(d)
        assert np.allclose(oracle.fwht(v), H @ v, rtol=0, atol=1e-12 * d)
    # natural (Hadamard) order, entry formula (-1)^popcount(i & j)  (reading A3)
    i, j = np.meshgrid(np.arange(d), np.arange(d), indexing="ij")
    pop = np.vectorize(lambda a: bin(a).count("1"))(i & j)
    assert np.array_equal(H, (-1.0) ** pop)
    for k in range(d):
        ek = np.zeros(d); ek[k] = 1.0
        assert np.array_equal(oracle.fwht(ek), H[:, k])


@pytest.mark.parametrize("d", [2, 16, 128, 1024])
def test_fwht_involution_and_symmetry(d):
    rng = np.random.default_rng(100 + d)
    v, w = rng.standard_normal(d), rng.standard_normal(d)
    assert np.allclose(oracle.fwht(oracle.fwht(v)), d * v, rtol=1e-12, atol=1e-10)       # H H = d I
    assert np.isclose(w @ oracle.fwht(v), oracle.fwht(w) @ v, rtol=1e-11)                # H = H^T
    assert np.allclose(oracle.fwht(2.0 * v - 3.0 * w), 2.0 * oracle.fwht(v) - 3.0 * oracle.fwht(w), atol=1e-10)
    assert np.isclose(np.sum(oracle.fwht(v) ** 2), d * np.sum(v ** 2), rtol=1e-11)       # Parseval


# ----------------------------------------------------------------------------- SORF map (a1, scale c)
@pytest.mark.parametrize("T", [1, 2, 3])
@pytest.mark.parametrize("d", [2, 8, 64])
def test_sorf_u_equals_dense_W(d, T):
    model = make_model(seed=7 * d + T, d=d, D=4 * d, T=T, sigma=1.7, n_elem=3)
    rng = np.random.default_rng(d + T)
    for e in range(3):
        x = rng.standard_normal(d).astype(np.float32)
        u = oracle.sorf_u(x, e, d, 4 * d, T, model.sigma, model.signs)
        assert np.allclose(u, dense_W(model, e) @ x.astype(np.float64), rtol=1e-12, atol=1e-12)


def test_closed_form_all_plus_signs():
    """All signs +1, x = a e_0, T = 3:  H H H x = d H x = d a 1, so u[l] = a/sigma for every l and
    z[l] = sqrt(2/D) cos(a/sigma + b[l]) (eq. 14 with eq. 20, reading A2)."""
    d, D, T, sigma, a = 64, 256, 3, 2.0, 0.8125
    model = make_model(1, d, D, T, sigma, n_elem=1)
    model.signs[...] = 1
    x = np.zeros((1, d), np.float32); x[0, 0] = a
    u = oracle.sorf_u(x[0], 0, d, D, T, sigma, model.signs)
    assert np.allclose(u, a / sigma, rtol=1e-13)
    Z = oracle.forward(x, [0], [0, 1], d, D, T, sigma, model.signs, model.bias)
    assert np.allclose(Z[0], np.sqrt(2.0 / D) * np.cos(a / sigma + model.bias[0].astype(np.float64)), atol=1e-14)


@pytest.mark.parametrize("T", [1, 2, 3])
def test_per_stack_norm_invariant(T):
    """Each stack is sqrt(d)/sigma times an orthogonal matrix: sum_m u[s d + m]^2 = d |x|^2 / sigma^2."""
    d, D, sigma = 128, 1024, 3.0
    model = make_model(11 + T, d, D, T, sigma, n_elem=2)
    x = np.random.default_rng(5).standard_normal(d).astype(np.float32)
    u = oracle.sorf_u(x, 1, d, D, T, sigma, model.signs).reshape(D // d, d)
    want = d * np.sum(x.astype(np.float64) ** 2) / sigma ** 2
    assert np.allclose(np.sum(u ** 2, axis=1), want, rtol=1e-12)


def test_monte_carlo_gaussian_kernel():
    """z(x).z(y) -> exp(-|x-y|^2 / 2 sigma^2) as D grows (eq. 12-14; L156 'unbiased ... low
    variance').  Nearby pairs y = x + delta*sigma*unit, D = 16384, 8 seeds; the spread falls like 1/sqrt(D)."""
    d, T, sigma = 64, 3, 2.0
    rng = np.random.default_rng(2022)
    x = rng.standard_normal(d)
    dirn = rng.standard_normal(d); dirn /= np.linalg.norm(dirn)

    def estimates(D, delta, seeds):
        out = []
        for s in seeds:
            model = make_model(9000 + s, d, D, T, sigma, n_elem=1)
            xy = np.stack([x, x + delta * sigma * dirn]).astype(np.float32)
            Z = oracle.forward(xy, [0, 0], [0, 1, 2], d, D, T, sigma, model.signs, model.bias)
            out.append(Z[0] @ Z[1])
        return np.array(out)

    for delta in (0.5, 1.0, 2.0):
        est = estimates(16384, delta, range(8))
        xy = np.stack([x, x + delta * sigma * dirn]).astype(np.float32).astype(np.float64)
        k = np.exp(-np.sum((xy[0] - xy[1]) ** 2) / (2 * sigma ** 2))
        assert abs(est.mean() - k) <= 0.02, (delta, est.mean(), k)
    s_small = estimates(256, 1.0, range(24)).std()
    s_big = estimates(16384, 1.0, range(24)).std()
    assert 3.0 < s_small / s_big < 20.0          # ideal ratio sqrt(16384/256) = 8


def test_cross_element_features_are_uncorrelated():
    """Per-element signs and b (reading A6): z_e(x).z_e'(x) ~ 0 while z_e(x).z_e(x) ~ 1."""
    d, D, T, sigma = 64, 16384, 3, 2.0
    model = make_model(77, d, D, T, sigma, n_elem=2)
    x = np.random.default_rng(3).standard_normal((1, d)).astype(np.float32)
    xx = np.concatenate([x, x])
    Z = oracle.forward(xx, [0, 1], [0, 1, 2], d, D, T, sigma, model.signs, model.bias)
    assert abs(Z[0] @ Z[0] - 1.0) < 0.03
    assert abs(Z[0] @ Z[1]) < 0.03


# ----------------------------------------------------------------------------- whole path, brute force (C1)
def test_c1_brute_force_dense_W():
    """Config 1 computed with explicit D x d matrices and eq. 14/15 as dense mat-vecs."""
    w = make_workload("c1")
    m = w.model
    Wd = [dense_W(m, e) for e in range(m.n_elem)]
    nrm = np.sqrt(2.0 / m.D)
    x64 = w.x.astype(np.float64)
    Z = np.zeros((w.n_mol, m.D))
    g = np.zeros((w.n_atoms, m.d))
    G = np.zeros((3 * w.n_atoms, m.D))
    a64 = w.alpha.astype(np.float64)
    for M in range(w.n_mol):
        lo, hi = w.mol_off[M], w.mol_off[M + 1]
        n = hi - lo
        dx = w.grad.dense_block(M, n, m.d).astype(np.float64)          # (I, m, j, k)
        for I in range(lo, hi):
            e = w.elem[I]
            arg = Wd[e] @ x64[I] + m.bias[e].astype(np.float64)
            Z[M] += nrm * np.cos(arg)
            g[I] = Wd[e].T @ (-nrm * a64 * np.sin(arg))
            wcol = np.einsum("lm,mjk->jkl", Wd[e], dx[I - lo])         # W (dx_I[:, j, k])
            G[3 * lo:3 * hi] += (nrm * np.sin(arg))[None, :] * wcol.reshape(3 * n, m.D)
    F = np.zeros((w.n_atoms, 3))
    for M in range(w.n_mol):
        lo, hi = w.mol_off[M], w.mol_off[M + 1]
        dx = w.grad.dense_block(M, hi - lo, m.d).astype(np.float64)
        F[lo:hi] = -np.einsum("im,imjk->jk", g[lo:hi], dx)

    assert np.allclose(oracle.forward_w(w), Z, rtol=0, atol=1e-13)
    assert np.allclose(oracle.energy(oracle.forward_w(w), w.alpha), Z @ a64, atol=1e-13)
    assert np.allclose(oracle.backward_g_w(w), g, atol=1e-13)
    assert np.allclose(oracle.forces_w(w), F, atol=1e-12)
    assert np.allclose(oracle.force_rows_w(w), G, atol=1e-13)
    A = np.concatenate([Z, G]).astype(np.float32)
    ZtZ, Zty = oracle.normal_equations(A, w.y)
    A64 = A.astype(np.float64)
    assert np.allclose(ZtZ, A64.T @ A64, rtol=1e-12, atol=1e-15)        # BLAS dsyrk-style cross-check
    assert np.allclose(Zty, A64.T @ w.y.astype(np.float64), rtol=1e-12, atol=1e-15)


# ----------------------------------------------------------------------------- forces (a4-a7)
def _linear_descriptor_case(seed=0, n=3, d=8, D=64, T=3, sigma=1.5):
    """Hand-written descriptor x_I[m] = sum_{j,k} C[I,m,j,k] r[j,k] with small-integer C and dyadic r,
    so x is exact in fp32 at every finite-difference point and dx/dr = C exactly."""
    rng = np.random.default_rng(seed)
    C = rng.integers(-2, 3, size=(n, d, n, 3)).astype(np.float64)
    r0 = rng.integers(-128, 129, size=(n, 3)).astype(np.float64) / 256.0
    model = make_model(seed + 50, d, D, T, sigma, n_elem=2)
    elem = rng.integers(0, 2, size=n).astype(np.int32)
    alpha = rng.standard_normal(D).astype(np.float32)

    def workload(r):
        x = np.einsum("imjk,jk->im", C, r)
        x32 = x.astype(np.float32)
        assert np.array_equal(x32.astype(np.float64), x)
        grad = DescriptorGradient(layout="dense", dense=C.astype(np.float32).reshape(-1),
                                  dense_off=np.array([0, C.size], dtype=np.int64))
        return Workload(name="lin", model=model, elem=elem, mol_off=np.array([0, n], np.int32), x=x32,
                        alpha=alpha, grad=grad)
    return workload, r0


@pytest.mark.parametrize("T", [1, 2, 3])
def test_forces_match_finite_differences(T):
    workload, r0 = _linear_descriptor_case(seed=T, T=T)

    def E(r):
        w = workload(r)
        return oracle.energy(oracle.forward_w(w), w.alpha)[0]

    F = oracle.forces_w(workload(r0))
    h = 2.0 ** -9
    for j in range(r0.shape[0]):
        for k in range(3):
            def cd(step):
                rp, rm = r0.copy(), r0.copy()
                rp[j, k] += step; rm[j, k] -= step
                return (E(rp) - E(rm)) / (2 * step)
            fd = (4.0 * cd(h / 2) - cd(h)) / 3.0                      # Richardson, O(h^4)
            assert abs(-fd - F[j, k]) <= 1e-7 * max(1.0, abs(F[j, k])), (j, k, -fd, F[j, k])


def test_force_rows_times_alpha_equal_forces():
    """JVP/VJP consistency: G alpha = F from the backward path, for random alpha (two code paths)."""
    for layout in ("dense", "neighbor"):
        w = tiny_workload(31, d=16, D=64, T=3, sigma=2.0, counts=[3, 1, 5, 2], grad=layout, K=3)
        G = oracle.force_rows_w(w)
        for s in range(3):
            a = np.random.default_rng(s).standard_normal(w.model.D).astype(np.float32)
            F = oracle.forces_w(w, a)
            assert np.allclose(G @ a.astype(np.float64), F.reshape(-1), rtol=1e-11, atol=1e-12)


def test_force_rows_match_finite_difference_of_Z():
    workload, r0 = _linear_descriptor_case(seed=9, n=2, d=4, D=16)
    G = oracle.force_rows_w(workload(r0))
    h = 2.0 ** -9
    for j in range(2):
        for k in range(3):
            def cd(step):
                rp, rm = r0.copy(), r0.copy()
                rp[j, k] += step; rm[j, k] -= step
                return (oracle.forward_w(workload(rp))[0] - oracle.forward_w(workload(rm))[0]) / (2 * step)
            dZ = (4.0 * cd(h / 2) - cd(h)) / 3.0
            assert np.allclose(G[3 * j + k], -dZ, rtol=0, atol=1e-8)


def test_neighbor_gradient_equals_scattered_dense():
    """Reading A13: duplicates/self indices accumulate, -1 is padding; equals the dense layout built by
    scattering the sparse entries."""
    w = tiny_workload(5, d=8, D=32, T=3, sigma=1.0, counts=[6], grad="neighbor", K=5, pad_fraction=0.3)
    n, d = w.n_atoms, w.model.d
    idx, val = w.grad.nbr_idx, w.grad.nbr_val
    assert (idx == -1).any() and any(len(set(r[r >= 0])) < (r >= 0).sum() for r in idx)   # has pads + duplicates
    dense = np.zeros((n, d, n, 3), np.float32)
    for I in range(n):
        for q in range(idx.shape[1]):
            if idx[I, q] >= 0:
                dense[I, :, idx[I, q], :] += val[I, q]
    wd = Workload(name="d", model=w.model, elem=w.elem, mol_off=w.mol_off, x=w.x, alpha=w.alpha,
                  grad=DescriptorGradient(layout="dense", dense=dense.reshape(-1),
                                          dense_off=np.array([0, dense.size], np.int64)))
    assert np.allclose(oracle.forces_w(w), oracle.forces_w(wd), atol=1e-6)     # dense sums were rounded to fp32
    assert np.allclose(oracle.force_rows_w(w), oracle.force_rows_w(wd), atol=1e-6)


# ----------------------------------------------------------------------------- segment sum (a3)
def test_segment_sum_properties():
    w = tiny_workload(12, d=16, D=64, T=2, sigma=2.0, counts=[4, 0, 1, 3], grad="none")
    Z = oracle.forward_w(w)
    assert np.all(Z[1] == 0.0)                                       # empty molecule
    I = int(w.mol_off[2])                                            # the 1-atom molecule is z itself
    u = oracle.sorf_u(w.x[I], int(w.elem[I]), 16, 64, 2, 2.0, w.model.signs)
    assert np.allclose(Z[2], np.sqrt(2 / 64) * np.cos(u + w.model.bias[w.elem[I]].astype(np.float64)), atol=1e-15)
    perm = np.arange(w.n_atoms); perm[:4] = [2, 0, 3, 1]             # permute atoms inside molecule 0
    Zp = oracle.forward(w.x[perm], w.elem[perm], w.mol_off, 16, 64, 2, 2.0, w.model.signs, w.model.bias)
    assert np.allclose(Zp, Z, atol=1e-14)


# ----------------------------------------------------------------------------- normal equations (a8)
def test_gram_matrix_identities():
    rng = np.random.default_rng(8)
    A = rng.standard_normal((300, 48)).astype(np.float32)
    y = rng.standard_normal(300).astype(np.float32)
    ZtZ, Zty = oracle.normal_equations(A, y)
    A64 = A.astype(np.float64)
    assert np.array_equal(ZtZ, ZtZ.T)
    assert np.linalg.eigvalsh(ZtZ).min() > -1e-9
    assert np.isclose(np.trace(ZtZ), np.sum(A64 ** 2), rtol=1e-13)
    v = rng.standard_normal(48)
    assert np.allclose(ZtZ @ v, A64.T @ (A64 @ v), rtol=1e-11)
    assert np.allclose(ZtZ, A64.T @ A64, rtol=1e-12, atol=1e-13)
    assert np.allclose(Zty, A64.T @ y.astype(np.float64), rtol=1e-12)
    ii = np.array([0, 5, 47], np.int32); jj = np.array([3, 5, 0], np.int32)
    assert np.allclose(oracle.gram_entries(A, ii, jj), ZtZ[ii, jj], rtol=1e-14)
    rows, ry = oracle.gram_rows(A, y, ii)
    assert np.allclose(rows, ZtZ[ii], rtol=1e-14) and np.allclose(ry, Zty[ii], rtol=1e-14)


def test_normal_equations_recover_planted_alpha():
    """Reading A8/A11: with y := [Z; G] alpha*, Zty = ZtZ alpha* (sign and row order of the force rows)."""
    w = tiny_workload(3, d=8, D=32, T=3, sigma=1.0, counts=[2, 3, 2], grad="dense")
    Z, G = oracle.forward_w(w), oracle.force_rows_w(w)
    E, F = oracle.predict_w(w)
    A = np.concatenate([Z, G]).astype(np.float32)
    y = np.concatenate([E, F.reshape(-1)]).astype(np.float32)
    ZtZ, Zty = oracle.normal_equations(A, y)
    assert np.allclose(Zty, ZtZ @ w.alpha.astype(np.float64), rtol=0, atol=5e-6)


def test_c1_golden_regression():
    """tests/golden/c1_oracle.json was written by tests/golden/make_golden.py (oracle only)."""
    import json, os
    with open(os.path.join(os.path.dirname(__file__), "golden", "c1_oracle.json")) as f:
        gold = json.load(f)
    w = make_workload("c1")
    Z = oracle.forward_w(w)
    E, F = oracle.predict_w(w)
    assert np.allclose(Z[0, :8], gold["Z_0_first8"], rtol=1e-12, atol=1e-15)
    assert np.isclose(np.linalg.norm(Z), gold["Z_fro"], rtol=1e-12)
    assert np.allclose(E[:4], gold["energy_first4"], rtol=1e-11, atol=1e-14)
    assert np.allclose(F[0], gold["forces_atom0"], rtol=1e-11, atol=1e-14)
    assert np.isclose(np.linalg.norm(F), gold["forces_fro"], rtol=1e-12)


# ----------------------------------------------------------------------------- solve (NEXT #1; eq. 16-17)
def test_solve_matches_numpy_and_residual():
    rng = np.random.default_rng(11)
    for D, rows in ((1, 3), (7, 20), (64, 200), (130, 400)):
        A = rng.standard_normal((rows, D)).astype(np.float32)
        y = rng.standard_normal(rows).astype(np.float32)
        ZtZ = (A.astype(np.float64).T @ A.astype(np.float64)).astype(np.float32)
        Zty = (A.astype(np.float64).T @ y.astype(np.float64)).astype(np.float32)
        lam = 1e-3
        alpha, info = oracle.solve(ZtZ, Zty, lam)
        assert info == 0
        M = ZtZ.astype(np.float64) + lam * np.eye(D)
        assert np.allclose(alpha, np.linalg.solve(M, Zty.astype(np.float64)), rtol=1e-9, atol=1e-12)
        assert np.linalg.norm(M @ alpha - Zty) <= 1e-10 * np.linalg.norm(Zty)


def test_solve_closed_forms_and_failure():
    d = np.array([1.0, 4.0, 0.25, 9.0], dtype=np.float32)
    b = np.array([2.0, -8.0, 1.0, 3.0], dtype=np.float32)
    alpha, info = oracle.solve(np.diag(d), b, 0.5)                      # diagonal: alpha_i = b_i / (d_i + lambda)
    assert info == 0 and np.allclose(alpha, b.astype(np.float64) / (d.astype(np.float64) + 0.5), rtol=1e-14)
    alpha, info = oracle.solve(np.zeros((3, 3), np.float32), np.ones(3, np.float32), 2.0)   # pure ridge: b / lambda
    assert info == 0 and np.allclose(alpha, 0.5)
    bad = np.array([[1.0, 2.0], [2.0, 1.0]], dtype=np.float32)          # indefinite: second minor fails
    _, info = oracle.solve(bad, np.ones(2, np.float32), 0.0)
    assert info == 2


# ---------------------------------------------------------------------------------------------------
# Per-element PCA projection (eq. 21-22): oracle.project / project_gradient
# ---------------------------------------------------------------------------------------------------
def test_project_matches_definition_and_picks_the_element_matrix():
    """x_I = rho_I^T U_e with the matrix of the atom's OWN element (a shared matrix or a transposed one fails)."""
    from workloads import projection_inputs
    pi = projection_inputs(seed=5, counts=[4, 0, 7, 1], rep=37, d=16, n_elem=3)
    x = oracle.project(pi.rho, pi.elem, pi.U)
    for I in range(pi.rho.shape[0]):
        ref = pi.rho[I].astype(np.float64) @ pi.U[pi.elem[I]].astype(np.float64)
        assert np.allclose(x[I], ref, rtol=0, atol=1e-12)
    wrong = pi.rho.astype(np.float64) @ pi.U[0].astype(np.float64)
    assert not np.allclose(x[pi.elem != 0], wrong[pi.elem != 0], atol=1e-3)


def test_project_orthonormal_columns_identities():
    """U_e^T U_e = I: a kept singular vector projects onto a unit vector, vectors in the span keep their norm, and
    every other vector gets shorter (Bessel)."""
    from workloads import projection_inputs
    pi = projection_inputs(seed=6, counts=[8], rep=40, d=8, n_elem=2)
    for e in range(2):
        Ue = pi.U[e].astype(np.float64)
        cols = np.ascontiguousarray(Ue.T).astype(np.float32)             # the 8 kept columns as "atoms"
        x = oracle.project(cols, np.full(8, e, np.int32), pi.U)
        assert np.allclose(x, np.eye(8), atol=1e-6)
        coeff = np.random.default_rng(e).standard_normal((5, 8))
        inspan = (coeff @ Ue.T).astype(np.float32)
        xs = oracle.project(inspan, np.full(5, e, np.int32), pi.U)
        assert np.allclose(np.linalg.norm(xs, axis=1), np.linalg.norm(inspan.astype(np.float64), axis=1), rtol=1e-6)
    x = oracle.project(pi.rho, pi.elem, pi.U)
    assert np.all(np.linalg.norm(x, axis=1) <= np.linalg.norm(pi.rho.astype(np.float64), axis=1) * (1 + 1e-6))
    assert np.any(np.linalg.norm(x, axis=1) < 0.9 * np.linalg.norm(pi.rho.astype(np.float64), axis=1))


def test_project_gradient_is_the_jacobian_of_the_projected_descriptor():
    """Finite differences: rho_I(r) = sum_j tanh(A_I r_j + b) is a smooth made-up descriptor whose Jacobian the test
    writes by hand; the projected gradient must equal d(rho_I^T U_e)/dr (layout (I, m, j, c), A12)."""
    from workloads import projection_inputs
    n, rep, d = 3, 10, 4
    pi = projection_inputs(seed=7, counts=[n], rep=rep, d=d, n_elem=2, with_grad=True)
    rng = np.random.default_rng(70)
    A = rng.standard_normal((n, rep, 3)); b = rng.standard_normal((n, rep))
    r0 = rng.standard_normal((n, 3))

    def rho_of(r):
        return np.stack([np.sum(np.tanh(np.einsum("kc,jc->jk", A[I], r) + b[I]), axis=0) for I in range(n)])

    drho = np.zeros((n, rep, n, 3))
    for I in range(n):
        t = np.tanh(np.einsum("kc,jc->jk", A[I], r0) + b[I])               # [j, k]
        drho[I] = np.einsum("jk,kc->kjc", 1.0 - t * t, A[I])
    gout = oracle.project_gradient(drho.astype(np.float32).ravel(), pi.drho_off, pi.elem, pi.mol_off, pi.U, pi.dx_off)
    gout = gout.reshape(n, d, n, 3)
    h = 2e-3                     # central differences: O(h^2) truncation, fp32 rounding of rho / h ~ 3e-5
    for j in range(n):
        for c in range(3):
            rp, rm = r0.copy(), r0.copy()
            rp[j, c] += h; rm[j, c] -= h
            xp = oracle.project(rho_of(rp).astype(np.float32), pi.elem, pi.U)
            xm = oracle.project(rho_of(rm).astype(np.float32), pi.elem, pi.U)
            fd = (xp - xm) / (2 * h)                                         # [I, m]
            assert np.allclose(gout[:, :, j, c], fd, atol=2e-3 * np.abs(fd).max() + 1e-5)
    ref = np.einsum("ikjc,ikm->imjc", drho.astype(np.float32).astype(np.float64),
                    pi.U[pi.elem].astype(np.float64))
    assert np.allclose(gout, ref, atol=1e-10)


# ----------------------------------------------------------------------------- dense-matrix RFF (variant f4)
def test_rff_forward_equals_sorf_forward_for_the_dense_sorf_matrix():
    """The SORF map IS a random-feature map with a particular W (eq. 20 vs eq. 14/18): feeding the explicit D x d
    matrix of every element to the RFF oracle must reproduce the SORF oracle (two code paths, independent W)."""
    w = tiny_workload(seed=5, d=16, D=64, T=3, sigma=1.5, counts=[3, 1, 4, 2], n_elem=3, grad=None)
    m = w.model
    W = np.stack([dense_W(m, e) for e in range(m.n_elem)]).astype(np.float32)      # entries c * integer: exact in fp32?
    Zs = oracle.forward_w(w)
    Zr = oracle.rff_forward(W, m.bias, w.x, w.elem, w.mol_off)
    assert np.allclose(Zr, Zs, rtol=0, atol=2e-6)      # fp32 rounding of c * integer entries of W


def test_rff_forward_brute_force_and_gaussian_kernel():
    rng = np.random.default_rng(8)
    n_elem, D, d = 2, 96, 8
    W = rng.standard_normal((n_elem, D, d)).astype(np.float32)
    b = rng.uniform(0, 2 * np.pi, size=(n_elem, D)).astype(np.float32)
    x = rng.standard_normal((7, d)).astype(np.float32)
    elem = np.array([0, 1, 1, 0, 0, 1, 0], dtype=np.int32)
    mol_off = np.array([0, 3, 3, 7], dtype=np.int32)          # an empty molecule in the middle
    Z = oracle.rff_forward(W, b, x, elem, mol_off)
    z = np.sqrt(2.0 / D) * np.cos(np.einsum("alk,ak->al", W[elem].astype(np.float64), x.astype(np.float64)) + b[elem])
    ref = np.stack([z[0:3].sum(0), np.zeros(D), z[3:7].sum(0)])
    assert np.allclose(Z, ref, rtol=1e-13, atol=1e-14)
    # eq. 12-13: E[z(x).z(y)] = exp(-|x - y|^2 / 2 sigma^2) for w ~ N(0, I / sigma^2), b ~ U[0, 2 pi]
    d, D, sigma = 16, 65536, 1.7
    Wg = (rng.standard_normal((1, D, d)) / sigma).astype(np.float32)
    bg = rng.uniform(0, 2 * np.pi, size=(1, D)).astype(np.float32)
    xa = rng.standard_normal(d)
    for delta in (0.5, 1.0, 2.0):
        dirn = rng.standard_normal(d); dirn /= np.linalg.norm(dirn)
        xy = np.stack([xa, xa + delta * sigma * dirn]).astype(np.float32)
        Zg = oracle.rff_forward(Wg, bg, xy, [0, 0], [0, 1, 2])
        k = np.exp(-np.sum((xy[0].astype(np.float64) - xy[1]) ** 2) / (2 * sigma ** 2))
        assert abs(Zg[0] @ Zg[1] - k) < 0.015
