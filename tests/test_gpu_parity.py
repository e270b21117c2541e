"""GPU parity: the CUDA path (through the C-ABI library, via the thin binding) against the FP64 oracle on the
same seeded inputs.  Tolerances are BASELINE.json:north_star's: relative Frobenius error <= 1e-5 for Z,
energies and ZtZ (also used for G and Zty), <= 1e-4 for forces.
"""
import numpy as np
import pytest

import oracle
from workloads import make_workload, tiny_workload

pytestmark = pytest.mark.gpu

TOL, TOL_F = 1e-5, 1e-4


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


def run_all(q, w, check_ne=True):
    """Runs every export on workload w and compares with the oracle."""
    pkg, wio, torch = q
    dp = wio.device_problem(w)
    Zo = oracle.forward_w(w)
    # forward
    Z = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off)
    torch.cuda.synchronize()
    assert rel(Z.cpu().numpy(), Zo) <= TOL
    Eo = oracle.energy(Zo, w.alpha)
    if w.grad is None:
        E, F = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha)
        assert F is None
        assert rel(E.cpu().numpy(), Eo) <= TOL
        return
    # forward + force rows: the register-FWHT path and (dense gradient, d = 128 / 256) the tensor-core path
    Go = oracle.force_rows_w(w)
    modes = [pkg.ROWS_FWHT]
    if w.grad.layout == "dense" and w.model.d in (128, 256):
        modes += [pkg.ROWS_MMA, pkg.ROWS_MMA2]
    for mode in modes + [pkg.ROWS_AUTO]:
        Z2, G = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off, dp.grad, force_rows_mode=mode)
        assert rel(Z2.cpu().numpy(), Zo) <= TOL
        assert rel(G.cpu().numpy(), Go) <= TOL, mode
    # predict and backward
    Fo = oracle.forces_w(w)
    E, F = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, dp.grad)
    assert rel(E.cpu().numpy(), Eo) <= TOL
    assert rel(F.cpu().numpy(), Fo) <= TOL_F
    F2 = pkg.qmll_sorf_backward_forces(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, dp.grad)
    assert rel(F2.cpu().numpy(), Fo) <= TOL_F
    # G alpha = F (JVP/VJP consistency on the GPU results themselves, in fp64 on the host)
    if F.numel() > 0:
        Ga = G.cpu().numpy().astype(np.float64) @ w.alpha.astype(np.float64)
        assert rel(Ga.reshape(-1, 3), Fo) <= TOL_F
    if check_ne:
        A = torch.cat([Z2, G]).contiguous()
        y = dp.y
        ZtZ, Zty = pkg.qmll_normal_equations(A, y)
        An = A.cpu().numpy()
        ZtZo, Ztyo = oracle.normal_equations(An, w.y)
        ZtZn = ZtZ.cpu().numpy()
        assert rel(ZtZn, ZtZo) <= TOL
        assert rel(Zty.cpu().numpy(), Ztyo) <= TOL
        assert np.array_equal(ZtZn, ZtZn.T)


def test_c1_full(q):
    run_all(q, make_workload("c1"))


@pytest.mark.parametrize("T", [1, 2, 3])
@pytest.mark.parametrize("d,D", [(16, 64), (32, 96), (64, 448), (128, 4224), (256, 1024), (512, 1024), (1024, 2048)])
def test_tiny_ragged_dense(q, d, D, T):
    # ragged molecules incl. empty ones and one longer than a chunk; D/d not a multiple of the warp's stack count
    counts = [3, 0, 1, 7, 0, 40, 2, 5]
    if d >= 512:
        counts = [3, 0, 5, 2]
    w = tiny_workload(seed=1000 + d + T, d=d, D=D, T=T, sigma=1.5 * np.sqrt(d) / 4, counts=counts, n_elem=3,
                      grad="dense", x_std=1.0)
    run_all(q, w, check_ne=(d == 64))


@pytest.mark.parametrize("d,D", [(64, 256), (128, 1024), (256, 2048)])
def test_tiny_neighbor(q, d, D):
    w = tiny_workload(seed=77 + d, d=d, D=D, T=3, sigma=np.sqrt(d) / 2, counts=[50, 0, 13], n_elem=2,
                      grad="neighbor", K=6)
    run_all(q, w, check_ne=False)


def test_force_rows_cta_pairs_one_stack_and_many_molecules(q):
    """QMLL_ROWS_MMA2 edge cases: a single stack group (the peer CTA of every pair has nothing of its own), an odd
    number of groups, more tasks than CTA pairs (persistent loop), a one-atom molecule."""
    pkg, wio, torch = q
    for d, D, counts in ((256, 256, [3, 1]), (128, 128 * 9, [6] * 40), (256, 256 * 5, [9] * 100 + [1])):
        w = tiny_workload(seed=500 + D, d=d, D=D, T=3, sigma=np.sqrt(d) / 2, counts=counts, n_elem=3, grad="dense")
        dp = wio.device_problem(w)
        _, G = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off, dp.grad, force_rows_mode=pkg.ROWS_MMA2)
        assert rel(G.cpu().numpy(), oracle.force_rows_w(w)) <= TOL, (d, D)


def test_force_rows_mma_long_molecule_and_odd_stacks(q):
    """Tensor-core force rows: a molecule whose 3n columns need several column chunks (n = 50 > 42), mixed with small
    and empty ones, unsorted elements (a W reload per atom), stack counts that are not a multiple of the warp's."""
    pkg, wio, torch = q
    for d, D in ((128, 128 * 5), (256, 256 * 3)):
        w = tiny_workload(seed=300 + d, d=d, D=D, T=3, sigma=np.sqrt(d) / 2, counts=[50, 0, 2, 17], n_elem=4,
                          grad="dense")
        dp = wio.device_problem(w)
        Go = oracle.force_rows_w(w)
        Gs = {}
        for mode in (pkg.ROWS_MMA, pkg.ROWS_MMA2, pkg.ROWS_FWHT):
            _, G = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off, dp.grad, force_rows_mode=mode)
            assert rel(G.cpu().numpy(), Go) <= TOL, (d, mode)
            Gs[mode] = G
        assert torch.equal(Gs[pkg.ROWS_MMA], Gs[pkg.ROWS_MMA2])     # CTA pairs: the same MMAs in the same order
    w = tiny_workload(seed=9, d=64, D=128, T=3, sigma=2.0, counts=[2], grad="dense")
    dp = wio.device_problem(w)
    with pytest.raises(pkg.QmllError) as ei:                      # d = 64 has no tensor-core path
        pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off, dp.grad, force_rows_mode=pkg.ROWS_MMA)
    assert ei.value.status == -2


@pytest.mark.parametrize("T", [1, 2])
def test_force_rows_mma_fewer_transforms(q, T):
    pkg, wio, torch = q
    w = tiny_workload(seed=40 + T, d=128, D=1024, T=T, sigma=4.0, counts=[5, 9], n_elem=3, grad="dense")
    dp = wio.device_problem(w)
    for mode in (pkg.ROWS_MMA, pkg.ROWS_MMA2):
        _, G = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off, dp.grad, force_rows_mode=mode)
        assert rel(G.cpu().numpy(), oracle.force_rows_w(w)) <= TOL


@pytest.mark.parametrize("rep,d,counts,n_elem", [(37, 16, [4, 0, 7, 1], 3), (384, 128, [21] * 6, 3), (431, 256, [27, 3, 40], 5),
                                                 (100, 64, [70], 2)])
def test_project_matches_oracle(q, rep, d, counts, n_elem):
    """Per-element PCA projection (eq. 21-22) of descriptors and of a dense gradient: odd rep, ragged molecules, more
    than 32 columns per atom, several elements inside one 32-atom tile."""
    pkg, wio, torch = q
    from workloads import projection_inputs
    pi = projection_inputs(seed=rep + d, counts=counts, rep=rep, d=d, n_elem=n_elem, with_grad=True)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    x, g = pkg.qmll_project(t(pi.rho), t(pi.elem), t(pi.U), t(pi.mol_off), t(pi.drho), t(pi.drho_off), t(pi.dx_off))
    assert rel(x.cpu().numpy(), oracle.project(pi.rho, pi.elem, pi.U)) <= TOL
    go = oracle.project_gradient(pi.drho, pi.drho_off, pi.elem, pi.mol_off, pi.U, pi.dx_off)
    assert rel(g.cpu().numpy(), go) <= TOL
    x2, none = pkg.qmll_project(t(pi.rho), t(pi.elem), t(pi.U))
    assert none is None and torch.equal(x2, x)


def test_project_then_sorf_forward(q):
    """The projected descriptor and gradient feed the SORF path unchanged: Z, G from raw representations."""
    pkg, wio, torch = q
    from workloads import projection_inputs
    w = tiny_workload(seed=77, d=128, D=512, T=3, sigma=3.0, counts=[5, 8], n_elem=3, grad="dense")
    pi = projection_inputs(seed=78, counts=[5, 8], rep=200, d=128, n_elem=3, with_grad=True)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    x, g = pkg.qmll_project(t(pi.rho), t(w.elem), t(pi.U), t(w.mol_off), t(pi.drho), t(pi.drho_off), t(pi.dx_off))
    dp = wio.device_problem(w)
    Z, G = pkg.qmll_sorf_forward(dp.params, x, dp.elem, dp.mol_off, pkg.Grad.make_dense(g, t(pi.dx_off)))
    xo = oracle.project(pi.rho, w.elem, pi.U).astype(np.float32)
    go = oracle.project_gradient(pi.drho, pi.drho_off, w.elem, w.mol_off, pi.U, pi.dx_off).astype(np.float32)
    m = w.model
    Zo = oracle.forward(xo, w.elem, w.mol_off, m.d, m.D, m.T, m.sigma, m.signs, m.bias)
    Go = oracle.force_rows_dense(xo, w.elem, w.mol_off, m.d, m.D, m.T, m.sigma, m.signs, m.bias, go, pi.dx_off)
    assert rel(Z.cpu().numpy(), Zo) <= 2 * TOL          # two fp32 stages chained (projection, then SORF)
    assert rel(G.cpu().numpy(), Go) <= 2 * TOL


def test_c2_reduced(q):
    run_all(q, make_workload("c2", n_mol=12, D=2048))


def test_c3_reduced(q):
    run_all(q, make_workload("c3", n_mol=700, D=4096))


def test_c4_reduced(q):
    run_all(q, make_workload("c4", n_mol=6, D=2048), check_ne=False)
    run_all(q, make_workload("c4", n_mol=4, D=1024, part="infer"), check_ne=False)


def test_c5_reduced(q):
    run_all(q, make_workload("c5", n_atoms=1500, D=4096, K=8), check_ne=False)  # c5 is inference only (no y rows)


def test_empty_inputs(q):
    pkg, wio, torch = q
    w = tiny_workload(seed=5, d=64, D=128, T=3, sigma=2.0, counts=[0, 0], grad=None)
    dp = wio.device_problem(w)
    Z = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off)
    assert Z.shape == (2, 128) and float(Z.abs().max()) == 0.0
    E, _ = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha)
    assert float(E.abs().max()) == 0.0


@pytest.mark.parametrize("mode", [0, 1, 2])   # QMLL_NE_SPLIT_F16, QMLL_NE_SPLIT_TF32, QMLL_NE_SPLIT_F16_PAIRS
@pytest.mark.parametrize("rows,D", [(1, 256), (777, 384), (1500, 128), (2500, 520), (4096, 1024), (300, 451), (130, 7)])
def test_normal_equations_shapes(q, rows, D, mode):
    pkg, wio, torch = q
    rng = np.random.default_rng(rows + D)
    # correlated, non-zero-mean rows (like Z of near-identical molecules): the hard case for fp32 accumulation
    A = (0.7 + 0.3 * rng.standard_normal((rows, D))).astype(np.float32)
    y = rng.standard_normal(rows).astype(np.float32)
    Ad, yd = torch.from_numpy(A).cuda(), torch.from_numpy(y).cuda()
    ZtZ, Zty = pkg.qmll_normal_equations(Ad, yd, mode=mode)
    ZtZo, Ztyo = oracle.normal_equations(A, y)
    assert rel(ZtZ.cpu().numpy(), ZtZo) <= TOL
    assert rel(Zty.cpu().numpy(), Ztyo) <= TOL
    # accumulate a second block, with a workspace that forces several panels
    B = rng.standard_normal((rows, D)).astype(np.float32)
    yb = rng.standard_normal(rows).astype(np.float32)
    pkg.qmll_normal_equations(torch.from_numpy(B).cuda(), torch.from_numpy(yb).cuda(), ZtZ=ZtZ, Zty=Zty,
                              accumulate=True, workspace_limit=0, mode=mode)
    ZtZo2, Ztyo2 = oracle.normal_equations(B, yb)
    Zn = ZtZ.cpu().numpy()
    assert rel(Zn, ZtZo + ZtZo2) <= TOL
    assert rel(Zty.cpu().numpy(), Ztyo + Ztyo2) <= TOL
    assert np.array_equal(Zn, Zn.T)


def test_normal_equations_cta_pairs_are_bit_identical(q):
    """QMLL_NE_SPLIT_F16_PAIRS issues the same MMAs in the same order on cta_group::2: identical bits, also across
    several row panels and an odd number of 128-column tiles (the last pair has a CTA without a tile)."""
    pkg, wio, torch = q
    torch.manual_seed(4)
    for rows, D in ((3000, 384), (70000, 640), (900, 2176)):
        A = (0.3 + torch.randn((rows, D), device="cuda")).contiguous()
        y = torch.randn((rows,), device="cuda")
        Z1, t1 = pkg.qmll_normal_equations(A, y, mode=pkg.NE_SPLIT_F16)
        Z2, t2 = pkg.qmll_normal_equations(A, y, mode=pkg.NE_SPLIT_F16_PAIRS)
        assert torch.equal(Z1, Z2) and torch.equal(t1, t2), (rows, D)


def test_normal_equations_wide_dynamic_range(q):
    """Rows whose magnitudes differ by 2^40 and columns by 2^20 (energy rows next to tiny force rows): the fp16
    container's per-(chunk, column block) power-of-two scales must keep the relative Frobenius accuracy."""
    pkg, wio, torch = q
    rng = np.random.default_rng(99)
    rows, D = 1000, 512
    A = rng.standard_normal((rows, D))
    A *= np.exp2(rng.integers(-20, 20, size=(rows // 125, 1)).repeat(125, axis=0))   # per 125-row group (straddles chunks)
    A *= np.exp2(rng.integers(-10, 10, size=(1, D)))
    A = A.astype(np.float32)
    y = rng.standard_normal(rows).astype(np.float32)
    ZtZo, Ztyo = oracle.normal_equations(A, y)
    for mode in (0, 1):
        ZtZ, Zty = pkg.qmll_normal_equations(torch.from_numpy(A).cuda(), torch.from_numpy(y).cuda(), mode=mode)
        assert rel(ZtZ.cpu().numpy(), ZtZo) <= TOL
        assert rel(Zty.cpu().numpy(), Ztyo) <= TOL
    # every 128 x 128 block of the result individually (the scales are per block)
    Zn = ZtZ.cpu().numpy()
    ZtZ16, _ = pkg.qmll_normal_equations(torch.from_numpy(A).cuda(), torch.from_numpy(y).cuda(), mode=0)
    Z16 = ZtZ16.cpu().numpy()
    for i in range(0, D, 128):
        for j in range(0, D, 128):
            assert rel(Z16[i:i + 128, j:j + 128], ZtZo[i:i + 128, j:j + 128]) <= TOL


@pytest.mark.parametrize("D", [1, 33, 520, 2048])
def test_pack_unpack_lower_triangle(q, D):
    """The multi-GPU exchange helpers: row-packed lower triangle and its symmetric unpack (bit-exact data movement)."""
    pkg, wio, torch = q
    from paper_2206_01580_b200.distributed import pack_lower_reference
    g = torch.Generator(device="cuda").manual_seed(D)
    S = torch.randn((D, D), device="cuda", generator=g)
    S = (S + S.T).contiguous()
    packed = pkg.qmll_pack_lower(S)
    assert torch.equal(packed, pack_lower_reference(S))
    out = torch.full((D, D), float("nan"), device="cuda")
    pkg.qmll_unpack_lower(packed, out)
    assert torch.equal(out, S)


def test_normal_equations_zero_rows(q):
    pkg, wio, torch = q
    A = torch.empty((0, 256), dtype=torch.float32, device="cuda")
    y = torch.empty((0,), dtype=torch.float32, device="cuda")
    ZtZ, Zty = pkg.qmll_normal_equations(A, y)
    assert float(ZtZ.abs().max()) == 0.0 and float(Zty.abs().max()) == 0.0


def test_error_codes(q):
    pkg, wio, torch = q
    w = tiny_workload(seed=9, d=64, D=128, T=3, sigma=2.0, counts=[2], grad="dense")
    dp = wio.device_problem(w)
    bad = pkg.SorfParams(d=48, D=96, n_transform=3, n_elem=3, sigma=1.0, signs=dp.params.signs, bias=dp.params.bias)
    with pytest.raises(pkg.QmllError) as ei:
        pkg.qmll_sorf_forward(bad, dp.x, dp.elem, dp.mol_off)
    assert ei.value.status == -1
    bad2 = pkg.SorfParams(d=64, D=128, n_transform=4, n_elem=3, sigma=1.0, signs=dp.params.signs, bias=dp.params.bias)
    with pytest.raises(pkg.QmllError):
        pkg.qmll_sorf_forward(bad2, dp.x, dp.elem, dp.mol_off)


@pytest.mark.parametrize("D,rows", [(1, 4), (37, 100), (50, 300), (256, 448), (321, 700), (577, 900), (1000, 3000),
                                    (4096, 6000)])
def test_solve_matches_oracle(q, D, rows):
    """qmll_solve (blocked FP64 Cholesky) against the oracle's unblocked one on the same fp32 ZtZ / Zty."""
    pkg, wio, torch = q
    rng = np.random.default_rng(D)
    A = rng.standard_normal((rows, D)).astype(np.float32)
    y = rng.standard_normal(rows).astype(np.float32)
    ZtZ = (A.astype(np.float64).T @ A.astype(np.float64)).astype(np.float32)
    Zty = (A.astype(np.float64).T @ y.astype(np.float64)).astype(np.float32)
    lam = 1e-2
    alpha, info = pkg.qmll_solve(torch.from_numpy(ZtZ).cuda(), torch.from_numpy(Zty).cuda(), lam)
    ao, io = oracle.solve(ZtZ, Zty, lam)
    assert int(info.item()) == 0 and io == 0
    assert rel(alpha.cpu().numpy(), ao) <= 1e-6          # fp32 output of an FP64 solve


def test_solve_reports_non_positive_definite(q):
    pkg, wio, torch = q
    bad = torch.tensor([[1.0, 2.0], [2.0, 1.0]], device="cuda")
    _, info = pkg.qmll_solve(bad, torch.ones(2, device="cuda"), 0.0)
    assert int(info.item()) == 2
    # the first bad pivot lies in a later panel (order 334 = second 256-wide panel, second 64-wide step)
    diag = torch.ones(600, device="cuda")
    diag[333] = -1.0
    diag[500] = -1.0
    _, info = pkg.qmll_solve(torch.diag(diag), torch.ones(600, device="cuda"), 0.0)
    assert int(info.item()) == 334


def test_solve_is_bit_reproducible_across_repeats_and_streams(q):
    """The look-ahead fork / join and the flag hand-over of the backward substitution leave no room for a race: every
    element of the factor has one writer, so repeated solves (alternating streams) must be bit-identical."""
    pkg, wio, torch = q
    g = torch.Generator(device="cuda").manual_seed(11)
    for D in (577, 1000, 2048):
        A = torch.randn((D + 300, D), device="cuda", generator=g) / D ** 0.5
        ZtZ = A.T @ A
        Zty = torch.randn((D,), device="cuda", generator=g)
        ref, info = pkg.qmll_solve(ZtZ, Zty, 1e-3)
        torch.cuda.synchronize()
        assert int(info.item()) == 0
        s = torch.cuda.Stream()
        for k in range(24):
            if k % 2:
                with torch.cuda.stream(s):
                    a, _ = pkg.qmll_solve(ZtZ, Zty, 1e-3)
                s.synchronize()
            else:
                a, _ = pkg.qmll_solve(ZtZ, Zty, 1e-3)
                torch.cuda.synchronize()
            assert torch.equal(a, ref)


def test_solve_on_a_side_stream_and_under_graph_capture(q):
    """qmll_solve forks panel work onto an internal stream (look-ahead): the result must not depend on the caller's
    stream, and the fork / join must be capturable."""
    pkg, wio, torch = q
    rng = np.random.default_rng(5)
    D = 700
    A = rng.standard_normal((1500, D)).astype(np.float32)
    ZtZ = torch.from_numpy((A.T @ A).astype(np.float32)).cuda()
    Zty = torch.from_numpy((A.T @ rng.standard_normal(1500).astype(np.float32))).cuda()
    ref, info = pkg.qmll_solve(ZtZ, Zty, 1e-2)
    assert int(info.item()) == 0
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        for _ in range(3):
            a2, _ = pkg.qmll_solve(ZtZ, Zty, 1e-2)
    s.synchronize()
    assert torch.equal(a2, ref)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        a3, _ = pkg.qmll_solve(ZtZ, Zty, 1e-2)          # warm-up on the capture stream (workspace allocation)
    s.synchronize()
    with torch.cuda.graph(g, stream=s):
        a3, info3 = pkg.qmll_solve(ZtZ, Zty, 1e-2)
    a3.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(a3, ref) and int(info3.item()) == 0


def test_train_then_predict_recovers_targets(q):
    """Closes the loop on config 1: y := [Z; G] alpha*, normal equations, solve, predict -> E, F reproduce y."""
    pkg, wio, torch = q
    w = make_workload("c1", D=256)
    dp = wio.device_problem(w)
    Z, G = pkg.qmll_sorf_forward(dp.params, dp.x, dp.elem, dp.mol_off, dp.grad)
    A = torch.cat([Z, G]).contiguous()
    y = (A.double() @ dp.alpha.double()).float()
    ZtZ, Zty = pkg.qmll_normal_equations(A, y)
    lam = 1e-9 * float(torch.trace(ZtZ)) / 256
    alpha, info = pkg.qmll_solve(ZtZ, Zty, lam)
    assert int(info.item()) == 0
    E, F = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, alpha, dp.grad)
    pred = torch.cat([E, F.reshape(-1)]).cpu().numpy()
    assert rel(pred, y.cpu().numpy()) <= 1e-3
