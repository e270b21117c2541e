"""qmll_predict_static (include/qmll.h): qmll_predict on the library's static device scratch, for callers that cannot
allocate.  Checked against the existing workspace path (qmll_predict, itself checked against the FP64 oracle in
test_gpu_parity.py / test_gpu_fullsize.py) within the tolerances those tests use, on calls in a row whose problems
differ in size, d, D and gradient layout -- so that anything a call left in the shared scratch would show.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

from workloads import make_workload, tiny_workload

pytestmark = pytest.mark.gpu

TOL, TOL_F = 1e-5, 1e-4          # relative Frobenius error: energies, forces


def rel(a, b):
    a = a.double().cpu().numpy()
    b = b.double().cpu().numpy()
    den = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / den) if den > 0 else float(np.linalg.norm(a))


@pytest.fixture(scope="module")
def q():
    import torch
    import paper_2206_01580_b200 as pkg
    from paper_2206_01580_b200 import workload_io
    pkg.load_library()
    assert torch.cuda.is_available()
    yield pkg, workload_io, torch
    pkg.release_workspaces()
    torch.cuda.empty_cache()


def both_paths(q, dp, with_forces=True):
    """(E, F) of the existing path and of the static-scratch entry point; the latter's outputs start as NaN."""
    pkg, wio, torch = q
    n_mol, n_atoms = dp.mol_off.numel() - 1, dp.x.shape[0]
    grad = dp.grad if with_forces else None
    E_ref, F_ref = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, grad)
    E = torch.full((n_mol,), float("nan"), dtype=torch.float32, device="cuda")
    F = torch.full((n_atoms, 3), float("nan"), dtype=torch.float32, device="cuda") if with_forces else None
    pkg.qmll_predict_static(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, E, grad, F)
    torch.cuda.synchronize()
    return E_ref, F_ref, E, F


def check(q, dp, with_forces=True):
    E_ref, F_ref, E, F = both_paths(q, dp, with_forces)
    assert bool(q[2].isfinite(E).all())
    assert rel(E, E_ref) <= TOL
    if with_forces:
        assert bool(q[2].isfinite(F).all())
        assert rel(F, F_ref) <= TOL_F


def test_static_scratch_matches_the_workspace_path_on_calls_in_a_row(q):
    pkg, wio, torch = q
    big = wio.device_problem(make_workload("c2", n_mol=300))                     # d 128, D 8192, dense gradients
    small = wio.device_problem(tiny_workload(seed=5, d=64, D=512, T=2, sigma=2.0, counts=[4, 0, 7, 1, 0, 9], n_elem=3,
                                             grad="neighbor", K=5))             # ragged, empty molecules, neighbour layout
    wide = wio.device_problem(tiny_workload(seed=6, d=256, D=2048, T=3, sigma=6.0, counts=[3, 12, 5], n_elem=4,
                                            grad="dense"))                      # d 256: cross-lane stages
    for dp in (big, small, big, wide, small):                                  # every call after a different one
        check(q, dp)
    check(q, small)                                                             # and the same problem twice in a row
    check(q, big, with_forces=False)                                            # energies only (no gradient, no forces)
    check(q, big)


def test_static_scratch_call_allocates_no_device_memory(q):
    """cudaMemGetInfo before and after a (repeated, so every kernel is already loaded) call: nothing was allocated."""
    pkg, wio, torch = q
    dp = wio.device_problem(make_workload("c1"))
    n_mol, n_atoms = dp.mol_off.numel() - 1, dp.x.shape[0]
    E = torch.empty((n_mol,), dtype=torch.float32, device="cuda")
    F = torch.empty((n_atoms, 3), dtype=torch.float32, device="cuda")
    pkg.qmll_predict_static(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, E, dp.grad, F)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    allocated0 = torch.cuda.memory_allocated()
    for _ in range(3):
        pkg.qmll_predict_static(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, E, dp.grad, F)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0 and torch.cuda.memory_allocated() == allocated0      # free device memory did not shrink
    E_ref, F_ref = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, dp.grad)
    assert rel(E, E_ref) <= TOL and rel(F, F_ref) <= TOL_F


def test_static_scratch_rejects_problems_beyond_its_size(q):
    pkg, wio, torch = q
    lib = pkg.load_library()
    assert int(lib.qmll_predict_static_max_bytes()) == 4 << 20
    n_mol = 600_000                                       # FP64 energy accumulators alone: 4.8 MB > 4 MiB
    w = tiny_workload(seed=9, d=16, D=64, T=1, sigma=1.0, counts=np.ones(n_mol, dtype=np.int32), n_elem=2, grad=None)
    dp = wio.device_problem(w)
    E = torch.full((n_mol,), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(pkg.QmllError) as ei:
        pkg.qmll_predict_static(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, E)
    assert ei.value.status == -3 and "static" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((E == 7.0).all())                         # nothing was launched
    E_ref, _ = pkg.qmll_predict(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha)     # the workspace path takes it
    assert bool(torch.isfinite(E_ref).all())
    with pytest.raises(ValueError):
        pkg.qmll_predict_static(dp.params, dp.x, dp.elem, dp.mol_off, dp.alpha, None)
