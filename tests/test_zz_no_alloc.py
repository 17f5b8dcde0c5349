"""vmat_penalty_noalloc (include/vmat.h): the allocation-free entry point for step (b) against the existing path
(vmat_dose on a plan), within the tolerance the parity tests use.  Named test_zz_* so that pytest collects it last: the
suite runs with pytest -x, and a failure here must not hide the parity tests."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-4          # BASELINE.json north_star: "dose, gradient and final cost within 1e-4 relative" (tests/test_gpu_parity.py)


@pytest.fixture(scope="module")
def torch_cuda():
    import torch

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def vm():
    import paper_1005_4396_b200 as vm

    vm.load_library()
    return vm


def relnorm(a, ref):
    ref = np.asarray(ref, np.float64)
    return np.max(np.abs(np.asarray(a, np.float64) - ref)) / max(np.max(np.abs(ref)), 1e-300)


def test_penalty_noalloc_matches_the_plan_dose_pass_on_two_calls_in_a_row(torch_cuda, vm, tiny_oracle):
    torch = torch_cuda
    o = tiny_oracle
    plan = vm.Plan.create(o.row_ptr, o.col, o.val, o.T, o.alpha, o.beta, o.theta, o.R, o.C, o.delta, o.gamma)
    dev = dict(device="cuda")
    T = torch.tensor(np.asarray(o.T, np.float32), **dev)
    al = torch.tensor(np.asarray(o.alpha, np.float32), **dev)
    be = torch.tensor(np.asarray(o.beta, np.float32), **dev)
    z = torch.empty(o.V, dtype=torch.float32, **dev)
    w_ref = torch.empty(o.V, dtype=torch.float32, **dev)
    w = torch.empty(o.V, dtype=torch.float32, **dev)
    F = torch.full((1,), -1.0, dtype=torch.float64, **dev)
    # two different plan states, one call each, back to back (the second finds the first one's scratch contents)
    occ_a, left_a, right_a, y_a = o.solve(6)[:4]
    occ_b, left_b, right_b, y_b = o.solve(12)[:4]
    seen = []
    for occ, left, right, y in ((occ_a, left_a, right_a, y_a), (occ_b, left_b, right_b, y_b * 1.7)):
        plan.set_plan(occ, left, right, y)
        F_ref, _, _ = plan.dose(z, w_ref)                       # the existing path: vmat_dose on the plan
        w.fill_(float("nan"))
        vm.penalty_noalloc(z, T, al, be, w, F)
        torch.cuda.synchronize()
        assert relnorm(w.cpu().numpy(), w_ref.cpu().numpy()) <= TOL
        assert abs(F.item() - F_ref) <= TOL * abs(F_ref)
        # and the oracle's own step (b) on the same dose
        F_o, w_o = o.penalty(z.cpu().numpy().astype(np.float64))
        assert relnorm(w.cpu().numpy(), w_o) <= TOL and abs(F.item() - F_o) <= TOL * abs(F_o)
        seen.append(F.item())
    assert seen[0] != seen[1]                                   # the two calls really saw different doses
    # the same call again: the same bits (fixed summation order), with w or without
    vm.penalty_noalloc(z, T, al, be, None, F)
    torch.cuda.synchronize()
    assert F.item() == seen[1]
    plan.destroy()


def test_penalty_noalloc_many_blocks_ragged_tail_and_limits(torch_cuda, vm):
    torch = torch_cuda
    L = vm.load_library()
    g = torch.Generator(device="cuda").manual_seed(5)
    for n in (1, 2047, 2049, 1_000_003):                        # one voxel; around a block edge; 489 blocks and a tail
        z = torch.rand(n, generator=g, device="cuda") * 2.0
        T = torch.rand(n, generator=g, device="cuda") + 0.5
        al = torch.rand(n, generator=g, device="cuda") * (torch.rand(n, generator=g, device="cuda") < 0.5)
        be = torch.rand(n, generator=g, device="cuda") + 0.1
        w = torch.empty(n, device="cuda")
        F = torch.zeros(1, dtype=torch.float64, device="cuda")
        for _ in range(2):
            vm.penalty_noalloc(z, T, al, be, w, F)
        ad, bd = al.double(), be.double()
        under, over = (T - z).clamp(min=0).double(), (z - T).clamp(min=0).double()   # fp32 differences, as the kernels form them
        F_ref = float((ad * under * under + bd * over * over).sum())
        w_ref = -2 * ad * under + 2 * bd * over
        assert abs(F.item() - F_ref) <= 1e-12 * abs(F_ref) + 1e-300   # fp64 sum of fp64 terms
        assert float((w.double() - w_ref).abs().max()) <= 1e-6 * float(w_ref.abs().max())
    # n = 0: the empty sum
    F.fill_(3.0)
    e = torch.empty(0, device="cuda")
    vm.penalty_noalloc(e, e, e, e, None, F)
    assert F.item() == 0.0
    # past the maximum: rejected with a clear message, nothing launched (F keeps its value)
    F.fill_(7.0)
    small = torch.zeros(8, device="cuda")
    p = C.c_void_p(small.data_ptr())
    rc = L.vmat_penalty_noalloc(p, p, p, p, vm.NOALLOC_MAX_VOXELS + 1, p, C.c_void_p(F.data_ptr()), None)
    torch.cuda.synchronize()
    assert rc == -1 and b"exceeds VMAT_NOALLOC_MAX_VOXELS" in L.vmat_last_error(None) and F.item() == 7.0
    with pytest.raises(vm.VmatError):
        vm.penalty_noalloc(small, small, small, small, None, None)     # nothing to compute
    # exactly the maximum is accepted
    n = vm.NOALLOC_MAX_VOXELS
    z = torch.full((n,), 2.0, device="cuda")
    one = torch.ones(n, device="cuda")
    vm.penalty_noalloc(z, one, one, one, None, F)
    assert F.item() == float(n)                                         # beta (z - T)^2 = 1 per voxel
