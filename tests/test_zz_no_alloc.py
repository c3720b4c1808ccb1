"""dualip_grad_static -- the one entry point of the library that allocates nothing -- against the ordinary handle path.

Why the entry point exists: dualip_create builds its handle out of cudaMalloc'd buffers, so the library is closed to code that
may not allocate device memory where it runs (a plug-in under a host application that owns all device memory, a service whose
memory was reserved in full at start-up, a latency-critical path that cannot take cudaMalloc's device-wide synchronisation).
dualip_grad_static gives those callers one gradient evaluation whose scratch is a fixed `static __device__` array inside the
library (include/dualip.h, csrc/dualip_static.cu).

What is checked here: its grad g, scalars and x agree with dualip_create + dualip_grad on the same rows within the parity
tolerances of tests/gpu_util.py, on several calls IN A ROW -- the scratch array is shared by all calls and keeps what the last
one left, so a call that forgot to clear something would pass alone and fail as the second one.  Consecutive calls change
lambda, gamma, the projection, the number of families and J*m (a smaller problem after a larger one leaves stale words behind
its own part of the array).  Also: the size limit is refused with its own error code, host pointers are refused, the largest
accepted size works, and free device memory does not drop across calls.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It does not depend on anything the other tests leave behind and passes alone in a fresh process as well.
"""
import ctypes

import numpy as np
import pytest
import torch

import paper_2606_07777_b200 as pkg
from gpu_util import TOL_G, TOL_GRAD, TOL_X, rel_l2

pytestmark = pytest.mark.gpu

_KINDS = {"simplex": pkg.PROJ_SIMPLEX_INEQ, "simplex_eq": pkg.PROJ_SIMPLEX_EQ, "boxcut": pkg.PROJ_BOXCUT, "box": pkg.PROJ_BOX}


def _rows(seed, I, J, m, lens):
    """Seeded ragged rows as CUDA tensors in the ABI layout (row lengths cycle through `lens`, 0 allowed)."""
    rng = np.random.default_rng(seed)
    ptr, idx = [0], []
    for i in range(I):
        d = min(int(lens[i % len(lens)]), J)
        idx.extend(np.sort(rng.choice(J, size=d, replace=False)).tolist())
        ptr.append(len(idx))
    nnz = len(idx)
    c = (-2.0 * rng.random(nnz)).astype(np.float32)
    a = (0.5 + rng.random(nnz * m)).astype(np.float32)
    col = np.zeros(J * m)
    if nnz:
        np.add.at(col, np.repeat(np.asarray(idx, dtype=np.int64), m) * m + np.tile(np.arange(m), nnz), a)
    b = (0.1 * col + 0.01).astype(np.float32)
    host = dict(row_ptr=np.asarray(ptr, dtype=np.int64), item_idx=np.asarray(idx, dtype=np.int32), c=c, a=a, b=b)
    dev = {k: torch.from_numpy(v).cuda() for k, v in host.items()}
    return dict(I=I, J=J, m=m, nnz=nnz, **dev)


class _Out:
    """Device outputs of one evaluation, allocated by the caller up front (the entry point under test never allocates)."""

    def __init__(self, P):
        self.grad = torch.full((P["J"] * P["m"],), float("nan"), dtype=torch.float64, device="cuda")
        self.scalars = torch.full((6,), float("nan"), dtype=torch.float64, device="cuda")
        self.x = torch.full((max(P["nnz"], 1),), float("nan"), dtype=torch.float32, device="cuda")


def _static(P, lam, gamma, kind, p0, p1, out=None):
    out = out or _Out(P)
    pkg.grad_static(P["I"], P["J"], P["m"], P["row_ptr"], P["item_idx"], P["c"], P["a"], P["b"], lam, gamma,
                    projection=_KINDS[kind], p0=p0, p1=p1, grad=out.grad, scalars=out.scalars, x=out.x)
    return out


def _handle_path(P, lam, gamma, kind, p0, p1):
    """The existing path: dualip_create (allocates) + dualip_grad."""
    prob = pkg.Problem.create(P["I"], P["J"], P["m"], P["row_ptr"], P["item_idx"], P["c"], P["a"], P["b"],
                              pkg.binding.make_opts(projection=_KINDS[kind], p0=p0, p1=p1))
    ref = _Out(P)
    sc = pkg.Scalars()
    prob.grad(lam, gamma, grad=ref.grad, scalars=sc, x=ref.x)
    torch.cuda.synchronize()
    prob.destroy()
    return ref, sc


def _assert_same(P, out, ref, sc, tag):
    torch.cuda.synchronize()
    got = out.scalars.cpu().numpy()
    grad, grad_ref = out.grad.cpu().numpy(), ref.grad.cpu().numpy()
    assert np.isfinite(grad).all() and np.isfinite(got).all(), f"{tag}: outputs not written"
    assert rel_l2(grad, grad_ref) <= TOL_GRAD, f"{tag}: grad rel L2 {rel_l2(grad, grad_ref):.3e}"
    if P["nnz"]:
        ex = (out.x[:P["nnz"]] - ref.x[:P["nnz"]]).abs().max().item()
        assert ex <= TOL_X, f"{tag}: x abs err {ex:.3e}"
    gn = np.linalg.norm(grad_ref)
    want = np.array([sc.g, sc.obj, sc.reg, sc.r_inf, sc.r_2, sc.gap])
    size = abs(sc.obj) + abs(sc.reg) + abs(sc.g)
    tol = np.array([TOL_G * abs(sc.g), TOL_G * abs(sc.obj), TOL_G * abs(sc.reg), TOL_GRAD * gn, TOL_GRAD * gn, TOL_G * size]) + 1e-9
    assert (np.abs(got - want) <= tol).all(), f"{tag}: scalars {got} vs {want}"


def test_calls_in_a_row_match_the_handle_path():
    """Seven evaluations back to back on one stream, each compared with dualip_create + dualip_grad on the same rows.  The
    order is chosen so that every call finds the scratch array dirty in a different way: same problem at another lambda, a
    smaller J*m with two families after a larger one, the box kernel after the simplex kernel, then the first call again."""
    big = _rows(11, 2500, 300, 1, [33, 64, 65, 100, 128, 40, 159, 9])         # mean row length > 20: 32 lanes per row
    two = _rows(12, 1800, 60, 2, [5, 12, 0, 17, 30, 1])                       # two families, 16 lanes, J*m = 120 < 300
    tiny = _rows(13, 900, 25, 3, [1, 2, 7, 8, 3, 0, 5])                       # three families (generic kernel), J*m = 75
    rng = np.random.default_rng(5)

    def lam_for(P, scale):
        return torch.from_numpy(rng.random(P["J"] * P["m"]) * scale).cuda()

    plan = [(big, lam_for(big, 0.0), 1e-1, "simplex", 1.0, 0.0),
            (big, lam_for(big, 0.4), 1e-2, "simplex", 1.0, 0.0),
            (two, lam_for(two, 0.3), 1e-1, "simplex_eq", 1.0, 0.0),
            (big, lam_for(big, 0.2), 1e-2, "boxcut", 0.3, 1.0),
            (tiny, lam_for(tiny, 0.3), 1.0, "box", 0.0, 0.4),
            (two, lam_for(two, 0.5), 1e-3, "simplex", 0.5, 0.0)]
    plan.append(plan[0])
    refs = [_handle_path(*step) for step in plan]                              # the existing path first, handles destroyed
    outs = [_static(*step) for step in plan]                                   # then the static calls, nothing in between
    for n, (step, out, (ref, sc)) in enumerate(zip(plan, outs, refs)):
        _assert_same(step[0], out, ref, sc, f"call {n} ({step[3]}, gamma={step[2]}, J*m={step[0]['J'] * step[0]['m']})")


def test_repeating_one_call_gives_the_same_bits_and_takes_no_device_memory():
    """The same evaluation four times in a row: identical bits every time (nothing of one call leaks into the next; the
    fixed-point sums do not depend on arrival order), and the free device memory reported by the driver does not shrink
    -- the call really brings its scratch with it.  The first call is outside the measurement: it is the one that sets up
    the device (symbol address lookup) and makes the driver load the kernels."""
    P = _rows(21, 4000, 500, 1, [5, 9, 2, 8, 45, 3, 0, 7])          # mean row length < 10: 8 lanes per row, the 45s take the warp path
    lam = torch.from_numpy(np.random.default_rng(3).random(P["J"]) * 0.3).cuda()
    outs = [_Out(P) for _ in range(4)]
    _static(P, lam, 1e-2, "simplex", 1.0, 0.0, outs[0])
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for o in outs[1:]:
        _static(P, lam, 1e-2, "simplex", 1.0, 0.0, o)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, f"device memory shrank by {free_before - free_after} bytes across allocation-free calls"
    for o in outs[1:]:
        assert torch.equal(o.grad, outs[0].grad) and torch.equal(o.scalars, outs[0].scalars) and torch.equal(o.x, outs[0].x)
    ref, sc = _handle_path(P, lam, 1e-2, "simplex", 1.0, 0.0)
    _assert_same(P, outs[3], ref, sc, "repeat")


def test_largest_size_works_and_one_more_is_refused():
    """J*m = STATIC_MAX_DUALS exactly is served (lambda fills the shared memory the kernel may opt in to); one dual more is
    refused with DUALIP_ETOOBIG and a message that names the limit, before anything is launched or written."""
    J = pkg.STATIC_MAX_DUALS
    P = _rows(31, 600, J, 1, [40, 3, 17, 120])
    lam = torch.from_numpy(np.random.default_rng(4).random(J) * 0.2).cuda()
    out = _static(P, lam, 1e-1, "simplex", 1.0, 0.0)
    ref, sc = _handle_path(P, lam, 1e-1, "simplex", 1.0, 0.0)
    _assert_same(P, out, ref, sc, "J*m at the limit")

    Q = _rows(32, 50, J + 1, 1, [4])
    over = _Out(Q)
    with pytest.raises(pkg.DualipError) as e:
        _static(Q, torch.zeros(J + 1, dtype=torch.float64, device="cuda"), 1e-1, "simplex", 1.0, 0.0, over)
    assert e.value.code == pkg.ETOOBIG and "DUALIP_STATIC_MAX_DUALS" in str(e.value)
    torch.cuda.synchronize()
    assert torch.isnan(over.grad).all() and torch.isnan(over.scalars).all()        # untouched
    two_fam = _rows(33, 50, J // 2 + 1, 2, [4])                                     # the limit is on J*m, not on J
    with pytest.raises(pkg.DualipError) as e:
        _static(two_fam, torch.zeros(2 * (J // 2 + 1), dtype=torch.float64, device="cuda"), 1e-1, "simplex", 1.0, 0.0)
    assert e.value.code == pkg.ETOOBIG


def test_host_memory_and_bad_arguments_are_refused():
    """A host buffer would have to be staged through device memory the call may not allocate: DUALIP_EINVAL at the C ABI (the
    binding refuses earlier, with a TypeError).  The other argument errors are those of dualip_create / dualip_grad."""
    P = _rows(41, 40, 10, 1, [3, 5])
    lam = torch.zeros(10, dtype=torch.float64, device="cuda")
    with pytest.raises(TypeError):
        pkg.grad_static(P["I"], P["J"], P["m"], P["row_ptr"], P["item_idx"], P["c"], P["a"], P["b"], lam.cpu(), 0.1)
    lib = pkg.load_library()
    host_lam = np.zeros(10)
    out = _Out(P)

    def call(lam_ptr, gamma=0.1, projection=0, p0=1.0, grad_ptr=out.grad.data_ptr()):
        return lib.dualip_grad_static(P["I"], P["J"], P["m"], P["row_ptr"].data_ptr(), P["item_idx"].data_ptr(), P["c"].data_ptr(),
                                      P["a"].data_ptr(), P["b"].data_ptr(), projection, p0, 0.0, lam_ptr, gamma, grad_ptr, None, None,
                                      None)

    assert call(ctypes.c_void_p(host_lam.ctypes.data)) == -1                       # host lambda
    host_grad = np.zeros(10)
    assert call(lam.data_ptr(), grad_ptr=ctypes.c_void_p(host_grad.ctypes.data)) == -1   # host output
    assert call(None) == -1 and call(lam.data_ptr(), gamma=0.0) == -1 and call(lam.data_ptr(), projection=9) == -1
    assert call(lam.data_ptr(), p0=-1.0) == -1
    assert call(lam.data_ptr()) == 0                                               # and the well-formed call goes through
    torch.cuda.synchronize()
    assert torch.isfinite(out.grad).all()
