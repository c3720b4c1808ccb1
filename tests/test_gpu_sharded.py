"""`-m gpu` test of the user-sharded path on ONE GPU: the instance is cut into two contiguous user
ranges, each behind its own handle; the "all-reduce" is the integer sum of the two handles' fixed-point accumulators, done in
the reduce hook of shard 0.  With the create-time constants agreed through integer sums as well, the sharded evaluation must be
BIT-identical to the unsharded one: grad g, every scalar, x, and the whole AGD trajectory.  The hooked shard-0 handle is also
compared with the ORACLE directly (grad g, scalars, both shards' x, and every iteration of the trajectory), so the row stands on
the oracle and not only on the unsharded handle's own parity tests.  (Two ranks on two GPUs run the same
calls with torch.distributed's all_reduce in the hook: paper_2606_07777_b200/sharded.py; unmeasured on multi-GPU hardware.)"""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu

if torch.cuda.is_available():
    import paper_2606_07777_b200 as pkg
    from paper_2606_07777_b200.binding import ShardExtents
    from paper_2606_07777_b200.sharded import split_users
    import oracle
    from gpu_util import _KIND, TOL_G, TOL_GRAD, TOL_X, gpu_solve, rel_l2


def _shard(inst, u0, u1, **opt):
    p0, p1 = int(inst.row_ptr[u0]), int(inst.row_ptr[u1])
    rp = (inst.row_ptr[u0:u1 + 1] - inst.row_ptr[u0]).contiguous()
    kind, q0, q1 = synth.proj_spec(inst.cfg)
    proj = {"simplex": pkg.PROJ_SIMPLEX_INEQ, "boxcut": pkg.PROJ_BOXCUT, "box": pkg.PROJ_BOX}[kind]
    return pkg.Problem.create(u1 - u0, inst.J, inst.m, rp, inst.item_idx[p0:p1].contiguous(), inst.c[p0:p1].contiguous(),
                              inst.a[p0 * inst.m:p1 * inst.m].contiguous(), inst.b, pkg.binding.make_opts(projection=proj, p0=q0, p1=q1, **opt))


@pytest.mark.parametrize("name,I,jacobi", [("cfg2-tight", 60_000, False), ("cfg3-tight", 30_000, True), ("cfg4-tight", 8_000, True)])
def test_two_shards_on_one_gpu_are_bit_identical_to_the_unsharded_problem(name, I, jacobi):
    inst = synth.generate(synth.get_config(name, I=I), device="cuda")
    Jm = inst.J * inst.m
    whole = _shard(inst, 0, inst.I, jacobi=jacobi)
    cuts = split_users(inst.row_ptr, 2)
    assert cuts[0] == 0 and cuts[2] == inst.I and 0 < cuts[1] < inst.I
    nz = [int(inst.row_ptr[c]) for c in cuts]
    assert abs((nz[1] - nz[0]) - (nz[2] - nz[1])) <= 40 * 400                     # balanced by nonzeros
    assert cuts[1] % 2 == 0 and nz[1] % 4 == 0                                       # 16-byte aligned slices: same lane assignment
    # the same kernel instantiation on every shard (a production run configures all ranks alike): a row's arithmetic depends on
    # the lanes per row, not on which tile, step or CTA it lands in
    G = whole.info().group_lanes
    A, B = _shard(inst, cuts[0], cuts[1], jacobi=jacobi, group_lanes=G), _shard(inst, cuts[1], cuts[2], jacobi=jacobi, group_lanes=G)
    # a0 across shards: extents (SUM, MAX), then the fixed-point column sums (int64 SUM) -- what sharded.py all-reduces
    ea, eb = A.shard_extents(), B.shard_extents()
    g = ShardExtents(ea.I + eb.I, ea.nnz + eb.nnz, max(ea.max_abs_a, eb.max_abs_a), max(ea.max_abs_c, eb.max_abs_c))
    sa = A.column_stats(g, torch.empty(2 * Jm + 1, dtype=torch.int64, device="cuda"))
    sb = B.column_stats(g, torch.empty(2 * Jm + 1, dtype=torch.int64, device="cuda"))
    for P in (A, B):
        P.set_shard_constants(g, sa + sb)
    wi, ai = whole.info(), A.info()
    assert (ai.L, ai.L_step, ai.fix_scale_s) == (wi.L, wi.L_step, wi.fix_scale_s)   # derived from the same integers

    tmp = torch.empty(A.acc_words, dtype=torch.int64, device="cuda")
    calls = []

    def hook(acc_ptr, n_words, lam_ptr, gamma, stream):                              # shard 0's hook: + shard 1's accumulators
        assert n_words == A.acc_words
        B.eval_partial(lam_ptr, gamma)
        B.export_accumulators(tmp, clear=True)
        A.import_accumulators(tmp, accumulate=True)
        calls.append(gamma)

    A.set_reduce_hook(hook)
    d = inst.numpy()
    kind, q0, q1 = synth.proj_spec(inst.cfg)
    po = oracle.Problem(inst.I, inst.J, inst.m, d["row_ptr"], d["item_idx"], d["c"], d["a"], d["b"], _KIND[kind][0], q0, q1)
    for lam, gamma in ((torch.zeros(Jm, dtype=torch.float64, device="cuda"), inst.cfg.gammas[-1]),
                       (synth.probe_lambda(inst, 0, 0.05 if "3" in name else 0.5), inst.cfg.gammas[-1]),
                       (synth.probe_lambda(inst, 1, 0.05 if "3" in name else 0.5), 0.1)):
        gw, ga = torch.empty(Jm, dtype=torch.float64, device="cuda"), torch.empty(Jm, dtype=torch.float64, device="cuda")
        xw = torch.empty(inst.nnz, dtype=torch.float32, device="cuda")
        xa, xb = torch.empty(nz[1], dtype=torch.float32, device="cuda"), torch.empty(nz[2] - nz[1], dtype=torch.float32, device="cuda")
        sw, ss = pkg.Scalars(), pkg.Scalars()
        whole.grad(lam, gamma, grad=gw, scalars=sw, x=xw)
        A.grad(lam, gamma, grad=ga, scalars=ss, x=xa)
        B.eval_partial(lam, gamma, x=xb); B.export_accumulators(tmp, clear=True)
        torch.cuda.synchronize()
        assert torch.equal(gw, ga), "sharded grad g differs from the unsharded one"
        assert sw.as_dict() == ss.as_dict(), (sw.as_dict(), ss.as_dict())
        assert torch.equal(xw[:nz[1]], xa) and torch.equal(xw[nz[1]:], xb)
        # ... and the sharded evaluation against the oracle itself
        ref = oracle.grad(po, lam.cpu().numpy(), gamma)
        assert rel_l2(ga.cpu().numpy(), ref.grad) <= TOL_GRAD
        assert abs(ss.g - ref.g) <= TOL_G * abs(ref.g) + 1e-12 and abs(ss.obj - ref.obj) <= TOL_G * abs(ref.obj) + 1e-9
        assert abs(ss.reg - ref.reg) <= TOL_G * abs(ref.reg) + 1e-9 and abs(ss.r_inf - ref.r_inf) <= TOL_GRAD * np.linalg.norm(ref.grad) + 1e-12
        assert np.abs(torch.cat([xa, xb]).cpu().numpy().astype(np.float64) - ref.x).max() <= TOL_X
    n0 = len(calls)
    gam, its = [10 * inst.cfg.gammas[-1], inst.cfg.gammas[-1]], [20, 20]
    ow = gpu_solve(whole, gam, its, want_x=False)
    oa = gpu_solve(A, gam, its, want_x=False)
    assert len(calls) - n0 == sum(its) + 1                                           # one exchange per evaluation
    assert np.array_equal(ow["tr_lam"], oa["tr_lam"]) and np.array_equal(ow["tr_grad"], oa["tr_grad"]) and np.array_equal(ow["tr_g"], oa["tr_g"])
    assert np.array_equal(ow["lam"], oa["lam"]) and (ow["lam"] > 0).sum() > 5
    # the sharded trajectory against the oracle's own solve, iteration by iteration
    rs = oracle.solve(po, gam, its, trace_grad=True, trace_lambda=True, jacobi=jacobi)
    for n in range(sum(its)):
        assert rel_l2(oa["tr_grad"][n], rs.trace_grad[n]) <= TOL_GRAD, f"sharded iteration {n}"
    assert np.abs(oa["tr_g"] - rs.trace_g).max() <= TOL_G * np.abs(rs.trace_g).max() + 1e-12
    assert np.abs(oa["tr_lam"] - rs.trace_lambda).max() <= 1e-6 * max(np.abs(rs.trace_lambda).max(), 1e-300) + 1e-12
    assert rel_l2(oa["grad"], rs.final.grad) <= TOL_GRAD and abs(oa["sc"].g - rs.final.g) <= TOL_G * abs(rs.final.g) + 1e-12
    A.set_reduce_hook(None)
    for P in (A, B):
        P.destroy()
    # an UNALIGNED cut: rows of the second shard sit at other positions modulo 4, so their candidates land in other lanes and the
    # fp32 sums inside a fractional row's projection run in another order -- equal to the unsharded result to rounding, not bits
    cut = cuts[1] + 1
    while int(inst.row_ptr[cut]) % 4 == 0:
        cut += 1
    A, B = _shard(inst, 0, cut, jacobi=jacobi, group_lanes=G), _shard(inst, cut, inst.I, jacobi=jacobi, group_lanes=G)
    for P in (A, B):
        P.set_shard_constants(g, sa + sb)
    A.set_reduce_hook(hook)
    lam, gamma = synth.probe_lambda(inst, 1, 0.05 if "3" in name else 0.5), 0.1
    gw, ga = torch.empty(Jm, dtype=torch.float64, device="cuda"), torch.empty(Jm, dtype=torch.float64, device="cuda")
    whole.grad(lam, gamma, grad=gw); A.grad(lam, gamma, grad=ga)
    torch.cuda.synchronize()
    assert float((gw - ga).norm() / gw.norm()) <= 1e-6
    A.set_reduce_hook(None)
    for P in (whole, A, B):
        P.destroy()


def test_set_c_on_shards_keeps_one_scale_and_demands_a_new_agreement():
    """dualip_set_c on a sharded handle (config 5's perturbed re-solve): a shard must not derive the objective's
    fixed-point scale from its OWN sum |c| -- ranks would then all-reduce integers of different scales.  The handle keeps the
    agreed constants, refuses to evaluate (DUALIP_ESTALE) until the shards have agreed again, and after that is bit-identical to
    the unsharded handle given the same new c.  The two shards' c are made very unequal in size so that per-shard scales WOULD
    differ."""
    inst = synth.generate(synth.get_config("cfg5-tight", I=40_000), device="cuda")
    Jm = inst.J * inst.m
    whole = _shard(inst, 0, inst.I)
    cuts = split_users(inst.row_ptr, 2)
    nz = [int(inst.row_ptr[c]) for c in cuts]
    G = whole.info().group_lanes
    A, B = _shard(inst, cuts[0], cuts[1], group_lanes=G), _shard(inst, cuts[1], cuts[2], group_lanes=G)
    tmp = torch.empty(A.acc_words, dtype=torch.int64, device="cuda")

    def agree():
        ea, eb = A.shard_extents(), B.shard_extents()
        g = ShardExtents(ea.I + eb.I, ea.nnz + eb.nnz, max(ea.max_abs_a, eb.max_abs_a), max(ea.max_abs_c, eb.max_abs_c))
        sa = A.column_stats(g, torch.empty(2 * Jm + 1, dtype=torch.int64, device="cuda"))
        sb = B.column_stats(g, torch.empty(2 * Jm + 1, dtype=torch.int64, device="cuda"))
        for P in (A, B):
            P.set_shard_constants(g, sa + sb)

    def hook(acc_ptr, n_words, lam_ptr, gamma, stream):
        B.eval_partial(lam_ptr, gamma)
        B.export_accumulators(tmp, clear=True)
        A.import_accumulators(tmp, accumulate=True)

    def same_as_whole(tag):
        lam, gamma = synth.probe_lambda(inst, 0, 0.5), inst.cfg.gammas[-1]
        gw, ga = torch.empty(Jm, dtype=torch.float64, device="cuda"), torch.empty(Jm, dtype=torch.float64, device="cuda")
        sw, ss = pkg.Scalars(), pkg.Scalars()
        whole.grad(lam, gamma, grad=gw, scalars=sw)
        A.grad(lam, gamma, grad=ga, scalars=ss)
        torch.cuda.synchronize()
        assert torch.equal(gw, ga), tag
        assert sw.as_dict() == ss.as_dict(), (tag, sw.as_dict(), ss.as_dict())
        return sw

    agree()
    A.set_reduce_hook(hook)
    s0 = same_as_whole("before set_c")
    c2 = synth.perturb_c(inst, 0.01)
    c2[nz[1]:] *= 37.0                                                               # shard 1's |c| dwarfs shard 0's
    whole.set_c(c2)
    A.set_c(c2[:nz[1]].contiguous()); B.set_c(c2[nz[1]:].contiguous())
    lam = torch.zeros(Jm, dtype=torch.float64, device="cuda")
    for call in (lambda: A.grad(lam, 0.1, grad=torch.empty(Jm, dtype=torch.float64, device="cuda")),
                 lambda: A.solve([0.1], [2], lam.clone()),
                 lambda: B.eval_partial(lam, 0.1)):
        with pytest.raises(pkg.DualipError) as e:
            call()
        assert e.value.code == pkg.ESTALE
    agree()
    s1 = same_as_whole("after set_c + new agreement")
    assert s1.obj != s0.obj
    assert A.info().L == whole.info().L
    A.set_reduce_hook(None)
    for P in (whole, A, B):
        P.destroy()


def test_a_failing_hook_abandons_the_evaluation_and_leaves_nothing_behind():
    """The reduce hook returns non-zero, or raises (a failed all-reduce): the evaluation must not be finalised from this shard's
    sums alone -- dualip_grad / dualip_solve return DUALIP_EHOOK, the Python exception is chained to the DualipError, the outputs
    stay untouched, and the partial sums are dropped so that the next evaluation, with a working hook, is exact again.  The
    hook's `stream` argument is the stream of the call (here a side stream), and work it enqueues there is ordered with the kernels."""
    inst = synth.generate(synth.get_config("cfg2-tight", I=30_000), device="cuda")
    Jm = inst.J * inst.m
    whole = _shard(inst, 0, inst.I)
    lam, gamma = synth.probe_lambda(inst, 0, 0.5), inst.cfg.gammas[-1]
    want = torch.empty(Jm, dtype=torch.float64, device="cuda")
    whole.grad(lam, gamma, grad=want)
    A = _shard(inst, 0, inst.I, group_lanes=whole.info().group_lanes)
    seen = []

    def bad_return(acc_ptr, n_words, lam_ptr, gamma, stream):
        seen.append(stream)
        return 3

    def raises(acc_ptr, n_words, lam_ptr, gamma, stream):
        raise RuntimeError("all-reduce timed out")

    def fine(acc_ptr, n_words, lam_ptr, gamma, stream):
        seen.append(stream)

    side = torch.cuda.Stream()
    got = torch.full((Jm,), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()                                                        # inputs were made on the default stream
    A.set_reduce_hook(bad_return)
    with pytest.raises(pkg.DualipError) as e:
        A.grad(lam, gamma, grad=got, stream=side)
    assert e.value.code == pkg.EHOOK and e.value.__cause__ is None and seen == [side.cuda_stream]
    A.set_reduce_hook(raises)
    with pytest.raises(pkg.DualipError) as e:
        A.grad(lam, gamma, grad=got)
    assert e.value.code == pkg.EHOOK and isinstance(e.value.__cause__, RuntimeError)
    with pytest.raises(pkg.DualipError) as e:
        A.solve([gamma], [3], lam.clone())
    assert e.value.code == pkg.EHOOK and isinstance(e.value.__cause__, RuntimeError)
    torch.cuda.synchronize()
    assert torch.isnan(got).all()                                                   # no epilogue ran
    A.set_reduce_hook(fine)
    A.grad(lam, gamma, grad=got, stream=side)
    side.synchronize()
    assert torch.equal(got, want), "partial sums of the abandoned evaluations leaked into this one"
    A.set_reduce_hook(None)
    for P in (whole, A):
        P.destroy()
