"""`-m gpu` parity of the SURVEY 8(f) rows on the CUDA path (through the C ABI) against the fp64 oracle:

  f-2  range-clipped adaptive step (R20) -- per-iteration eta, grad, lambda
  f-4  global-count row (R21) -- one more dual gathered by every nonzero; Table-4 gap column;
       equality rows in the FINAL scalars (R19)
and the boundary findings of the round-1 review: two live handles sharing one kernel instantiation with different
shared-memory plans, and dualip_set_c with a misaligned borrowed pointer.
"""
import numpy as np
import pytest
import torch

import oracle
import synth
from conftest import random_problem

pytestmark = pytest.mark.gpu

if torch.cuda.is_available():
    import paper_2606_07777_b200 as pkg
    from gpu_util import assert_adaptive_step_parity, assert_grad_parity, assert_trajectory_parity, both, from_instance, gpu_grad, gpu_solve, rel_l2
    from test_gpu_parity import _ragged


# ---------------------------------------------------------------- f-2: range-clipped adaptive step (R20)

@pytest.mark.parametrize("jacobi", [False, True])
@pytest.mark.parametrize("kernel", ["streaming", "direct"])
def test_adaptive_step_trajectory(jacobi, kernel):
    """Three continuation stages; the clip range is chosen around gamma_1 / L so that the secant step is sometimes inside
    the range and sometimes clipped; in the later stages gamma_s / L is below eta_min, so the stage opens with gamma_s / L
    itself (lo_s = min(eta_min, gamma_s / L), R20) and the scaled maximum caps the secant steps."""
    rng = np.random.default_rng(17)
    d = _ragged(rng, 3000, 80, 2, [4, 9, 17, 30, 0, 12, 41])
    d["b"] = (d["b"] * 0.25).astype(np.float32)                  # binding: lambda moves
    po = oracle.Problem(d["I"], d["J"], d["m"], d["row_ptr"], d["item_idx"], d["c"], d["a"], d["b"])
    L = 2.0 if jacobi else oracle.lipschitz(po)
    gam, its = [0.4, 0.04, 0.004], [25, 25, 25]
    rng_eta = (0.5 * gam[0] / L, 30.0 * gam[0] / L)       # the secant step runs at 12..55 x gamma / L on this instance
    po, pg = both(d, jacobi=jacobi, adaptive=True, eta_min=rng_eta[0], eta_max=rng_eta[1], direct_kernel=(kernel == "direct"))
    ref, out = assert_adaptive_step_parity(po, pg, gam, its, rng_eta, jacobi=jacobi, tag=f"adaptive/{kernel}/jacobi={jacobi}")
    eta = out["tr_eta"]
    assert (eta[1:25] > rng_eta[0] * 1.001).any() and (eta[1:25] < rng_eta[1] * 0.999).any()      # really adaptive somewhere
    hi3 = rng_eta[1] * gam[2] / gam[0]
    assert abs(eta[-25] / (gam[2] / L) - 1.0) <= 1e-12 and gam[2] / L < rng_eta[0]                   # opens with the analytic step, below eta_min
    assert eta[-24:].max() <= hi3 * (1 + 1e-15) and (eta[-24:] == hi3).any()                       # the scaled maximum caps the secant
    assert (ref.lam > 0).sum() >= 5
    pg.destroy()


def test_adaptive_point_range_is_the_fixed_step_bit_for_bit():
    cfg = synth.get_config("cfg2-tight", I=20_000)
    inst = synth.generate(cfg)
    po, fixed = from_instance(inst)
    eta = 1e-2 / fixed.info().L
    _, ada = from_instance(inst, adaptive=True, eta_min=eta, eta_max=eta)
    a = gpu_solve(fixed, [1e-2], [30])
    b = gpu_solve(ada, [1e-2], [30])
    assert np.array_equal(a["tr_lam"], b["tr_lam"]) and np.array_equal(a["tr_g"], b["tr_g"]) and np.array_equal(a["x"], b["x"])
    assert np.all(b["tr_eta"] == eta) and np.all(a["tr_eta"] == eta)
    fixed.destroy(); ada.destroy()


def test_adaptive_on_a_scaled_config_with_graph_replay():
    """cfg3-tight (Zipf items: the fixed scalar step stalls) with the adaptive Jacobi step, CUDA-graph replay on: the graph's
    launches all carry the same arguments, the step comes from device state."""
    cfg = synth.get_config("cfg3-tight", I=30_000)
    inst = synth.generate(cfg)
    rng_eta = (1e-5, 1e-1)
    po, pg = from_instance(inst, jacobi=True, adaptive=True, eta_min=rng_eta[0], eta_max=rng_eta[1], use_graph=True, group_lanes=8)
    assert_adaptive_step_parity(po, pg, [1e-1, 1e-2], [45, 45], rng_eta, jacobi=True, tag="cfg3-tight/adaptive+graph")
    pg.destroy()


# ---------------------------------------------------------------- f-4: global-count row (R21), gap, R19 final scalars

@pytest.mark.parametrize("kind,p0,p1", [("simplex", 1.0, 0.0), ("simplex_eq", 1.0, 0.0), ("boxcut", 0.3, 1.0), ("box", 0.0, 0.4)])
@pytest.mark.parametrize("kernel", ["streaming", "direct"])
def test_count_row_gradient(kind, p0, p1, kernel):
    if kernel == "direct" and kind == "box":
        pytest.skip("the box projection has a single element-wise kernel")
    rng = np.random.default_rng(23)
    d = _ragged(rng, 2500, 90, 2, [3, 8, 16, 33, 0, 70, 140])
    M = 900.0
    po, pg = both(d, kind, p0, p1, count_M=M, direct_kernel=(kernel == "direct"))
    assert pg.info().duals == 181 and pg.duals == 181
    for gamma in (1.0, 1e-1, 1e-2, 1e-3):
        for mu in (0.0, 0.07, 0.6, 3.0):                         # 3.0: larger than every |c|: every row of the inequality kinds is dead
            lam = np.concatenate([rng.random(180) * 0.3, [mu]])
            assert_grad_parity(po, pg, lam, gamma, tag=f"count/{kind}/{kernel}/g={gamma}/mu={mu}")
    lam = np.concatenate([rng.normal(size=180) * 0.2, [-0.4]])   # g is defined for a negative mu too
    ex, eg = assert_grad_parity(po, pg, lam, 0.05, tag=f"count/{kind}/neg")
    sc, grad, x = gpu_grad(pg, lam, 0.05)
    assert abs(grad[-1] - (x.astype(np.float64).sum() - M)) <= 1e-5 * M
    # a budget that is not an fp32 number (2^24 + 1; config 3-5 sized budgets are tens of millions): the row's right-hand side
    # is fp64 on both sides, so its gradient entry sum x - M matches to the accuracy of sum x, not to an ulp of fp32(M) = 2
    Mbig = float(2 ** 24 + 1)
    pg.set_global_count(Mbig)
    pob = oracle.Problem(po.I, po.J, po.m, po.row_ptr, po.item_idx, po.c, po.a, po.b, po.proj_kind, po.p0, po.p1, Mbig)
    ref = oracle.grad(pob, lam, 0.05)
    sc, grad, x = gpu_grad(pg, lam, 0.05)
    assert abs(grad[-1] - ref.grad[-1]) <= 1e-3 and abs(ref.grad[-1] - (ref.x.sum() - Mbig)) <= 1e-6
    assert_grad_parity(pob, pg, lam, 0.05, tag=f"count/{kind}/M=2^24+1")
    # switching the row off restores the plain problem
    pg.set_global_count(None)
    po0 = oracle.Problem(po.I, po.J, po.m, po.row_ptr, po.item_idx, po.c, po.a, po.b, po.proj_kind, po.p0, po.p1)
    assert_grad_parity(po0, pg, lam[:-1], 0.05, tag="count/off")
    pg.destroy()


@pytest.mark.parametrize("jacobi", [False, True])
def test_count_row_trajectory(jacobi):
    """The count row binds (M below the unconstrained sum of x): its dual moves, per-iteration parity of the whole dual
    vector; every third row an equality on top (mask of J*m + 1 entries)."""
    rng = np.random.default_rng(29)
    d = _ragged(rng, 3000, 60, 1, [4, 9, 17, 30, 0, 12])
    d["b"] = (d["b"] * 4.0).astype(np.float32)
    M = 700.0
    po, pg = both(d, count_M=M, jacobi=jacobi)
    info = pg.info()
    assert info.L_step == (2.0 if jacobi else info.L + po.nnz)
    gam, its = [0.3, 0.03], [60, 60]
    worst, ex, ref, out = assert_trajectory_parity(po, pg, gam, its, tag=f"count/jacobi={jacobi}", jacobi=jacobi)
    if jacobi:                                                    # the unscaled step is L + nnz: the dual barely moves in 120 its
        assert ref.lam[-1] > 0 and ref.final.x.sum() < 0.9 * oracle.grad(po, np.zeros(61), 0.03).x.sum()
    mask = (np.arange(61) % 3 == 0).astype(np.uint8)
    pg.set_equality_rows(mask)
    assert_trajectory_parity(po, pg, gam, its, tag=f"count+eq/jacobi={jacobi}", jacobi=jacobi, is_eq=mask)
    pg.destroy()


def test_count_row_on_one_item_is_a_second_family_on_the_gpu():
    """The oracle's pin of R21 (J = 1: the count row IS a second coupling family with a = 1), repeated on the CUDA path:
    two different code paths of the kernel (uniform shift mu vs the m = 2 gather) must give the same x and gradients."""
    rng = np.random.default_rng(5)
    I = 5000
    d = dict(I=I, J=1, m=1, row_ptr=np.arange(I + 1, dtype=np.int64), item_idx=np.zeros(I, dtype=np.int32),
             c=(-rng.random(I)).astype(np.float32), a=(0.5 + rng.random(I)).astype(np.float32), b=np.array([400.0], dtype=np.float32))
    M = np.float32(900.0)
    d2 = dict(d, m=2, a=np.stack([d["a"], np.ones(I, dtype=np.float32)], axis=1).reshape(-1), b=np.array([400.0, M], dtype=np.float32))
    _, pc = both(d, count_M=float(M))
    _, p2 = both(d2)
    for lam in ([0.0, 0.0], [0.2, 0.1], [0.05, 0.4]):
        sc_c, g_c, x_c = gpu_grad(pc, lam, 0.3)
        sc_2, g_2, x_2 = gpu_grad(p2, lam, 0.3)
        assert np.abs(x_c - x_2).max() <= 1e-6 and rel_l2(g_c, g_2) <= 1e-6 and abs(sc_c.g - sc_2.g) <= 1e-6 * abs(sc_2.g)
    pc.destroy(); p2.destroy()


def test_gap_vanishes_at_the_optimum_and_final_scalars_respect_equality_rows():
    """Table 4's columns from dualip_scalars: primal = obj + reg, dual = g, gap = primal - dual -> 0 and slack = r_inf -> 0
    as the solve converges; with equality rows the FINAL r_inf / r_2 count |grad| on them (R19), as the oracle's do."""
    rng = np.random.default_rng(31)
    d = random_problem(rng, I=400, J=12, m=1, deg=(2, 6), tight=0.6)
    d["b"][::2] *= 5.0                                             # every other row is slack at the optimum
    po, pg = both(d, jacobi=True)
    ref = oracle.solve(po, [0.5], [3000], jacobi=True)
    out = gpu_solve(pg, [0.5], [3000], want_trace=False)
    sc = out["sc"]
    assert abs(sc.gap - (sc.obj + sc.reg - sc.g)) <= 1e-9 * (abs(sc.obj) + abs(sc.g))
    assert abs(ref.final.gap) < 1e-6 and abs(sc.gap) < 1e-5 * abs(sc.g) and sc.r_inf < 1e-5
    mask = np.zeros(12, dtype=np.uint8); mask[::2] = 1
    pg.set_equality_rows(mask)
    ref = oracle.solve(po, [0.5], [40], jacobi=True, is_eq=mask)
    out = gpu_solve(pg, [0.5], [40], want_trace=False)
    gn = np.linalg.norm(ref.final.grad)
    neg = (ref.final.grad < 0) & (mask == 1)
    assert neg.any() and ref.final.r_inf >= np.abs(ref.final.grad[neg]).max() - 1e-12    # a negative equality residual counts
    assert abs(out["sc"].r_inf - ref.final.r_inf) <= 1e-5 * gn and abs(out["sc"].r_2 - ref.final.r_2) <= 1e-5 * gn
    pg.destroy()


# ---------------------------------------------------------------- boundary

def test_two_live_handles_share_an_instantiation_with_different_plans():
    """The dynamic shared-memory attribute is per FUNCTION and process-wide: a second handle on the same kernel
    instantiation with a smaller plan must not break the launches of the first (alternating launches)."""
    rng = np.random.default_rng(37)
    big = _ragged(rng, 4000, 6000, 1, [30, 90, 200, 380])         # J = 6000, long rows: large stages
    small = _ragged(rng, 4000, 50, 1, [3, 9, 20])                 # same (G, M, reduction) instantiation, small plan
    po_b, pg_b = both(big, group_lanes=8, reduction=pkg.RED_GLOBAL)
    po_s, pg_s = both(small, group_lanes=8, reduction=pkg.RED_GLOBAL)
    ib, is_ = pg_b.info(), pg_s.info()
    assert ib.streaming == 1 and is_.streaming == 1 and ib.smem_bytes != is_.smem_bytes
    for rep in range(3):
        assert_grad_parity(po_b, pg_b, rng.random(6000) * 0.2, 1e-2, tag=f"big/{rep}")
        assert_grad_parity(po_s, pg_s, rng.random(50) * 0.2, 1e-2, tag=f"small/{rep}")
    pg_b.destroy(); pg_s.destroy()


def test_set_c_rejects_a_misaligned_borrowed_pointer():
    inst = synth.generate(synth.get_config("cfg2", I=20_000), device="cuda")
    kind, p0, p1 = synth.proj_spec(inst.cfg)
    pg = pkg.Problem.create(inst.I, inst.J, inst.m, inst.row_ptr, inst.item_idx, inst.c, inst.a, inst.b,
                            pkg.binding.make_opts(borrow=True))
    assert pg.info().streaming == 1
    lam = torch.zeros(inst.J, dtype=torch.float64, device="cuda")
    sc0 = pkg.Scalars(); pg.grad(lam, 1e-3, scalars=sc0)
    buf = torch.empty(inst.nnz + 1, dtype=torch.float32, device="cuda")
    buf[1:] = inst.c * 0.5
    with pytest.raises(pkg.DualipError) as e:
        pg.set_c(buf[1:])                                          # 4 bytes off a 16-byte boundary
    assert e.value.code == -1
    sc1 = pkg.Scalars(); pg.grad(lam, 1e-3, scalars=sc1)
    torch.cuda.synchronize()
    assert sc1.g == sc0.g                                          # the handle kept the old c
    c2 = (inst.c * 0.5).contiguous()
    pg.set_c(c2)
    sc2 = pkg.Scalars(); pg.grad(lam, 1e-3, scalars=sc2)
    torch.cuda.synchronize()
    assert abs(sc2.obj - 0.5 * sc0.obj) <= 1e-4 * abs(sc0.obj)      # x changes only where |c| / gamma < 1
    pg.destroy()


def test_per_launch_lambda_plan_decides_from_lambda_and_gamma_and_changes_no_bit():
    """J*m = 10,000 duals: too many for lambda's low word to be sized into the plan, so each LAUNCH decides (k_grad_tma prologue):
    at lambda = 0 the fp32 dual is exact enough and every stage is kept; at a busy lambda and small gamma the low word is staged
    and a stage given up.  Forcing either choice (tuning.lambda_plan) gives the same bits: both exact paths use the two-word dual."""
    cfg = synth.get_config("cfg3-tight", I=30_000)
    inst = synth.generate(cfg)
    po, auto = from_instance(inst, group_lanes=8)
    _, never = from_instance(inst, group_lanes=8, lambda_plan=1)
    _, always = from_instance(inst, group_lanes=8, lambda_plan=2)
    lam0, lam1 = np.zeros(inst.J), synth.probe_lambda(inst, 0, 0.05).numpy()
    sc, g0, x0 = gpu_grad(auto, lam0, 1e-3)
    assert auto.info().lambda_lo_smem == 0
    sc, g1, x1 = gpu_grad(auto, lam1, 1e-3)
    assert auto.info().lambda_lo_smem == 1
    sc, g2, x2 = gpu_grad(auto, lam1, 10.0)                      # the same lambda at a gamma where its fp32 rounding cannot matter
    assert auto.info().lambda_lo_smem == 0
    for other, want in ((never, 0), (always, 1)):
        sc, g, x = gpu_grad(other, lam1, 1e-3)
        assert other.info().lambda_lo_smem == want
        assert np.array_equal(g, g1) and np.array_equal(x, x1)
    assert_grad_parity(po, auto, lam1, 1e-3, tag="lambda plan")
    for P in (auto, never, always):
        P.destroy()


def test_table4_columns():
    sc = pkg.Scalars(g=-10.0, obj=-9.0, reg=0.5, r_inf=1e-3, r_2=2e-3, gap=1.5)
    assert sc.table4() == {"primal_obj": -9.0, "primal_reg": 0.5, "dual": -10.0, "gap": 1.5, "slack": 1e-3}       # selection only, no arithmetic
