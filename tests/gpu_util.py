"""Helpers shared by the `-m gpu` parity tests: build the oracle problem and the CUDA problem from the
SAME arrays and compare at the tolerances BASELINE.json's north_star states."""
import numpy as np
import torch

import oracle
import paper_2606_07777_b200 as pkg
import synth
from conftest import ADAPTIVE_DRIFT

TOL_X = 1e-5        # x: element-wise absolute
TOL_GRAD = 1e-5     # grad g: relative L2, per evaluation / per iteration
TOL_G = 1e-5        # dual objective: relative

_KIND = {"simplex": (oracle.PROJ_SIMPLEX_INEQ, pkg.PROJ_SIMPLEX_INEQ), "box": (oracle.PROJ_BOX, pkg.PROJ_BOX),
         "boxcut": (oracle.PROJ_BOXCUT, pkg.PROJ_BOXCUT), "simplex_eq": (oracle.PROJ_SIMPLEX_EQ, pkg.PROJ_SIMPLEX_EQ)}


def both(d, kind="simplex", p0=1.0, p1=0.0, count_M=None, **opt):
    """d: dict of numpy arrays (I,J,m,row_ptr,item_idx,c,a,b) -> (oracle.Problem, pkg.Problem).  count_M: right-hand side of
    the global-count row sum x <= M (R21) on both sides, or None."""
    ko, kg = _KIND[kind]
    po = oracle.Problem(d["I"], d["J"], d["m"], d["row_ptr"], d["item_idx"], d["c"], d["a"], d["b"], ko, p0, p1, count_M)
    t = {k: torch.from_numpy(np.ascontiguousarray(getattr(po, k))).cuda() for k in ("row_ptr", "item_idx", "c", "a", "b")}
    pg = pkg.Problem.create(po.I, po.J, po.m, t["row_ptr"], t["item_idx"], t["c"], t["a"], t["b"],
                            pkg.binding.make_opts(projection=kg, p0=p0, p1=p1, **opt))
    if count_M is not None:
        pg.set_global_count(count_M)
    return po, pg


def from_instance(inst: synth.Instance, **opt):
    d = inst.numpy()
    d.update(I=inst.I, J=inst.J, m=inst.m)
    kind, p0, p1 = synth.proj_spec(inst.cfg)
    return both(d, kind, p0, p1, **opt)


def gpu_grad(pg, lam, gamma, want_x=True):
    lam_t = torch.as_tensor(np.asarray(lam, dtype=np.float64)).cuda()
    grad = torch.empty(pg.duals, dtype=torch.float64, device="cuda")
    x = torch.empty(pg.nnz, dtype=torch.float32, device="cuda") if want_x else None
    sc = pkg.Scalars()
    pg.grad(lam_t, gamma, grad=grad, scalars=sc, x=x)
    torch.cuda.synchronize()
    return sc, grad.cpu().numpy(), (x.cpu().numpy() if want_x else None)


def rel_l2(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (nb if nb > 0 else 1.0)


def assert_grad_parity(po, pg, lam, gamma, tag="", is_eq=None):
    ref = oracle.grad(po, lam, gamma, is_eq=is_eq)
    sc, grad, x = gpu_grad(pg, lam, gamma)
    ex = np.abs(x.astype(np.float64) - ref.x).max() if ref.x.size else 0.0
    eg = rel_l2(grad, ref.grad)
    assert ex <= TOL_X, f"{tag} x abs err {ex:.3e}"
    assert eg <= TOL_GRAD, f"{tag} grad rel L2 {eg:.3e}"
    scale = max(abs(ref.g), 1e-300)
    assert abs(sc.g - ref.g) <= TOL_G * scale + 1e-12, f"{tag} g {sc.g} vs {ref.g}"
    assert abs(sc.obj - ref.obj) <= TOL_G * max(abs(ref.obj), 1e-12) + 1e-9, f"{tag} obj {sc.obj} vs {ref.obj}"
    assert abs(sc.reg - ref.reg) <= TOL_G * max(abs(ref.reg), 1e-12) + 1e-9, f"{tag} reg {sc.reg} vs {ref.reg}"
    assert abs(sc.r_inf - ref.r_inf) <= TOL_GRAD * np.linalg.norm(ref.grad) + 1e-12, f"{tag} r_inf"
    assert abs(sc.r_2 - ref.r_2) <= TOL_GRAD * np.linalg.norm(ref.grad) + 1e-12, f"{tag} r_2"
    # gap = (obj + reg) - g = -lambda'grad (Table 4): absolute against the size of the terms it is the difference of
    assert abs(sc.gap - ref.gap) <= TOL_G * (abs(ref.obj) + abs(ref.reg) + abs(ref.g)) + 1e-9, f"{tag} gap {sc.gap} vs {ref.gap}"
    return ex, eg


def gpu_solve(pg, gammas, iters, lam0=None, want_trace=True, want_x=True):
    Jm, T = pg.duals, int(np.sum(iters))
    lam = torch.zeros(Jm, dtype=torch.float64, device="cuda") if lam0 is None else torch.as_tensor(lam0).double().cuda().clone()
    x = torch.empty(pg.nnz, dtype=torch.float32, device="cuda") if want_x else None
    grad = torch.empty(Jm, dtype=torch.float64, device="cuda")
    tr = None
    if want_trace:
        tr = {"g": torch.empty(T, dtype=torch.float64, device="cuda"), "r_inf": torch.empty(T, dtype=torch.float64, device="cuda"),
              "r_2": torch.empty(T, dtype=torch.float64, device="cuda"), "grad": torch.empty(T * Jm, dtype=torch.float64, device="cuda"),
              "lambda": torch.empty(T * Jm, dtype=torch.float64, device="cuda"), "eta": torch.empty(T, dtype=torch.float64, device="cuda")}
    sc = pkg.Scalars()
    pg.solve(gammas, iters, lam, x=x, scalars=sc, grad=grad, trace=tr)
    torch.cuda.synchronize()
    out = {"lam": lam.cpu().numpy(), "x": x.cpu().numpy() if want_x else None, "grad": grad.cpu().numpy(), "sc": sc}
    if tr:
        out.update(tr_g=tr["g"].cpu().numpy(), tr_grad=tr["grad"].cpu().numpy().reshape(T, Jm),
                   tr_lam=tr["lambda"].cpu().numpy().reshape(T, Jm), tr_rinf=tr["r_inf"].cpu().numpy(), tr_r2=tr["r_2"].cpu().numpy(),
                   tr_eta=tr["eta"].cpu().numpy())
    return out


def assert_trajectory_parity(po, pg, gammas, iters, lam0=None, momentum=True, tag="", jacobi=False, is_eq=None, ref=None):
    """Independent solves compared per iteration (parity mode B of SURVEY 8(c)).  jacobi: the oracle iterates on the
    literally row-scaled system; pg must have been created with jacobi=True (per-coordinate step).
    is_eq: equality-row mask (pg.set_equality_rows must have been called with it).  ref: the oracle's solve of exactly this
    call when the caller already has it (a concurrent.futures future or the result; full-size tests run it on a host thread)."""
    if ref is None:
        ref = oracle.solve(po, gammas, iters, lam0=lam0, momentum=momentum, trace_grad=True, trace_lambda=True, jacobi=jacobi,
                           is_eq=is_eq)
    elif hasattr(ref, "result"):
        ref = ref.result()
    out = gpu_solve(pg, gammas, iters, lam0=lam0)
    T = int(np.sum(iters))
    worst = 0.0
    for n in range(T):
        e = rel_l2(out["tr_grad"][n], ref.trace_grad[n])
        worst = max(worst, e)
        assert e <= TOL_GRAD, f"{tag} iteration {n}: grad rel L2 {e:.3e}"
    assert np.abs(out["tr_g"] - ref.trace_g).max() <= TOL_G * np.abs(ref.trace_g).max() + 1e-12, f"{tag} trace g"
    ex = np.abs(out["x"].astype(np.float64) - ref.x).max()
    assert ex <= TOL_X, f"{tag} final x abs err {ex:.3e}"
    assert abs(out["sc"].g - ref.final.g) <= TOL_G * abs(ref.final.g) + 1e-12, f"{tag} final g"
    assert rel_l2(out["grad"], ref.final.grad) <= TOL_GRAD, f"{tag} final grad"
    gn = np.linalg.norm(ref.final.grad)
    assert abs(out["sc"].r_inf - ref.final.r_inf) <= TOL_GRAD * gn + 1e-12, f"{tag} final r_inf"
    assert abs(out["sc"].r_2 - ref.final.r_2) <= TOL_GRAD * gn + 1e-12, f"{tag} final r_2"
    assert abs(out["sc"].gap - ref.final.gap) <= TOL_G * (abs(ref.final.obj) + abs(ref.final.reg) + abs(ref.final.g)) + 1e-9, f"{tag} final gap"
    lam_scale = max(np.abs(ref.lam).max(), 1e-300)
    assert np.abs(out["lam"] - ref.lam).max() <= 1e-6 * lam_scale + 1e-12, f"{tag} lambda_T"
    el = np.abs(out["tr_lam"] - ref.trace_lambda).max()
    assert el <= 1e-6 * max(np.abs(ref.trace_lambda).max(), 1e-300) + 1e-12, f"{tag} lambda trace {el:.3e}"
    return worst, ex, ref, out


def assert_adaptive_step_parity(po, pg, gammas, iters, eta_range, jacobi=False, momentum=True, tag=""):
    """The range-clipped secant step (R20) divides by |grad_t - grad_{t-1}|, a DIFFERENCE of gradients: a relative error eps in
    the gradients moves eta_t by eps |grad| / |grad_t - grad_{t-1}|, so two correct implementations drift apart along the
    trajectory faster than with a fixed step, and per-iteration trajectory parity at 1e-5 is not a property the rule has.
    What is checked instead, on the CUDA path's OWN trajectory (y_t rebuilt from the traced lambda_{t+1}):
      (A) same-lambda parity of every iteration: the oracle's grad g(y_t) against the traced gradient (1e-5);
      (B) the rule: eta_t recomputed in fp64 from the traced (y, grad) pairs by R20's definition (norms in the iterated system:
          y / d and d grad under Jacobi scaling, d from the oracle), and lambda_{t+1} = max(0, y_t + eta_t d^2 grad_t), to 1e-9;
      (C) the two INDEPENDENT trajectories (this one and the oracle's own solve) stay as close as the oracle's trajectory stays
          to itself when its gradients carry 1e-7 relative noise -- conftest.ADAPTIVE_DRIFT, measured on the oracle alone by
          tests/test_oracle_extensions.py::test_adaptive_step_sensitivity_to_gradient_noise: every lambda_t within 2.5e-6 of
          the scale of lambda, lambda_T within 5e-8, every eta_t within 3e-5 relative; the final dual value within 1e-9
          relative (its drift part is 2e-11; the rest is the accuracy of one evaluation of g).  The CUDA path shows 1.8e-7 /
          1.5e-8 / 1.2e-6 / 1.3e-10 on the test instances ("Adaptive step and parity")."""
    emin, emax = eta_range
    out = gpu_solve(pg, gammas, iters)
    ref = oracle.solve(po, gammas, iters, momentum=momentum, jacobi=jacobi, adaptive=True, eta_min=emin, eta_max=emax, trace_lambda=True, trace_grad=True)
    R = pg.duals
    d = np.ones(R)
    if jacobi:
        d[:po.J * po.m] = oracle.jacobi_scaling(po)
        if po.count_M is not None:
            d[-1] = 1.0 / np.sqrt(po.nnz)
    L = oracle.lipschitz(po) if not jacobi else None
    if jacobi:                                                   # L' of the row-scaled system (R18, R21)
        nz = (np.bincount(np.repeat(po.item_idx.astype(np.int64), po.m) * po.m + np.tile(np.arange(po.m), po.nnz),
                          weights=np.abs(po.a), minlength=po.J * po.m) > 0).reshape(po.J, po.m)
        L = float(nz.sum(axis=1).max()) + (1.0 if po.count_M is not None else 0.0)
    n = 0
    lam_prev = np.zeros(R)
    worst_eta = 0.0
    for s, (gam, T) in enumerate(zip(gammas, iters)):
        hi = emax * gam / gammas[0]
        clip = lambda e, lo=min(emin, gam / L), hi=hi: min(max(e, lo), hi)
        y = lam_prev.copy()
        for t in range(T):
            g_gpu = out["tr_grad"][n]
            rg = oracle.grad(po, y, gam, want_x=False)
            e = rel_l2(g_gpu, rg.grad)
            assert e <= TOL_GRAD, f"{tag} stage {s} iteration {t}: grad at the CUDA path's own y_t, rel L2 {e:.3e}"
            want = clip(gam / L)
            if t >= 1:
                dy, dg = np.linalg.norm((y - y_old) / d), np.linalg.norm((g_gpu - g_old) * d)
                if dy > 0 and dg > 0:
                    want = clip(dy / dg)
            worst_eta = max(worst_eta, abs(out["tr_eta"][n] / want - 1.0))
            assert abs(out["tr_eta"][n] / want - 1.0) <= 1e-9, f"{tag} stage {s} iteration {t}: eta {out['tr_eta'][n]} vs {want}"
            lam_new = np.maximum(0.0, y + want * d * d * g_gpu)
            assert np.abs(out["tr_lam"][n] - lam_new).max() <= 1e-9 * max(np.abs(lam_new).max(), 1e-300) + 1e-15, f"{tag} lambda update {s}/{t}"
            lam_new = out["tr_lam"][n]
            y_old, g_old = y, g_gpu
            beta = t / (t + 3.0) if momentum else 0.0
            y = lam_new + beta * (lam_new - lam_prev)
            lam_prev = lam_new
            n += 1
    lam_scale = max(np.abs(ref.trace_lambda).max(), 1e-300)
    seen = {"lam_t": np.abs(out["tr_lam"] - ref.trace_lambda).max() / lam_scale, "lam_T": np.abs(out["lam"] - ref.lam).max() / lam_scale,
            "g_T": abs(out["sc"].g - ref.final.g) / abs(ref.final.g), "eta_t": np.abs(out["tr_eta"] / ref.trace_eta - 1.0).max(),
            "grad_t": max(rel_l2(out["tr_grad"][k], ref.trace_grad[k]) for k in range(n))}
    print(f"{tag} adaptive drift CUDA vs oracle: " + " ".join(f"{k}={v:.3e}" for k, v in seen.items()))
    for k in ("lam_t", "lam_T", "eta_t"):
        assert seen[k] <= ADAPTIVE_DRIFT[k], f"{tag} {k}: {seen[k]:.3e} exceeds the oracle's own drift under 1e-7 gradient noise ({ADAPTIVE_DRIFT[k]:g})"
    assert seen["g_T"] <= 1e-9, f"{tag} final g {out['sc'].g} vs {ref.final.g}"
    return ref, out
