"""Pins for the oracle's AGD / gamma-continuation loop.  The paper prints no update formula (P:123,
P:145 give words only) so parity with the paper is UNPINNED for this part (readings R1-R4);
what is pinned: the optimum it converges to (brute-force KKT active-set enumeration on <= 3 users x
2 items; I=J=1 closed form), the lambda==0 fixed point, monotone ascent of the beta==0 variant at
eta = gamma/L, the accelerated O(1/T^2) bound, stage/warm-start semantics and the drift bound."""
import itertools

import numpy as np
import pytest

import oracle
from conftest import random_problem


def _problem(d, kind=oracle.PROJ_SIMPLEX_INEQ, p0=1.0, p1=0.0):
    return oracle.Problem(d["I"], d["J"], d["m"], d["row_ptr"], d["item_idx"], d["c"], d["a"], d["b"], kind, p0, p1)


def _kkt_brute_force(d, gamma, eq_items=()):
    """min c'x + (gamma/2)|x|^2  s.t. x>=0, per-user sum<=1, per-item sum_i a_ij x_ij <= b_j, by
    enumerating active sets and solving each equality-constrained QP (Eq. 1).  Items in eq_items have
    sum_i a_ij x_ij = b_j instead: always active, multiplier free in sign."""
    n, I, J = d["item_idx"].size, d["I"], d["J"]
    c, a, b = d["c"].astype(np.float64), d["a"].astype(np.float64), d["b"].astype(np.float64)
    G, h = [], []
    for p in range(n):
        r = np.zeros(n); r[p] = -1.0; G.append(r); h.append(0.0)
    for i in range(I):
        r = np.zeros(n); r[d["row_ptr"][i]:d["row_ptr"][i + 1]] = 1.0; G.append(r); h.append(1.0)
    for j in range(J):
        r = np.zeros(n); sel = d["item_idx"] == j; r[sel] = a[sel]; G.append(r); h.append(b[j])
    G, h = np.array(G), np.array(h)
    forced = [n + I + j for j in eq_items]
    free = [k for k in range(len(h)) if k not in forced]
    best = None
    for r in range(0, min(n, len(h)) + 1):
        for S in itertools.combinations(free, r):
            S = forced + list(S)
            if S:
                GS = G[S]
                if np.linalg.matrix_rank(GS) < len(S):
                    continue
                mu = np.linalg.solve(GS @ GS.T, -(gamma * h[S] + GS @ c))
                x = -(c + GS.T @ mu) / gamma
                if (mu[len(forced):] < -1e-10).any():
                    continue
            else:
                x = -c / gamma
            if (G @ x <= h + 1e-10).all():
                val = c @ x + 0.5 * gamma * x @ x
                if best is None or val < best[0] - 1e-13:
                    best = (val, x)
    return best


@pytest.mark.parametrize("seed", range(6))
def test_converges_to_kkt_optimum(seed):
    rng = np.random.default_rng(seed)
    d = random_problem(rng, I=int(rng.integers(1, 4)), J=2, m=1, deg=(1, 2), tight=0.7)
    d["b"] = (0.15 + 0.5 * rng.random(2)).astype(np.float32)
    gamma = float(rng.choice([1.0, 0.3]))
    p_star, x_star = _kkt_brute_force(d, gamma)
    res = oracle.solve(_problem(d), [gamma], [4000])
    assert abs(res.final.g - p_star) < 1e-8 * (1 + abs(p_star))          # strong duality
    np.testing.assert_allclose(res.x, x_star, atol=1e-5)
    assert np.all(res.lam >= 0)
    assert np.max(np.abs(res.lam * res.final.grad)) < 1e-6                # complementary slackness
    assert res.final.r_inf < 1e-6
    # every iterate's dual value is a lower bound on p* (weak duality)
    assert np.all(res.trace_g <= p_star + 1e-10)


def test_single_variable_closed_form():
    """I=J=1: x = clip(-(c + a lam)/gamma, 0, 1); if 0 < b/a < 1 binds, lam* = max(0, -(c + gamma b/a)/a)."""
    c, a, b, gamma = -1.0, 2.0, 0.5, 0.25
    d = dict(I=1, J=1, m=1, row_ptr=np.array([0, 1]), item_idx=np.array([0], dtype=np.int32),
             c=np.array([c], dtype=np.float32), a=np.array([a], dtype=np.float32), b=np.array([b], dtype=np.float32))
    res = oracle.solve(_problem(d), [gamma], [3000])
    lam_star = max(0.0, -(c + gamma * b / a) / a)
    assert abs(res.lam[0] - lam_star) < 1e-9
    assert abs(res.x[0] - b / a) < 1e-9


def test_lambda_zero_is_a_fixed_point_when_slack():
    """grad g(0) <= 0  =>  lambda_t = 0 for all t (what every verbatim BASELINE.json config does)."""
    rng = np.random.default_rng(3)
    d = random_problem(rng, I=50, J=6, m=1, deg=(2, 5))
    d["b"] = np.full(6, 1e3, dtype=np.float32)
    res = oracle.solve(_problem(d), [0.01], [25], trace_lambda=True)
    assert np.all(res.trace_lambda == 0.0)
    assert np.all(res.trace_g == res.trace_g[0])


@pytest.mark.parametrize("m", [1, 2])
def test_plain_ascent_is_monotone_at_eta_gamma_over_L(m):
    rng = np.random.default_rng(20 + m)
    d = random_problem(rng, I=120, J=8, m=m, deg=(2, 6), tight=0.4)
    p = _problem(d)
    res = oracle.solve(p, [0.2], [150], momentum=False, trace_lambda=True)
    g_at_iterates = np.array([oracle.grad(p, l, 0.2, want_x=False).g for l in res.trace_lambda[::10]])
    assert np.all(np.diff(g_at_iterates) >= -1e-12)
    assert np.all(np.diff(res.trace_g) >= -1e-12)                            # beta = 0: y_t = lambda_t


@pytest.mark.parametrize("seed", range(3))
def test_accelerated_rate_bound(seed):
    """p* - g(lambda_T) <= 4 L |lambda_0 - lambda*|^2 / (gamma (T+1)^2)   (FISTA-type bound)."""
    rng = np.random.default_rng(50 + seed)
    d = random_problem(rng, I=3, J=2, m=1, deg=(2, 2), tight=0.6)
    d["b"] = (0.2 + 0.3 * rng.random(2)).astype(np.float32)
    gamma = 0.5
    p = _problem(d)
    p_star, _ = _kkt_brute_force(d, gamma)
    lam_star = oracle.solve(p, [gamma], [6000]).lam
    L = oracle.lipschitz(p)
    for T in (5, 20, 80):
        res = oracle.solve(p, [gamma], [T])
        assert p_star - res.final.g <= 4.0 * L * (lam_star @ lam_star) / (gamma * (T + 1) ** 2) + 1e-12


def test_first_step_and_trace_semantics():
    rng = np.random.default_rng(31)
    d = random_problem(rng, I=60, J=7, m=2, deg=(2, 5), tight=0.4)
    p = _problem(d)
    gamma, lam0 = 0.3, rng.random(14) * 0.1
    res = oracle.solve(p, [gamma], [3], lam0=lam0, trace_grad=True, trace_lambda=True)
    g0 = oracle.grad(p, lam0, gamma)
    eta = gamma / oracle.lipschitz(p)
    np.testing.assert_allclose(res.trace_grad[0], g0.grad, atol=0)
    assert res.trace_g[0] == g0.g
    lam1 = np.maximum(0.0, lam0 + eta * g0.grad)
    np.testing.assert_allclose(res.trace_lambda[0], lam1, atol=1e-15)
    # t = 0: beta = 0 so y_1 = lambda_1; t = 1: beta = 1/4
    g1 = oracle.grad(p, lam1, gamma)
    np.testing.assert_allclose(res.trace_grad[1], g1.grad, atol=1e-15)
    lam2 = np.maximum(0.0, lam1 + eta * g1.grad)
    y2 = lam2 + 0.25 * (lam2 - lam1)
    np.testing.assert_allclose(res.trace_grad[2], oracle.grad(p, y2, gamma).grad, atol=1e-13)
    # final evaluation is at lambda_T (reading R3), not at y
    fin = oracle.grad(p, res.lam, gamma)
    assert fin.g == res.final.g
    np.testing.assert_allclose(fin.x, res.x, atol=0)


def test_continuation_equals_chained_warm_started_solves():
    rng = np.random.default_rng(32)
    d = random_problem(rng, I=80, J=6, m=1, deg=(2, 5), tight=0.4)
    p = _problem(d)
    full = oracle.solve(p, [1.0, 0.1, 0.01], [30, 20, 10], stage_x=True)
    lam = None
    for s, (gam, it) in enumerate(zip([1.0, 0.1, 0.01], [30, 20, 10])):
        part = oracle.solve(p, [gam], [it], lam0=lam)
        lam = part.lam
        np.testing.assert_allclose(full.stage_x[s], part.x, atol=0)
    np.testing.assert_allclose(full.lam, lam, atol=0)


def test_drift_bound():
    """At fixed lambda, |x(c) - x(c')|_2 <= |c - c'|_2 / gamma (non-expansive projection of -c/gamma);
    the closed form behind the paper's stability claim."""
    rng = np.random.default_rng(33)
    d = random_problem(rng, I=200, J=9, m=1, deg=(2, 8))
    lam = rng.random(9) * 0.2
    for gamma in (1.0, 0.1, 0.01):
        d2 = dict(d)
        d2["c"] = (d["c"] * (1 + 0.01 * rng.normal(size=d["c"].size))).astype(np.float32)
        x1 = oracle.grad(_problem(d), lam, gamma).x
        x2 = oracle.grad(_problem(d2), lam, gamma).x
        dc = np.linalg.norm(d["c"].astype(np.float64) - d2["c"].astype(np.float64))
        assert np.linalg.norm(x1 - x2) <= dc / gamma + 1e-12


# ---- Jacobi preconditioning / row normalisation (reading R18) ------------------------

def _explicit_A(d):
    """The (J*m) x nnz coupling matrix of Definition 1, row r = j*m + k, written out densely."""
    nnz, m = d["item_idx"].size, d["m"]
    A = np.zeros((d["J"] * m, nnz))
    for p, j in enumerate(d["item_idx"]):
        for k in range(m):
            A[j * m + k, p] = np.float64(d["a"][p * m + k])
    return A


@pytest.mark.parametrize("m", [1, 2])
def test_jacobi_scaling_is_inverse_row_norm(m):
    """D_rr = 1/|A_r*|_2 against numpy's norm of the explicit rows; diag(A'A'^T) = I;
    a row of zero norm keeps D_rr = 1."""
    rng = np.random.default_rng(7 + m)
    d = random_problem(rng, I=40, J=9, m=m, deg=(1, 5))
    d["item_idx"] = np.where(d["item_idx"] == 8, 7, d["item_idx"]).astype(np.int32)   # item 8 unused -> zero rows
    # the substitution may create duplicates inside a row; the scaling formula does not care
    dd = oracle.jacobi_scaling(_problem(d))
    A = _explicit_A(d)
    nrm = np.linalg.norm(A, axis=1)
    np.testing.assert_allclose(dd[nrm > 0], 1.0 / nrm[nrm > 0], rtol=1e-14)
    assert np.all(dd[nrm == 0] == 1.0) and (nrm == 0).sum() == m
    As = dd[:, None] * A
    np.testing.assert_allclose(np.diag(As @ As.T)[nrm > 0], 1.0, rtol=1e-13)


def test_jacobi_preserves_feasible_set():
    """{x : Ax <= b} = {x : A'x <= b'} on sampled x, including points near the boundary."""
    rng = np.random.default_rng(11)
    d = random_problem(rng, I=25, J=6, m=2, deg=(1, 4))
    dd = oracle.jacobi_scaling(_problem(d))
    A, b = _explicit_A(d), d["b"].astype(np.float64)
    for _ in range(200):
        x = rng.random(A.shape[1]) * rng.choice([0.05, 0.3, 1.0])
        assert np.array_equal(A @ x <= b, (dd[:, None] * A) @ x <= dd * b)


def test_jacobi_first_step_is_per_coordinate_step():
    """m = 1: A'A'^T = I exactly (Def. 1: each item's row touches its own columns only), so L' = 1, eta' = gamma, and
    lambda_1 = D max(0, gamma D grad g(0)) = max(0, gamma d^2 grad g(0)) -- from oracle.grad alone."""
    rng = np.random.default_rng(3)
    d = random_problem(rng, I=60, J=7, m=1, deg=(2, 5), tight=0.3)
    p, gamma = _problem(d), 0.05
    dd = oracle.jacobi_scaling(p)
    g0 = oracle.grad(p, np.zeros(7), gamma).grad
    res = oracle.solve(p, [gamma], [1], jacobi=True, trace_lambda=True, trace_grad=True)
    np.testing.assert_allclose(res.trace_lambda[0], np.maximum(0.0, gamma * dd ** 2 * g0), rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(res.trace_grad[0], g0, rtol=1e-12, atol=1e-13)      # reported in original units
    assert (res.trace_lambda[0] > 0).any()


def test_jacobi_equals_plain_solve_of_prescaled_problem():
    """With power-of-two row norms the scaling is exact in fp32, so solving the scaled data with the plain loop and
    mapping lambda = D lambda' must reproduce the jacobi solve to rounding (lambda = D lambda')."""
    rng = np.random.default_rng(5)
    J = 4
    col_val = np.array([0.5, 1.0, 2.0, 4.0])                          # 16 users of equal |a|: |col_j| = val_j * 4
    I = 16
    rows = np.arange(I + 1, dtype=np.int64) * J
    idx = np.tile(np.arange(J, dtype=np.int32), I)
    a = np.tile(col_val, I).astype(np.float32)
    c = (-rng.random(I * J)).astype(np.float32)
    b = (np.array([0.5, 1.0, 2.0, 4.0]) * 2.0).astype(np.float32)
    d = dict(I=I, J=J, m=1, row_ptr=rows, item_idx=idx, c=c, a=a, b=b)
    p = _problem(d)
    dd = oracle.jacobi_scaling(p)
    np.testing.assert_array_equal(dd, 1.0 / (col_val * 4.0))
    ds = dict(d, a=(a * np.tile(dd, I)).astype(np.float32), b=(b * dd).astype(np.float32))
    gam, its = [0.5, 0.05], [60, 60]
    rj = oracle.solve(p, gam, its, jacobi=True, trace_lambda=True)
    rs = oracle.solve(_problem(ds), gam, its, trace_lambda=True)
    np.testing.assert_allclose(rj.trace_lambda, rs.trace_lambda * dd, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(rj.trace_g, rs.trace_g, rtol=1e-12)
    np.testing.assert_allclose(rj.x, rs.x, atol=1e-12)
    assert (rj.lam > 0).any()


@pytest.mark.parametrize("seed", range(4))
def test_jacobi_converges_to_same_kkt_optimum(seed):
    """Row scaling leaves the primal problem unchanged, so the optimum is the brute-force one; the returned
    lambda is the dual of the ORIGINAL rows: complementary slackness holds against the unscaled gradient."""
    rng = np.random.default_rng(100 + seed)
    d = random_problem(rng, I=int(rng.integers(2, 4)), J=2, m=1, deg=(1, 2), tight=0.7)
    d["a"] = (d["a"] * np.where(d["item_idx"] == 0, 8.0, 0.25)).astype(np.float32)   # badly scaled rows
    d["b"] = (np.array([8.0, 0.25]) * (0.15 + 0.5 * rng.random(2))).astype(np.float32)
    gamma = 0.3
    p_star, x_star = _kkt_brute_force(d, gamma)
    res = oracle.solve(_problem(d), [gamma], [4000], jacobi=True)
    assert abs(res.final.g - p_star) < 1e-8 * (1 + abs(p_star))
    np.testing.assert_allclose(res.x, x_star, atol=1e-5)
    assert np.all(res.lam >= 0) and np.max(np.abs(res.lam * res.final.grad)) < 1e-6
    # and it gets there at least as fast as the scalar step on these badly scaled rows
    plain = oracle.solve(_problem(d), [gamma], [300])
    jac = oracle.solve(_problem(d), [gamma], [300], jacobi=True)
    assert p_star - jac.final.g <= p_star - plain.final.g + 1e-12


def test_jacobi_warm_start_and_stages_chain():
    """lambda in original units in and out: two chained jacobi solves == one two-stage jacobi solve (R4, R18)."""
    rng = np.random.default_rng(21)
    d = random_problem(rng, I=50, J=6, m=2, deg=(2, 5), tight=0.3)
    p = _problem(d)
    both = oracle.solve(p, [0.5, 0.1], [40, 30], jacobi=True)
    first = oracle.solve(p, [0.5], [40], jacobi=True)
    second = oracle.solve(p, [0.1], [30], lam0=first.lam, jacobi=True)
    np.testing.assert_allclose(second.lam, both.lam, rtol=1e-12, atol=1e-15)
    assert (both.lam > 0).any()


# ---- equality coupling rows: the dual of an equality is free in sign, so the lambda >= 0 projection applies to
# "inequality coordinates" only (reading R19) ---------------------------------------------------------

def test_equality_row_closed_form_needs_a_negative_dual():
    """I=J=1, c=-0.1, a=1, gamma=1: the unconstrained ridge primal is x = 0.1.  As an inequality x <= 0.9 is slack
    (lambda stays 0, x = 0.1); as an equality x = 0.9 needs lambda* = -(c + gamma b/a)/a = -0.8 < 0."""
    d = dict(I=1, J=1, m=1, row_ptr=np.array([0, 1]), item_idx=np.array([0], dtype=np.int32),
             c=np.array([-0.1], dtype=np.float32), a=np.array([1.0], dtype=np.float32), b=np.array([0.9], dtype=np.float32))
    ineq = oracle.solve(_problem(d), [1.0], [2000])
    assert ineq.lam[0] == 0.0 and abs(ineq.x[0] - np.float64(np.float32(0.1))) < 1e-12
    eq = oracle.solve(_problem(d), [1.0], [2000], is_eq=[1])
    lam_star = -(np.float64(np.float32(-0.1)) + np.float64(np.float32(0.9)))
    assert abs(eq.lam[0] - lam_star) < 1e-9 and lam_star < -0.7
    assert abs(eq.x[0] - np.float64(np.float32(0.9))) < 1e-9
    assert eq.trace_rinf[0] == pytest.approx(abs(0.1 - 0.9), rel=1e-6)       # |Ax - b| at lambda = 0, not max(.,0) = 0
    assert eq.trace_rinf[-1] < 1e-8


@pytest.mark.parametrize("seed", range(5))
def test_equality_rows_converge_to_kkt_optimum(seed):
    """Item 0 is an equality row, item 1 an inequality: brute force with the equality always active."""
    rng = np.random.default_rng(300 + seed)
    d = random_problem(rng, I=int(rng.integers(2, 4)), J=2, m=1, deg=(2, 2), tight=0.7)
    # a feasible, not-trivially-slack right-hand side: item 0 must carry exactly 30-60 % of what its users could give
    sel0 = d["item_idx"] == 0
    d["b"] = np.array([(0.3 + 0.3 * rng.random()) * d["a"][sel0].min(), 0.15 + 0.5 * rng.random()], dtype=np.float32)
    gamma = 0.5
    best = _kkt_brute_force(d, gamma, eq_items=(0,))
    assert best is not None
    p_star, x_star = best
    res = oracle.solve(_problem(d), [gamma], [6000], is_eq=[1, 0])
    np.testing.assert_allclose(res.x, x_star, atol=1e-5)
    assert abs(res.final.g - p_star) < 1e-7 * (1 + abs(p_star))
    A0 = sum(np.float64(d["a"][p]) * res.x[p] for p in range(d["item_idx"].size) if d["item_idx"][p] == 0)
    assert abs(A0 - np.float64(d["b"][0])) < 1e-6                          # the equality holds at the limit
    assert res.lam[1] >= 0.0                                               # the inequality's dual stays projected


def test_equality_mask_all_zero_is_the_plain_loop():
    rng = np.random.default_rng(9)
    d = random_problem(rng, I=40, J=5, m=2, deg=(2, 4), tight=0.3)
    a = oracle.solve(_problem(d), [0.2], [50], trace_lambda=True)
    b = oracle.solve(_problem(d), [0.2], [50], trace_lambda=True, is_eq=np.zeros(10, dtype=np.uint8))
    np.testing.assert_array_equal(a.trace_lambda, b.trace_lambda)
    np.testing.assert_array_equal(a.trace_rinf, b.trace_rinf)
