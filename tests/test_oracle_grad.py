"""Pins for the oracle's g, grad g, x* (Eq. 2-4): hand-worked examples, the definition of g
as a minimum of the Lagrangian, a library re-computation of A x - b, central finite differences,
concavity, weak duality, row-scaling invariance, additivity over users.  CPU only."""
import numpy as np
import pytest

import oracle
from conftest import random_problem, read_worked_examples


def _problem(d, kind=oracle.PROJ_SIMPLEX_INEQ, p0=1.0, p1=0.0):
    return oracle.Problem(d["I"], d["J"], d["m"], d["row_ptr"], d["item_idx"], d["c"], d["a"], d["b"], kind, p0, p1)


@pytest.mark.parametrize("ex", read_worked_examples(), ids=lambda e: e["case"])
def test_worked_examples(ex):
    r = oracle.grad(_problem(ex), ex["lambda"], ex["gamma"])
    np.testing.assert_allclose(r.x, ex["x"], atol=1e-14)
    np.testing.assert_allclose(r.grad, ex["grad"], atol=1e-14)
    for key in ("g", "obj", "reg", "r_inf", "r_2"):
        assert abs(getattr(r, key) - ex[key]) < 1e-13, key


def _lagrangian(d, x, lam, gamma):
    """c'x + (gamma/2)|x|^2 + lambda'(Ax - b) with A x by numpy scatter-add (library routine)."""
    m, J = d["m"], d["J"]
    s = np.zeros(J * m)
    a = d["a"].astype(np.float64).reshape(-1, m)
    for k in range(m):
        np.add.at(s, d["item_idx"].astype(np.int64) * m + k, a[:, k] * x)
    c = d["c"].astype(np.float64)
    return c @ x + 0.5 * gamma * (x @ x) + lam @ (s - d["b"].astype(np.float64)), s


@pytest.mark.parametrize("m", [1, 2, 3])
@pytest.mark.parametrize("kind,p0,p1", [(oracle.PROJ_SIMPLEX_INEQ, 1.0, 0.0), (oracle.PROJ_BOXCUT, 0.4, 1.0),
                                        (oracle.PROJ_BOX, 0.0, 0.6), (oracle.PROJ_SIMPLEX_EQ, 1.0, 0.0)])
def test_g_is_the_minimum_of_the_lagrangian(m, kind, p0, p1):
    rng = np.random.default_rng(10 * m + kind)
    d = random_problem(rng, I=40, J=7, m=m, deg=(3, 6))
    p = _problem(d, kind, p0, p1)
    for gamma in (1.0, 0.05):
        lam = rng.random(d["J"] * m) * rng.choice([0.0, 0.3, 2.0])
        r = oracle.grad(p, lam, gamma)
        L_star, s = _lagrangian(d, r.x, lam, gamma)
        assert abs(L_star - r.g) <= 1e-12 * (1 + abs(r.g))                      # g = L(x*, lambda)
        np.testing.assert_allclose(r.grad, s - d["b"].astype(np.float64), atol=1e-12)   # Eq. 4 via numpy
        for _ in range(30):                                                      # ... and x* minimises L over C
            xt = np.empty_like(r.x)
            for i in range(d["I"]):
                lo, hi = d["row_ptr"][i], d["row_ptr"][i + 1]
                v = rng.normal(0.2, 0.5, hi - lo)
                xt[lo:hi] = {0: oracle.project_simplex, 3: oracle.project_simplex_eq}.get(
                    kind, None)(v, p0) if kind in (0, 3) else (
                    oracle.project_boxcut(v, p0, p1) if kind == oracle.PROJ_BOXCUT else oracle.project_box(v, p0, p1))
            assert _lagrangian(d, xt, lam, gamma)[0] >= r.g - 1e-10
            mix = 0.9 * r.x + 0.1 * xt                                           # nearby feasible point (C convex)
            assert _lagrangian(d, mix, lam, gamma)[0] >= r.g - 1e-10


@pytest.mark.parametrize("m", [1, 2])
def test_finite_differences(m):
    rng = np.random.default_rng(100 + m)
    d = random_problem(rng, I=60, J=9, m=m, deg=(2, 6))
    p = _problem(d)
    for gamma in (0.5, 0.05):
        for _ in range(10):
            lam = rng.random(d["J"] * m) * 0.5
            dirn = rng.normal(size=lam.size); dirn /= np.linalg.norm(dirn)
            h = 1e-6
            fd = (oracle.grad(p, lam + h * dirn, gamma).g - oracle.grad(p, lam - h * dirn, gamma).g) / (2 * h)
            an = oracle.grad(p, lam, gamma).grad @ dirn
            assert abs(fd - an) <= 1e-6 * (1 + abs(an)), (fd, an)


def test_concavity_and_weak_duality():
    rng = np.random.default_rng(11)
    d = random_problem(rng, I=80, J=10, m=1, deg=(2, 7), tight=0.6)
    p = _problem(d)
    gamma = 0.1
    for _ in range(20):
        l1, l2 = rng.random(10) * 0.8, rng.random(10) * 0.8
        r1, r2 = oracle.grad(p, l1, gamma), oracle.grad(p, l2, gamma)
        assert r2.g <= r1.g + r1.grad @ (l2 - l1) + 1e-10                       # concave: below every tangent
        assert r1.g <= 1e-12                                                     # x = 0 feasible (b>=0) => g <= 0
        # weak duality against a feasible primal point: shrink x*(l2) until A x <= b
        x = r2.x.copy()
        _, s = _lagrangian(d, x, np.zeros(10), gamma)
        scale = min(1.0, float(np.min(np.where(s > 0, d["b"] / np.maximum(s, 1e-300), np.inf))))
        xf = x * scale
        primal = d["c"].astype(np.float64) @ xf + 0.5 * gamma * xf @ xf
        assert r1.g <= primal + 1e-10


def test_row_scaling_invariance():
    """(a_.j, b_j) -> d_j (a_.j, b_j), lambda_j -> lambda_j / d_j leaves x* and g unchanged."""
    rng = np.random.default_rng(12)
    d = random_problem(rng, I=50, J=8, m=1, deg=(2, 5))
    scale = np.array([0.5, 2.0, 4.0, 0.25, 1.0, 8.0, 2.0, 0.5])              # powers of two: exact in fp32
    d2 = dict(d)
    d2["a"] = (d["a"] * scale[d["item_idx"]]).astype(np.float32)
    d2["b"] = (d["b"] * scale).astype(np.float32)
    lam = rng.random(8)
    r1, r2 = oracle.grad(_problem(d), lam, 0.2), oracle.grad(_problem(d2), lam / scale, 0.2)
    np.testing.assert_allclose(r1.x, r2.x, atol=1e-13)
    assert abs(r1.g - r2.g) < 1e-12
    np.testing.assert_allclose(r2.grad, r1.grad * scale, atol=1e-12)


def test_additivity_over_users():
    rng = np.random.default_rng(13)
    d = random_problem(rng, I=30, J=6, m=2, deg=(1, 5))
    p = _problem(d)
    lam = rng.random(12) * 0.3
    full = oracle.grad(p, lam, 0.3)
    cut = 11
    k = d["row_ptr"][cut]
    zero_b = np.zeros_like(d["b"])
    pa = oracle.Problem(cut, 6, 2, d["row_ptr"][:cut + 1], d["item_idx"][:k], d["c"][:k], d["a"][:2 * k], zero_b)
    pb = oracle.Problem(30 - cut, 6, 2, d["row_ptr"][cut:] - k, d["item_idx"][k:], d["c"][k:], d["a"][2 * k:], zero_b)
    ra, rb = oracle.grad(pa, lam, 0.3), oracle.grad(pb, lam, 0.3)
    np.testing.assert_allclose(full.grad, ra.grad + rb.grad - d["b"].astype(np.float64), atol=1e-12)
    np.testing.assert_allclose(full.x, np.concatenate([ra.x, rb.x]), atol=0)
    assert abs(full.obj - (ra.obj + rb.obj)) < 1e-12 and abs(full.reg - (ra.reg + rb.reg)) < 1e-12


def test_empty_rows_and_negative_lambda():
    d = dict(I=3, J=2, m=1, row_ptr=np.array([0, 0, 2, 2]), item_idx=np.array([0, 1], dtype=np.int32),
             c=np.array([-1.0, -0.5], dtype=np.float32), a=np.ones(2, dtype=np.float32),
             b=np.array([0.3, 0.3], dtype=np.float32))
    r = oracle.grad(_problem(d), np.array([-0.5, 0.0]), 1.0)      # g is defined on all of R^{mJ}
    np.testing.assert_allclose(r.x, [1.0, 0.0], atol=1e-15)        # v = (1.5, 0.5) -> theta = 0.5
    np.testing.assert_allclose(r.grad, [0.7, -0.3], atol=1e-15)


def test_lipschitz_constant():
    rng = np.random.default_rng(14)
    d = random_problem(rng, I=40, J=5, m=2, deg=(1, 4))
    col = np.zeros(5)
    np.add.at(col, d["item_idx"], (d["a"].astype(np.float64).reshape(-1, 2) ** 2).sum(1))
    assert abs(oracle.lipschitz(_problem(d)) - col.max()) < 1e-12
    # m = 1: equals |A|_2^2 of the explicit mJ x nnz coupling matrix (Def. 1)
    d1 = random_problem(rng, I=25, J=4, m=1, deg=(1, 4))
    A = np.zeros((4, d1["item_idx"].size))
    A[d1["item_idx"], np.arange(d1["item_idx"].size)] = d1["a"]
    assert abs(oracle.lipschitz(_problem(d1)) - np.linalg.norm(A, 2) ** 2) < 1e-10
    # m = 2: an upper bound on |A|_2^2
    A2 = np.zeros((10, d["item_idx"].size))
    for k in range(2):
        A2[d["item_idx"] * 2 + k, np.arange(d["item_idx"].size)] = d["a"].reshape(-1, 2)[:, k]
    assert np.linalg.norm(A2, 2) ** 2 <= oracle.lipschitz(_problem(d)) + 1e-10
