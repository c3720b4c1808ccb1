"""Pins for the oracle's projections: hand-worked closed forms, a second independent
method (bisection on theta), brute force over supports / partitions, the variational inequality that
characterises a Euclidean projection, and structural invariants.  CPU only."""
import itertools

import numpy as np
import pytest

import oracle
from conftest import read_projection_cases


def _call(kind, params, v):
    if kind == "simplex":
        return oracle.project_simplex(v, params[0])
    if kind == "simplex_eq":
        return oracle.project_simplex_eq(v, params[0])
    if kind == "box":
        return oracle.project_box(v, params[0], params[1])
    if kind == "boxcut":
        return oracle.project_boxcut(v, params[0], params[1])
    raise ValueError(kind)


@pytest.mark.parametrize("kind,params,v,x", read_projection_cases())
def test_hand_worked_cases(kind, params, v, x):
    np.testing.assert_allclose(_call(kind, params, v), x, rtol=0, atol=1e-14)


def _bisect_theta(v, ub, z, iters=200):
    """Second method: x = clip(v - theta, 0, ub) with theta >= 0 the root of sum x = z (if needed)."""
    phi = lambda th: np.clip(v - th, 0.0, ub).sum()
    if phi(0.0) <= z:
        return np.clip(v, 0.0, ub)
    lo, hi = 0.0, float(v.max())
    for _ in range(iters):
        mid = 0.5 * (lo + hi)
        if phi(mid) > z:
            lo = mid
        else:
            hi = mid
    return np.clip(v - 0.5 * (lo + hi), 0.0, ub)


@pytest.mark.parametrize("seed", range(6))
def test_against_bisection(seed):
    rng = np.random.default_rng(seed)
    for _ in range(200):
        n = int(rng.integers(1, 40))
        v = rng.normal(0.2, rng.choice([0.3, 2.0, 30.0]), size=n)
        z = float(rng.choice([1.0, 0.5, 2.5]))
        np.testing.assert_allclose(oracle.project_simplex(v, z), _bisect_theta(v, np.inf, z), atol=1e-12)
        ub = float(rng.choice([0.15, 0.3, 0.6, 1.0, 3.0]))
        np.testing.assert_allclose(oracle.project_boxcut(v, ub, z), _bisect_theta(v, ub, z), atol=1e-12)


def _brute_simplex(v, z):
    """Enumerate supports S: on the face sum=z, x_S = v_S - (sum v_S - z)/|S|; keep feasible, nearest."""
    p = np.maximum(v, 0.0)
    if p.sum() <= z:
        return p
    best, bd = None, np.inf
    n = v.size
    for r in range(1, n + 1):
        for S in itertools.combinations(range(n), r):
            S = list(S)
            x = np.zeros(n)
            x[S] = v[S] - (v[S].sum() - z) / r
            if (x >= -1e-15).all():
                d = np.sum((x - v) ** 2)
                if d < bd:
                    best, bd = x, d
    return np.maximum(best, 0.0)


def _brute_boxcut(v, ub, z):
    """Enumerate (lower, free, upper) partitions on the face sum = z."""
    p = np.clip(v, 0.0, ub)
    if p.sum() <= z:
        return p
    best, bd = None, np.inf
    n = v.size
    for lab in itertools.product((0, 1, 2), repeat=n):
        lab = np.array(lab)
        F, U = np.where(lab == 1)[0], np.where(lab == 2)[0]
        x = np.zeros(n)
        x[U] = ub
        if F.size:
            x[F] = v[F] - (v[F].sum() + ub * U.size - z) / F.size
        if abs(x.sum() - z) > 1e-12 or (x < -1e-15).any() or (x > ub + 1e-15).any():
            continue
        d = np.sum((x - v) ** 2)
        if d < bd:
            best, bd = x, d
    return best


def test_brute_force_small():
    rng = np.random.default_rng(42)
    for _ in range(300):
        n = int(rng.integers(1, 6))
        v = rng.normal(0.3, 1.0, size=n)
        np.testing.assert_allclose(oracle.project_simplex(v, 1.0), _brute_simplex(v, 1.0), atol=1e-12)
    for _ in range(150):
        n = int(rng.integers(1, 5))
        v = rng.normal(0.4, 1.0, size=n)
        ub = float(rng.choice([0.3, 0.45, 0.7]))
        if ub * n < 1.0 and np.clip(v, 0, ub).sum() > 1.0:
            continue  # face unreachable: clipping alone is the projection only if sum<=z (excluded above)
        np.testing.assert_allclose(oracle.project_boxcut(v, ub, 1.0), _brute_boxcut(v, ub, 1.0), atol=1e-12)


def _sample_feasible(rng, kind, n, params):
    if kind == "box":
        return rng.uniform(params[0], params[1], size=n)
    ub = params[0] if kind == "boxcut" else np.inf
    z = params[1] if kind == "boxcut" else params[0]
    y = rng.random(n) ** rng.choice([1, 4]) * min(ub, z)
    s = y.sum()
    if kind == "simplex_eq":
        return y * (z / s)
    if s > z:
        y *= z / s * rng.random()
    return y


@pytest.mark.parametrize("kind,params", [("simplex", [1.0]), ("simplex", [0.4]), ("simplex_eq", [1.0]),
                                         ("box", [-0.5, 0.7]), ("boxcut", [0.3, 1.0]), ("boxcut", [0.8, 1.5])])
def test_variational_inequality(kind, params):
    """x = Proj_C(v)  <=>  x in C and (v - x).(y - x) <= 0 for every y in C."""
    rng = np.random.default_rng(7)
    for _ in range(100):
        n = int(rng.integers(1, 30))
        if kind == "boxcut" and params[0] * n < params[1]:
            n = int(np.ceil(params[1] / params[0])) + 1
        v = rng.normal(0.2, rng.choice([0.5, 5.0]), size=n)
        x = _call(kind, params, v)
        if kind == "box":
            assert (x >= params[0] - 1e-15).all() and (x <= params[1] + 1e-15).all()
        else:
            z = params[1] if kind == "boxcut" else params[0]
            assert (x >= 0).all() and x.sum() <= z + 1e-12
            if kind == "simplex_eq":
                assert abs(x.sum() - z) < 1e-12
            if kind == "boxcut":
                assert (x <= params[0] + 1e-15).all()
        for _ in range(20):
            y = _sample_feasible(rng, kind, n, params)
            assert np.dot(v - x, y - x) <= 1e-10 * (1 + np.abs(v).max())


def test_invariants():
    rng = np.random.default_rng(3)
    for _ in range(200):
        n = int(rng.integers(1, 50))
        u, v = rng.normal(0, 2, n), rng.normal(0, 2, n)
        for f in (lambda t: oracle.project_simplex(t, 1.0), lambda t: oracle.project_boxcut(t, 0.4, 1.0),
                  lambda t: oracle.project_box(t, 0.0, 1.0), lambda t: oracle.project_simplex_eq(t, 1.0)):
            xu, xv = f(u), f(v)
            np.testing.assert_allclose(f(xu), xu, atol=1e-13)                         # idempotent
            assert np.linalg.norm(xu - xv) <= np.linalg.norm(u - v) + 1e-12           # non-expansive
            perm = rng.permutation(n)
            np.testing.assert_allclose(f(u[perm]), xu[perm], atol=1e-13)              # permutation equivariant


def test_boxcut_reduces_to_simplex_when_ub_ge_z():
    """DESIGN.md reading R10: configs 3 and 5's "simplex with box x<=1" is the unit simplex itself."""
    rng = np.random.default_rng(5)
    for _ in range(300):
        v = rng.normal(0.3, rng.choice([0.5, 3.0, 50.0]), size=int(rng.integers(1, 60)))
        np.testing.assert_allclose(oracle.project_boxcut(v, 1.0, 1.0), oracle.project_simplex(v, 1.0), atol=1e-12)
        np.testing.assert_allclose(oracle.project_boxcut(v, 2.0, 1.0), oracle.project_simplex(v, 1.0), atol=1e-12)


def test_empty_row():
    assert oracle.project_simplex(np.zeros(0)).size == 0
    assert oracle.project_boxcut(np.zeros(0), 0.5, 1.0).size == 0
