"""pytest configuration: registers the `gpu` marker and shared helpers/fixtures."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: full-size GPU parity cases (minutes)")
    if os.environ.get("DUALIP_TEST_CHECKED") == "1":
        _use_checked_build()


# ---- checked build (tests/test_gpu_checked_build.py re-runs GPU tests with DUALIP_TEST_CHECKED=1): the binding loads the
# -DDUALIP_CHECKED library, and every handle's bounds-violation mask is read before the handle goes away.
_CHECK_FAILURES = []


def _use_checked_build():
    from paper_2606_07777_b200 import binding, build
    lib = build.build_checked()
    binding.lib_path = lambda: lib
    orig = binding.Problem.destroy

    def destroy(self):
        if self._h:
            inf = self.info()
            if inf.checked_build != 1 or inf.checks_failed != 0:
                _CHECK_FAILURES.append(f"checked_build={inf.checked_build} checks_failed={inf.checks_failed:#x} (I={inf.I}, J={inf.J}, G={inf.group_lanes})")
        orig(self)

    binding.Problem.destroy = destroy


@pytest.fixture(autouse=True)
def _no_bounds_violations():
    yield
    if os.environ.get("DUALIP_TEST_CHECKED") == "1":
        import gc
        gc.collect()
        assert not _CHECK_FAILURES, _CHECK_FAILURES


# How far the ORACLE's own adaptive-step trajectory (R20) moves when every gradient it sees carries ADAPTIVE_NOISE relative
# noise -- upper bounds, measured and asserted by tests/test_oracle_extensions.py::test_adaptive_step_sensitivity_to_gradient_noise
# on the instance of tests/test_gpu_extensions.py::test_adaptive_step_trajectory.  gpu_util.assert_adaptive_step_parity holds the
# CUDA path's independent trajectory to these (its gradients are good to about 1e-7; what it shows is 10-20 x smaller).
# lam_t: max over iterations of |lambda_t - lambda_t'|_inf / max|lambda|;  lam_T: the same at the end;  eta_t: max relative
# difference of the steps;  g_T: relative difference of the final dual value.
ADAPTIVE_NOISE = 1e-7
ADAPTIVE_DRIFT = {"lam_t": 2.5e-6, "lam_T": 5e-8, "eta_t": 3e-5, "g_T": 2e-11}


def ragged_problem(rng, I, J, m, lens):
    """rows with prescribed lengths (0 allowed), items unsorted in every third row (tests only)."""
    rows, idx = [0], []
    for i in range(I):
        d = int(lens[i % len(lens)])
        it = rng.choice(J, size=min(d, J), replace=False)
        it = it if i % 3 == 0 else np.sort(it)
        idx.extend(it.tolist()); rows.append(len(idx))
    nnz = len(idx)
    c = (-rng.random(nnz) * rng.choice([1.0, 3.0])).astype(np.float32)
    a = (0.5 + rng.random(nnz * m)).astype(np.float32)
    col = np.zeros(J * m)
    np.add.at(col, (np.repeat(np.array(idx, dtype=np.int64), m) * m + np.tile(np.arange(m), nnz)), a)
    b = (0.1 * col + 0.01).astype(np.float32)
    return dict(I=I, J=J, m=m, row_ptr=np.array(rows, dtype=np.int64), item_idx=np.array(idx, dtype=np.int32), c=c, a=a, b=b)


def read_projection_cases():
    cases = []
    with open(os.path.join(GOLDEN, "projection_cases.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            kind, params, v, x = [s.strip() for s in line.split("|")]
            cases.append((kind, [float(t) for t in params.split()], np.array(v.split(), dtype=np.float64),
                          np.array(x.split(), dtype=np.float64)))
    return cases


def read_worked_examples():
    cases, cur = [], None
    with open(os.path.join(GOLDEN, "worked_example_grad.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            if line == "end":
                cases.append(cur); cur = None; continue
            key, val = [s.strip() for s in line.split(":", 1)]
            if key == "case":
                cur = {"case": val}
            elif key in ("I", "J", "m"):
                cur[key] = int(val)
            elif key in ("row_ptr", "item_idx"):
                cur[key] = np.array(val.split(), dtype=np.int64)
            elif key in ("gamma", "g", "obj", "reg", "r_inf", "r_2"):
                cur[key] = float(val)
            else:
                cur[key] = np.array(val.split(), dtype=np.float64)
    return cases


def random_problem(rng, I, J, m=1, deg=(1, 4), tight=0.5, c_scale=1.0):
    """Small random matching instance as plain numpy arrays (tests only)."""
    rows, idx = [0], []
    for _ in range(I):
        d = int(rng.integers(deg[0], min(deg[1], J) + 1))
        idx.extend(sorted(rng.choice(J, size=d, replace=False).tolist()))
        rows.append(len(idx))
    nnz = len(idx)
    c = (-c_scale * rng.random(nnz)).astype(np.float32)
    a = (0.5 + rng.random(nnz * m)).astype(np.float32)
    col = np.zeros(J * m)
    for p, j in enumerate(idx):
        for k in range(m):
            col[j * m + k] += a[p * m + k]
    b = (tight * col / max(1.0, np.mean(np.diff(rows))) + 0.05).astype(np.float32)
    return dict(I=I, J=J, m=m, row_ptr=np.array(rows, dtype=np.int64), item_idx=np.array(idx, dtype=np.int32),
                c=c, a=a, b=b)
