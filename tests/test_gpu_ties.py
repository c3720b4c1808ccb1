"""`-m gpu`: the hand-worked projections of tests/golden/projection_cases.txt and EXACTLY tied rows through the CUDA path.

The golden file pins the oracle (tests/test_oracle_projection.py); here every one of its lines is also sent through the
library as a one-row-per-user problem, and the x the kernel writes is compared with the hand-worked numbers themselves, not
only with the oracle.  The construction: one user per case, items 0..n-1, a = 1, lambda = 0, c = -gamma v with gamma a power
of two, so that the kernel's candidate -(c + a lambda)/gamma (Eq. 3) is exactly fp32(v); b is large and plays no part.

Exact ties are what random data never produces: an all-equal row (every entry is the maximum, the threshold cuts all of them
alike -- SURVEY 8(c) pins "(0.6,0.6,0.6) -> (1/3,1/3,1/3)", "(1,1) -> (1/2,1/2)"), and two equal maxima far above the rest,
which is the streaming kernel's "the second largest equals the largest: not a vertex" branch, with the two maxima in one lane's
four slots, in neighbouring lanes and in different chunks of a row.  Both gradient kernels, every lane-group width, m = 1 and 2.
Checked: x against the closed form, tied inputs get bit-identical outputs, and full parity (x, grad g, scalars) with the oracle.
"""
import numpy as np
import pytest
import torch

from conftest import read_projection_cases

pytestmark = pytest.mark.gpu

if torch.cuda.is_available():
    from gpu_util import assert_grad_parity, both, gpu_grad

# (kernel, lanes per row); 0 = the library's choice
PLANS = [("streaming", 0), ("streaming", 4), ("streaming", 8), ("streaming", 16), ("streaming", 32),
         ("direct", 8), ("direct", 16), ("direct", 32)]


def _one_row_per_case(rows, gamma, m, J):
    """rows: list of fp64 vectors v.  User i gets items 0..len(v_i)-1 with c = -gamma v_i (fp32) and a = 1."""
    ptr = np.concatenate([[0], np.cumsum([len(v) for v in rows])]).astype(np.int64)
    idx = np.concatenate([np.arange(len(v)) for v in rows]).astype(np.int32)
    c = (-gamma * np.concatenate(rows)).astype(np.float32)
    a = np.ones(len(idx) * m, dtype=np.float32)
    return dict(I=len(rows), J=J, m=m, row_ptr=ptr, item_idx=idx, c=c, a=a, b=np.full(J * m, 1e3, dtype=np.float32))


def _run(rows, kind, p0, p1, gamma, m, kernel, lanes):
    J = max(max(len(v) for v in rows), 2)
    d = _one_row_per_case(rows, gamma, m, J)
    po, pg = both(d, kind, p0, p1, direct_kernel=(kernel == "direct"), group_lanes=lanes)
    if kind != "box":
        assert pg.info().streaming == (1 if kernel == "streaming" else 0)
    lam = np.zeros(J * m)
    assert_grad_parity(po, pg, lam, gamma, tag=f"{kind}/{kernel}/G={lanes}/m={m}")
    _, _, x = gpu_grad(pg, lam, gamma)
    pg.destroy()
    return np.split(x.astype(np.float64), d["row_ptr"][1:-1])


def _golden_groups():
    groups = {}
    for kind, params, v, x in read_projection_cases():
        groups.setdefault((kind, tuple(params)), []).append((v, x))
    return sorted(groups.items())


@pytest.mark.parametrize("kernel,lanes", PLANS, ids=[f"{k}-G{g}" for k, g in PLANS])
@pytest.mark.parametrize("group", _golden_groups(), ids=lambda g: f"{g[0][0]}-{'-'.join(str(p) for p in g[0][1])}")
def test_hand_worked_projections_through_the_cuda_path(group, kernel, lanes):
    (kind, params), cases = group
    if kind == "box" and (kernel, lanes) != ("streaming", 0):
        pytest.skip("the box projection has a single element-wise kernel")
    p0, p1 = (params + (0.0,))[:2]
    for gamma in (1.0, 0.25):
        got = _run([v for v, _ in cases], kind, p0, p1, gamma, 1, kernel, lanes)
        for (v, want), x in zip(cases, got):
            # inputs reach the kernel as fp32(v): the hand-worked x moves by at most a few ulp of fp32
            assert np.abs(x - want).max() <= 2e-6, f"{kind} {params} v={v}: x={x} hand-worked {want}"


def _tied_rows():
    """(row, closed-form x for the unit simplex inequality set, closed-form x for the equality set).  All values are fp32
    numbers, so the ties survive the conversion exactly."""
    rows = []
    for n in (2, 3, 33, 65, 129):
        v = np.full(n, 0.75)                                        # n * 0.75 > 1: the budget binds, theta = 0.75 - 1/n
        rows.append((v, np.full(n, 1.0 / n), np.full(n, 1.0 / n)))
    rows.append((np.full(5, 0.125), np.full(5, 0.125), np.full(5, 0.2)))      # interior for <=, lifted onto the face for =
    rows.append((np.full(4, -0.5), np.zeros(4), np.full(4, 0.25)))            # all-equal and negative: dead row for <=
    for n, (i, j) in ((8, (0, 1)), (8, (2, 3)), (12, (3, 4)), (40, (0, 39)), (70, (5, 64)), (140, (1, 130))):
        v = -1.0 - np.arange(n) * 0.0078125                         # distinct, far below the two maxima
        v[i] = v[j] = 1.5                                           # theta = (1.5 + 1.5 - 1) / 2 = 1: the rest stay out
        want = np.zeros(n); want[i] = want[j] = 0.5
        rows.append((v, want, want.copy()))
    v = np.array([0.875, 0.875, 0.875, 0.25, 0.875])                # four-way tie around one lower entry: theta = 0.625
    want = np.array([0.25, 0.25, 0.25, 0.0, 0.25])
    rows.append((v, want, want.copy()))
    return rows


@pytest.mark.parametrize("kernel,lanes", PLANS, ids=[f"{k}-G{g}" for k, g in PLANS])
@pytest.mark.parametrize("m", [1, 2])
@pytest.mark.parametrize("kind", ["simplex", "simplex_eq", "boxcut_wide"])
def test_exactly_tied_rows(kind, m, kernel, lanes):
    rows = _tied_rows()
    k, p0, p1 = ("boxcut", 1.0, 1.0) if kind == "boxcut_wide" else (kind, 1.0, 0.0)      # ub >= z: the simplex itself (R10)
    for gamma in (1.0, 0.125):
        got = _run([r[0] for r in rows], k, p0, p1, gamma, m, kernel, lanes)
        for (v, want_le, want_eq), x in zip(rows, got):
            want = want_eq if kind == "simplex_eq" else want_le
            assert np.abs(x - want).max() <= 2e-6, f"{kind}/m={m}/gamma={gamma} v={v[:6]}..: x={x[:6]} closed form {want[:6]}"
            for val in np.unique(v):                                # tied inputs -> bit-identical outputs
                tied = x[v == val]
                assert (tied == tied[0]).all(), f"{kind}/m={m}: tied entries of v={val} got different x: {tied}"


@pytest.mark.parametrize("kernel,lanes", PLANS, ids=[f"{k}-G{g}" for k, g in PLANS])
def test_tied_rows_under_a_genuine_box_cut(kernel, lanes):
    """Box-cut with ub < z: an all-equal row is cut at min(ub, z/n) whichever binds; two tied maxima are both capped."""
    ub, z = 0.25, 1.0
    rows = []
    for n in (2, 3, 33, 129):
        rows.append((np.full(n, 0.75), np.full(n, min(ub, z / n))))
    v = -1.0 - np.arange(40) * 0.0078125
    v[[0, 39]] = 1.5
    want = np.zeros(40); want[[0, 39]] = ub
    rows.append((v, want))
    # six tied entries that cannot all sit at the cap (6 * 0.25 > z): sum of min(max(v - t, 0), ub) = 1 with the 0.125s out
    # is 6 (0.5 - t) = 1, so t = 1/3 and x = 1/6 < ub on the six
    v = np.array([0.5, 0.5, 0.5, 0.5, 0.5, 0.5, 0.125, 0.125])
    rows.append((v, np.array([1 / 6] * 6 + [0.0, 0.0])))
    for gamma in (1.0, 0.125):
        got = _run([r[0] for r in rows], "boxcut", ub, z, gamma, 1, kernel, lanes)
        for (v, want), x in zip(rows, got):
            assert np.abs(x - want).max() <= 2e-6, f"boxcut gamma={gamma} v={v[:6]}..: x={x[:6]} closed form {want[:6]}"
            for val in np.unique(v):
                tied = x[v == val]
                assert (tied == tied[0]).all()
