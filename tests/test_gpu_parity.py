"""`-m gpu` parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by element on
the same seeded inputs.  Tolerances (BASELINE.json north_star): per-evaluation grad g relative L2 <= 1e-5,
x element-wise absolute <= 1e-5, dual objective relative <= 1e-5; integer work bit-exact."""
import numpy as np
import pytest
import torch

import oracle
import synth
from conftest import ragged_problem, random_problem, read_worked_examples

pytestmark = pytest.mark.gpu

if torch.cuda.is_available():
    import paper_2606_07777_b200 as pkg
    from gpu_util import (assert_grad_parity, assert_trajectory_parity, both, from_instance, gpu_grad, gpu_solve, rel_l2)


@pytest.mark.parametrize("ex", read_worked_examples(), ids=lambda e: e["case"])
def test_hand_worked_examples(ex):
    po, pg = both(ex)
    sc, grad, x = gpu_grad(pg, ex["lambda"], ex["gamma"])
    np.testing.assert_allclose(x, ex["x"], atol=1e-6)
    np.testing.assert_allclose(grad, ex["grad"], atol=1e-6)
    for key in ("g", "obj", "reg", "r_inf", "r_2"):
        assert abs(getattr(sc, key) - ex[key]) < 1e-6, key


_ragged = ragged_problem          # moved to conftest.py: the CPU-side sensitivity test builds the same instances


CASES = [
    # (tag, I, J, m, row lengths pattern)
    ("short8", 3000, 40, 1, [1, 2, 7, 8, 3, 0, 5]),
    ("mid16", 3000, 100, 1, [9, 16, 17, 31, 12, 0, 48, 20]),
    ("warp32", 2000, 300, 1, [33, 64, 65, 100, 128, 40, 159, 160]),
    ("long_rows", 300, 700, 1, [161, 200, 400, 650, 5, 32]),       # beyond the register budget -> warp path
    ("two_fam", 2000, 120, 2, [50, 99, 100, 150, 7, 0]),
    ("three_fam", 800, 60, 3, [5, 33, 40, 1]),
    ("four_fam", 500, 50, 4, [10, 45]),
    ("one_row", 1, 5, 1, [3]),
    ("all_empty", 7, 3, 1, [0]),
]


@pytest.mark.parametrize("tag,I,J,m,lens", CASES, ids=[c[0] for c in CASES])
@pytest.mark.parametrize("kind,p0,p1", [("simplex", 1.0, 0.0), ("simplex", 0.5, 0.0), ("simplex_eq", 1.0, 0.0),
                                        ("boxcut", 0.3, 1.0), ("boxcut", 1.0, 1.0), ("box", 0.0, 0.4), ("box", -0.2, 1.0)])
@pytest.mark.parametrize("kernel", ["streaming", "direct"])
def test_grad_parity_small(tag, I, J, m, lens, kind, p0, p1, kernel):
    """Both gradient kernels (TMA-staged k_grad_tma, direct-load k_grad) on ragged rows, every projection."""
    if kernel == "direct" and kind == "box":
        pytest.skip("the box projection has a single element-wise kernel")
    rng = np.random.default_rng(sum(map(ord, tag + kind)) * 131 + int(p0 * 1000))
    d = _ragged(rng, I, J, m, lens)
    po, pg = both(d, kind, p0, p1, direct_kernel=(kernel == "direct"))
    if kind != "box" and len(d["item_idx"]) > 0:
        assert pg.info().streaming == (1 if kernel == "streaming" else 0)
    for gamma in (1.0, 1e-1, 1e-2, 1e-3):
        for lam_scale in (0.0, 0.3):
            lam = rng.random(J * m) * lam_scale
            assert_grad_parity(po, pg, lam, gamma, tag=f"{tag}/{kind}/g={gamma}/l={lam_scale}")
    lam = rng.normal(size=J * m) * 0.2                     # g is defined for negative lambda too
    assert_grad_parity(po, pg, lam, 0.05, tag=f"{tag}/{kind}/neg")
    pg.destroy()


@pytest.mark.parametrize("G", [8, 16, 32])
def test_group_width_does_not_change_results(G):
    rng = np.random.default_rng(5)
    d = _ragged(rng, 4000, 200, 1, [3, 10, 20, 35, 70, 0, 150, 90])
    po, pg = both(d, group_lanes=G)
    assert pg.info().group_lanes == G
    lam = rng.random(200) * 0.4
    assert_grad_parity(po, pg, lam, 1e-2, tag=f"G={G}")
    assert_grad_parity(po, pg, lam, 1e-3, tag=f"G={G}")


@pytest.mark.parametrize("G", [1, 2, 4, 8, 16, 32])
@pytest.mark.parametrize("m", [1, 2])
def test_clustered_near_ties_take_the_compacted_candidate_path(G, m):
    """Rows whose k largest values are near-tied AND adjacent in the row (so several candidates sit in one lane's four
    slots), k = 1..40: fewer candidates than lanes (one per lane after compaction), up to 2G (two per lane) and beyond
    (the row falls through to the slow path).  Every row is fractional at gamma = 1e-2; at 1e-4 most are vertices."""
    rng = np.random.default_rng(100 * G + m)
    I, J = 1500, 400
    rows, idx, cs = [0], [], []
    for i in range(I):
        d = int(rng.integers(1, 120))
        it = np.sort(rng.choice(J, size=d, replace=False))
        c = -0.5 * rng.random(d)
        k = min(d, int(rng.integers(1, 41)))
        off = int(rng.integers(0, d - k + 1))
        c[off:off + k] = -1.0 - 2e-3 * rng.random(k)          # the cluster: within 2e-3 of each other, well above the rest
        idx.extend(it.tolist()); cs.extend(c.tolist()); rows.append(len(idx))
    nnz = len(idx)
    d_ = dict(I=I, J=J, m=m, row_ptr=np.array(rows, dtype=np.int64), item_idx=np.array(idx, dtype=np.int32),
              c=np.array(cs, dtype=np.float32), a=(0.5 + rng.random(nnz * m)).astype(np.float32),
              b=np.full(J * m, 0.5, dtype=np.float32))
    for kind, p0, p1 in (("simplex", 1.0, 0.0), ("simplex_eq", 1.0, 0.0), ("boxcut", 1.0, 1.0)):
        po, pg = both(d_, kind, p0, p1, group_lanes=G)
        assert pg.info().streaming == 1 and pg.info().group_lanes == G
        for gamma in (1e-2, 1e-3, 1e-4):
            assert_grad_parity(po, pg, np.zeros(J * m), gamma, tag=f"ties G={G} m={m} {kind} gamma={gamma}")
            assert_grad_parity(po, pg, 1e-4 * rng.random(J * m), gamma, tag=f"ties G={G} m={m} {kind} gamma={gamma} lam")
        pg.destroy()


def test_cfg1_verbatim_trajectory():
    """BASELINE config 1 as stated: 200 AGD iterations from lambda = 0 at gamma = 1e-2 (slack: lambda stays 0)."""
    inst = synth.generate("cfg1")
    po, pg = from_instance(inst)
    worst, ex, ref, out = assert_trajectory_parity(po, pg, inst.cfg.gammas, inst.cfg.iters, tag="cfg1")
    assert np.all(out["lam"] == 0.0) and np.all(ref.lam == 0.0)


def test_cfg1_tight_trajectory():
    inst = synth.generate("cfg1-tight")
    po, pg = from_instance(inst)
    worst, ex, ref, out = assert_trajectory_parity(po, pg, inst.cfg.gammas, inst.cfg.iters, tag="cfg1-tight")
    assert (ref.lam > 0).sum() >= 5                         # the update is really exercised
    frac = ((ref.x > 1e-9) & (ref.x < 1 - 1e-9)).sum()
    assert frac > 20                                        # fractional projections too


# lanes per row the library picks for each config at its FULL size (what bench.py times; kernel names in profiles/): the
# scaled-down instances would get wider groups from the tile heuristic, so the tests ask for the benchmarked instantiation
FULL_SIZE_G = {"cfg2": 4, "cfg3": 8, "cfg4": 16, "cfg5": 4}   # asserted at full size by tests/test_gpu_fullsize.py


@pytest.mark.parametrize("name,I,iters", [("cfg2-tight", 60_000, 40), ("cfg3-tight", 30_000, 30), ("cfg4-tight", 8_000, 30),
                                          ("cfg5-tight", 40_000, None), ("cfg2", 60_000, 20), ("cfg3", 30_000, 20),
                                          ("cfg4", 8_000, 20), ("cfg5", 40_000, None)])
def test_scaled_config_trajectories(name, I, iters):
    """Every BASELINE config (and its tight companion) at a user count the oracle finishes in seconds; the
    recipe (J, degrees, values, projection, gamma schedule) is the config's own; the kernel instantiation (lanes per row)
    is the one the full-size plan runs."""
    cfg = synth.get_config(name, I=I)
    inst = synth.generate(cfg)
    po, pg = from_instance(inst, group_lanes=FULL_SIZE_G[name[:4]])
    assert pg.info().group_lanes == FULL_SIZE_G[name[:4]] and pg.info().streaming == 1
    its = [iters] * len(cfg.gammas) if iters else [15] * len(cfg.gammas)
    assert_trajectory_parity(po, pg, cfg.gammas, its, tag=name)
    for which in range(2):                                   # same-lambda probes with a busy lambda
        lam = synth.probe_lambda(inst, which, 0.5 if "3" not in name else 0.05).numpy()
        assert_grad_parity(po, pg, lam, cfg.gammas[-1], tag=f"{name}/probe{which}")


def test_plain_ascent_option_and_warm_start():
    inst = synth.generate(synth.get_config("cfg2-tight", I=20_000))
    po, pg = from_instance(inst, momentum=False)
    assert_trajectory_parity(po, pg, [1e-2, 1e-3], [15, 15], momentum=False, tag="beta0")
    po2, pg2 = from_instance(inst)
    lam0 = synth.probe_lambda(inst, 3, 0.2).numpy()
    assert_trajectory_parity(po2, pg2, [1e-2], [10], lam0=lam0, tag="warm")


def test_run_to_run_and_geometry_bit_reproducible():
    """Fixed-point accumulation: for a given kernel and lane-group width, grad g and x carry the same bits run
    to run, for any grid size and for either reduction strategy.  Across kernels (different summation trees
    inside a row) results agree to rounding."""
    inst = synth.generate(synth.get_config("cfg3-tight", I=30_000))
    lam = synth.probe_lambda(inst, 0, 0.05).numpy()
    ref = {}
    for direct in (False, True):
        outs = []
        for grid, red in ((0, pkg.RED_AUTO), (0, pkg.RED_AUTO), (37, pkg.RED_AUTO), (0, pkg.RED_GLOBAL), (53, pkg.RED_SMEM)):
            po, pg = from_instance(inst, grid_ctas=grid, reduction=red, direct_kernel=direct, group_lanes=16)
            sc, grad, x = gpu_grad(pg, lam, 1e-3)
            outs.append((sc.g, grad.copy(), x.copy()))
            pg.destroy()
        assert outs[0][0] == outs[1][0]                      # same launch twice: scalars too
        for o in outs[1:]:
            assert np.array_equal(outs[0][1], o[1]) and np.array_equal(outs[0][2], o[2])
        ref[direct] = outs[0]
    assert rel_l2(ref[True][1], ref[False][1]) < 1e-7 and np.abs(ref[True][2] - ref[False][2]).max() < 1e-6


def test_host_pointers_take_the_same_path():
    rng = np.random.default_rng(9)
    d = random_problem(rng, I=500, J=30, m=2, deg=(2, 9))
    po, pg = both(d)
    lam = rng.random(60) * 0.2
    sc_d, grad_d, x_d = gpu_grad(pg, lam, 0.05)
    pg_h = pkg.Problem.create(po.I, po.J, po.m, po.row_ptr, po.item_idx, po.c, po.a, po.b)   # numpy = host pointers
    grad_h, x_h, sc_h = np.empty(60), np.empty(po.nnz, dtype=np.float32), pkg.Scalars()
    pg_h.grad(np.ascontiguousarray(lam), 0.05, grad=grad_h, scalars=sc_h, x=x_h)
    assert np.array_equal(grad_h, grad_d) and np.array_equal(x_h, x_d) and sc_h.g == sc_d.g
    lam_h = np.zeros(60)
    pg_h.solve([0.05], [7], lam_h, x=x_h, scalars=sc_h, grad=grad_h)
    out = gpu_solve(pg, [0.05], [7], want_trace=False)
    assert np.array_equal(lam_h, out["lam"]) and np.array_equal(x_h, out["x"]) and sc_h.g == out["sc"].g


def test_set_c_and_drift_bound():
    """Config 5's perturbed re-solve in miniature: replace c in place, re-solve, ||dx||_2 <= ||dc||_2/gamma at
    fixed lambda (the closed form behind the paper's stability claim)."""
    inst = synth.generate(synth.get_config("cfg5-tight", I=20_000))
    po, pg = from_instance(inst)
    lam = synth.probe_lambda(inst, 1, 0.3).numpy()
    c2 = synth.perturb_c(inst)
    for gamma in (1e-1, 1e-2):
        _, _, x1 = gpu_grad(pg, lam, gamma)
        pg.set_c(c2.cuda())
        po2 = oracle.Problem(po.I, po.J, po.m, po.row_ptr, po.item_idx, c2.numpy(), po.a, po.b, po.proj_kind, po.p0, po.p1)
        assert_grad_parity(po2, pg, lam, gamma, tag="set_c")
        _, _, x2 = gpu_grad(pg, lam, gamma)
        dc = np.linalg.norm(c2.numpy().astype(np.float64) - inst.c.numpy().astype(np.float64))
        assert np.linalg.norm(x1.astype(np.float64) - x2.astype(np.float64)) <= dc / gamma * (1 + 1e-5)
        pg.set_c(inst.c.cuda())


def test_create_rejects_bad_input():
    rp = np.array([0, 2, 4], dtype=np.int64)
    good = dict(I=2, J=3, m=1, row_ptr=rp, item_idx=np.array([0, 2, 1, 2], dtype=np.int32),
                c=-np.ones(4, dtype=np.float32), a=np.ones(4, dtype=np.float32), b=np.ones(3, dtype=np.float32))

    def code(**over):
        d = dict(good); d.update(over)
        try:
            pkg.Problem.create(d["I"], d["J"], d["m"], d["row_ptr"], d["item_idx"], d["c"], d["a"], d["b"]).destroy()
            return 0
        except pkg.DualipError as e:
            return e.code
    assert code() == 0
    assert code(item_idx=np.array([0, 0, 1, 2], dtype=np.int32)) == -3            # duplicate (sorted row)
    assert code(item_idx=np.array([2, 0, 1, 1], dtype=np.int32)) == -3            # duplicate (unsorted row)
    assert code(item_idx=np.array([0, 3, 1, 2], dtype=np.int32)) == -2            # index out of range
    assert code(item_idx=np.array([0, -1, 1, 2], dtype=np.int32)) == -2
    assert code(row_ptr=np.array([0, 3, 2], dtype=np.int64)) == -2                # not monotone
    assert code(row_ptr=np.array([1, 2, 4], dtype=np.int64)) == -2                # row_ptr[0] != 0
    assert code(J=0) == -1 and code(m=5) == -1
    po, pg = both(good)
    with pytest.raises(pkg.DualipError):
        pg.grad(torch.zeros(3, dtype=torch.float64, device="cuda"), 0.0)           # gamma must be > 0


@pytest.mark.parametrize("J,m,long_lens,streaming", [(30_000, 1, [6_000, 28_000, 12_000], 1), (12_000, 2, [6_000, 11_000, 9_000], 1),
                                                    (80_000, 1, [6_000, 70_000, 30_000], 0)])
def test_long_rows_among_short_ones_cta_per_row(J, m, long_lens, streaming):
    """A cfg3-like instance (a thousand short rows) with a handful of rows of 6,000-70,000 nonzeros in the middle of it.  On the
    streaming plan the short rows stream (each long row is a tile of its own that the producer skips) and k_grad_long takes the
    long ones, staged in shared memory; on the direct-load plan (J too large for lambda in shared memory) rows beyond 4096 go
    to k_grad_long as well, the 70,000-long one recomputed per pass (it does not fit the staging buffer).  The two launches add
    into the same accumulators.  Per-evaluation parity incl. a dense gamma (every nonzero of a long row in the support), the
    count row, and a Jacobi trajectory."""
    rng = np.random.default_rng(900 + m + J)
    lens = [40] * 400 + long_lens[:1] + [25] * 300 + [long_lens[1], 3, long_lens[2]] + [50] * 500
    d = _ragged(rng, len(lens), J, m, lens)
    d["b"] = (d["b"] * 0.2).astype(np.float32)
    for kind in ("simplex", "simplex_eq"):
        po, pg = both(d, kind, 1.0, 0.0, jacobi=True)
        info = pg.info()
        assert (info.long_rows, info.streaming, info.max_row_len) == (3, streaming, max(long_lens)), (info.long_rows, info.long_row_threshold, info.streaming)
        for gamma, ls in ((1e-3, 0.0), (1e-2, 0.3), (5.0, 0.3)):
            assert_grad_parity(po, pg, rng.random(J * m) * ls, gamma, tag=f"mixed-long/{kind}/J={J}/g={gamma}")
        assert_trajectory_parity(po, pg, [1e-1, 1e-2], [12, 12], tag=f"mixed-long/{kind}/J={J}/solve", jacobi=True)
        pg.destroy()
    po, pg = both(d, count_M=300.0)
    assert_grad_parity(po, pg, np.concatenate([rng.random(J * m) * 0.2, [0.1]]), 1e-2, tag=f"mixed-long/count/J={J}")
    pg.destroy()


def test_long_unsorted_rows_are_validated_by_warps():
    """Rows of thousands of nonzeros in random order: the duplicate check is warp-cooperative (k_validate_unsorted), not one
    thread walking len^2 pairs; a duplicate at the two ends of a 6,000-long row is found, a clean instance is accepted."""
    rng = np.random.default_rng(3)
    J, lens = 9000, [6000, 3, 4500, 0, 6000]
    rows, idx = [0], []
    for d in lens:
        idx.extend(rng.permutation(J)[:d].tolist()); rows.append(len(idx))
    nnz = len(idx)
    arr = dict(I=len(lens), J=J, m=1, row_ptr=np.array(rows, dtype=np.int64), item_idx=np.array(idx, dtype=np.int32),
               c=-rng.random(nnz).astype(np.float32), a=np.ones(nnz, dtype=np.float32), b=np.ones(J, dtype=np.float32))
    po, pg = both(arr)
    assert_grad_parity(po, pg, np.zeros(J), 1e-2, tag="long unsorted")
    pg.destroy()
    bad = arr["item_idx"].copy()
    bad[rows[5] - 1] = bad[rows[4]]                                  # last element of the last row := its first
    with pytest.raises(pkg.DualipError) as e:
        pkg.Problem.create(arr["I"], J, 1, arr["row_ptr"], bad, arr["c"], arr["a"], arr["b"])
    assert e.value.code == -3


def test_graph_replay_is_the_same_iteration():
    """use_graph: the stage loop replays a CUDA graph of chained one-launch iterations (beta_t and the trace row come
    from the device-side iteration state); lambda_T, x, the trace and the scalars carry the same bits as direct
    launches, across stages (momentum restart) and for iteration counts that are not a multiple of the graph length."""
    inst = synth.generate(synth.get_config("cfg2-tight", I=20_000))
    outs = []
    for graph in (False, True):
        po, pg = from_instance(inst, use_graph=graph)
        n0 = pg.info().launches
        out = gpu_solve(pg, [1e-2, 1e-3], [47, 63])
        assert pg.info().launches - n0 == 47 + 63 + 1        # one launch per iteration + the final evaluation
        outs.append(out)
        if graph:
            assert_trajectory_parity(po, pg, [1e-2, 1e-3], [47, 63], tag="graph")
        pg.destroy()
    a, b = outs
    assert np.array_equal(a["lam"], b["lam"]) and np.array_equal(a["x"], b["x"]) and a["sc"].g == b["sc"].g
    assert np.array_equal(a["tr_grad"], b["tr_grad"]) and np.array_equal(a["tr_lam"], b["tr_lam"]) and np.array_equal(a["tr_g"], b["tr_g"])


@pytest.mark.parametrize("tag,I,J,m,lens", [CASES[1], CASES[3], CASES[4], CASES[5], CASES[8]], ids=lambda c: c if isinstance(c, str) else None)
@pytest.mark.parametrize("kind,p0,p1", [("simplex", 1.0, 0.0), ("boxcut", 0.3, 1.0), ("box", 0.0, 0.4)])
def test_csc_reduction_parity_and_permutation(tag, I, J, m, lens, kind, p0, p1):
    """DUALIP_RED_CSC: the item-sorted permutation is bit-exact with a stable counting sort of item_idx, and the
    atomics-free reduction through it meets the same tolerances, evaluation and trajectory."""
    rng = np.random.default_rng(sum(map(ord, tag + kind)) * 17 + 3)
    d = _ragged(rng, I, J, m, lens)
    po, pg = both(d, kind, p0, p1, reduction=pkg.RED_CSC)
    assert pg.info().reduction == pkg.RED_CSC
    col_ptr, perm = np.empty(J + 1, dtype=np.int64), np.empty(po.nnz, dtype=np.int64)
    pg.get_csc(col_ptr, perm)
    assert np.array_equal(perm, np.argsort(po.item_idx, kind="stable"))
    assert np.array_equal(col_ptr, np.concatenate([[0], np.cumsum(np.bincount(po.item_idx, minlength=J))]))
    for gamma in (1e-1, 1e-3):
        lam = rng.random(J * m) * 0.3
        assert_grad_parity(po, pg, lam, gamma, tag=f"csc/{tag}/{kind}/g={gamma}")
    if po.nnz:
        assert_trajectory_parity(po, pg, [1e-1, 1e-2], [12, 9], tag=f"csc/{tag}/{kind}")
    with pytest.raises(pkg.DualipError):
        both(d, kind, p0, p1)[1].get_csc(col_ptr, perm)          # only the CSC mode has a permutation
    pg.destroy()


def test_csc_matches_atomic_modes_at_scale():
    """Config 3's recipe (Zipf columns: the longest column holds most users) at 200k users: CSC against the
    fixed-point modes, permutation against numpy, two launches bit-identical."""
    inst = synth.generate(synth.get_config("cfg3-tight", I=200_000))
    lam = synth.probe_lambda(inst, 0, 0.05).numpy()
    po, pg = from_instance(inst, reduction=pkg.RED_CSC)
    perm = np.empty(po.nnz, dtype=np.int64)
    pg.get_csc(None, perm)
    assert np.array_equal(perm, np.argsort(po.item_idx, kind="stable"))
    sc1, g1, x1 = gpu_grad(pg, lam, 1e-3)
    sc2, g2, x2 = gpu_grad(pg, lam, 1e-3)
    assert np.array_equal(g1, g2) and sc1.g == sc2.g
    assert_grad_parity(po, pg, lam, 1e-3, tag="csc/cfg3")
    po2, pg2 = from_instance(inst)
    sc3, g3, x3 = gpu_grad(pg2, lam, 1e-3)
    assert np.array_equal(x1, x3) and rel_l2(g1, g3) < 1e-9
    pg.destroy(); pg2.destroy()


# ---- Jacobi preconditioning (R18): the CUDA path never rescales the rows -- it takes the
# per-coordinate step eta' d_r^2 in the original variables -- while the oracle iterates on A' = D A, b' = D b literally.

@pytest.mark.parametrize("name,I,iters", [("cfg1-tight", None, 200), ("cfg2-tight", 60_000, 40), ("cfg3-tight", 30_000, 30),
                                          ("cfg4-tight", 8_000, 30), ("cfg5-tight", 40_000, None), ("cfg3", 30_000, 10)])
def test_jacobi_trajectories(name, I, iters):
    cfg = synth.get_config(name, I=I) if I else synth.get_config(name)
    inst = synth.generate(cfg)
    po, pg = from_instance(inst, jacobi=True, group_lanes=FULL_SIZE_G.get(name[:4], 0))
    info = pg.info()
    assert info.precondition == pkg.PRECOND_JACOBI and info.L_step == float(inst.m)
    its = [iters] * len(cfg.gammas) if iters else [15] * len(cfg.gammas)
    worst, ex, ref, out = assert_trajectory_parity(po, pg, cfg.gammas, its, tag=name + "/jacobi", jacobi=True)
    if name.endswith("tight"):
        assert (ref.lam > 0).sum() >= 5                     # the preconditioned update really moves lambda
    pg.destroy()


def test_jacobi_moves_where_the_scalar_step_stalls():
    """on the Zipf configs L is set by the hottest column, so the scalar step gamma/L barely moves
    lambda; the Jacobi step makes real progress on the same instance in the same number of iterations."""
    cfg = synth.get_config("cfg3-tight", I=30_000)
    inst = synth.generate(cfg)
    po, plain = from_instance(inst)
    _, jac = from_instance(inst, jacobi=True)
    its = [60]
    a = gpu_solve(plain, cfg.gammas[:1], its, want_trace=False, want_x=False)
    b = gpu_solve(jac, cfg.gammas[:1], its, want_trace=False, want_x=False)
    g0 = gpu_grad(plain, np.zeros(inst.J * inst.m), cfg.gammas[0], want_x=False)[0].g
    print(f"g(0)={g0:.6f} plain={a['sc'].g:.6f} jacobi={b['sc'].g:.6f}")
    assert a["sc"].g >= g0 - 1e-9 * abs(g0)                 # both ascend from g(0) ...
    assert b["sc"].g > a["sc"].g                            # ... the Jacobi step further (higher dual value)
    plain.destroy(); jac.destroy()


def test_jacobi_zero_rows_and_families():
    """Items nobody is eligible for (zero rows of A, D_rr = 1) and m = 2 (L' = 2), warm start in original units."""
    rng = np.random.default_rng(77)
    d = _ragged(rng, 1500, 90, 2, [6, 20, 33, 0, 12])
    d["item_idx"] = np.where(d["item_idx"] >= 80, d["item_idx"] - 40, d["item_idx"]).astype(np.int32)   # items 80.. unused
    # the remap may create duplicates inside a row: rebuild rows without them
    keep = np.ones(d["item_idx"].size, dtype=bool)
    for i in range(d["I"]):
        b, e = d["row_ptr"][i], d["row_ptr"][i + 1]
        _, first = np.unique(d["item_idx"][b:e], return_index=True)
        mask = np.zeros(e - b, dtype=bool); mask[first] = True
        keep[b:e] = mask
    lens = np.add.reduceat(keep, d["row_ptr"][:-1]) if d["I"] else np.array([], dtype=np.int64)
    lens[np.diff(d["row_ptr"]) == 0] = 0
    d["row_ptr"] = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    d["item_idx"], d["c"] = d["item_idx"][keep], d["c"][keep]
    d["a"] = d["a"].reshape(-1, 2)[keep].reshape(-1)
    d["b"] = (d["b"] * 0.5).astype(np.float32)
    po, pg = both(d, jacobi=True)
    assert pg.info().L_step == 2.0
    lam0 = rng.random(180) * 0.05
    assert_trajectory_parity(po, pg, [0.1, 0.01], [25, 25], lam0=lam0, tag="jacobi/zero-rows", jacobi=True)
    pg.destroy()


# ---- equality coupling rows (R19) --------------------------------------------------------------------

@pytest.mark.parametrize("jacobi", [False, True])
def test_equality_rows_trajectory(jacobi):
    """Every third coupling row is an equality: its dual goes negative where the row is slack, the others stay >= 0;
    per-iteration parity of grad, lambda and the |Ax-b| residuals with the oracle."""
    rng = np.random.default_rng(41)
    d = _ragged(rng, 2500, 60, 2, [4, 9, 17, 30, 0, 12])
    d["b"] = (d["b"] * 3.0).astype(np.float32)
    mask = (np.arange(120) % 3 == 0).astype(np.uint8)
    po, pg = both(d, jacobi=jacobi)
    pg.set_equality_rows(torch.from_numpy(mask).cuda())
    gam, its = [0.2, 0.02], [40, 40]
    ref = oracle.solve(po, gam, its, trace_grad=True, trace_lambda=True, jacobi=jacobi, is_eq=mask)
    out = gpu_solve(pg, gam, its)
    for n in range(80):
        assert rel_l2(out["tr_grad"][n], ref.trace_grad[n]) <= 1e-5, n
    scale = np.abs(ref.trace_lambda).max()
    assert np.abs(out["tr_lam"] - ref.trace_lambda).max() <= 1e-6 * scale + 1e-12
    gn = np.linalg.norm(ref.trace_grad, axis=1)
    assert np.all(np.abs(out["tr_rinf"] - ref.trace_rinf) <= 1e-5 * gn + 1e-12)
    assert np.all(np.abs(out["tr_r2"] - ref.trace_r2) <= 1e-5 * gn + 1e-12)
    assert np.abs(out["x"].astype(np.float64) - ref.x).max() <= 1e-5
    assert (ref.lam[mask == 1] < 0).any() and (ref.lam[mask == 0] >= 0).all()
    # host mask, and NULL restores the all-inequality loop
    pg.set_equality_rows(mask)
    out2 = gpu_solve(pg, gam, its, want_x=False)
    np.testing.assert_array_equal(out2["tr_lam"], out["tr_lam"])
    pg.set_equality_rows(None)
    ref0 = oracle.solve(po, gam, its, trace_lambda=True, jacobi=jacobi)
    out0 = gpu_solve(pg, gam, its, want_x=False)
    assert np.abs(out0["tr_lam"] - ref0.trace_lambda).max() <= 1e-6 * np.abs(ref0.trace_lambda).max() + 1e-12
    assert (out0["lam"] >= 0).all()
    pg.destroy()


def test_cfg5_continuation_then_perturbed_resolve_drift_per_gamma():
    """BASELINE config 5's whole workflow at a user count the oracle finishes in seconds: gamma 1e-1 -> 1e-4 (x0.1 per
    stage, warm-started lambda), x kept at every stage end; then c perturbed by N(0, (0.01|c|)^2) (R13), the same
    schedule re-solved from lambda = 0, and ||x - x_prev||_2 reported per gamma.  The CUDA path chains one
    dualip_solve per stage (lambda carried on the device); the oracle returns its stage-end x from ONE multi-stage
    solve.  Jacobi step, so that lambda really moves on this Zipf instance."""
    cfg = synth.get_config("cfg5-tight", I=40_000)
    inst = synth.generate(cfg)
    po, pg = from_instance(inst, jacobi=True)
    its = [15] * len(cfg.gammas)
    c2 = synth.perturb_c(inst)

    def gpu_run():
        lam = torch.zeros(inst.J * inst.m, dtype=torch.float64, device="cuda")
        xs = []
        for gam, it in zip(cfg.gammas, its):
            x = torch.empty(inst.nnz, dtype=torch.float32, device="cuda")
            pg.solve([gam], [it], lam, x=x)
            xs.append(x.cpu().numpy().astype(np.float64))
        return lam.cpu().numpy(), xs

    lam1, xs1 = gpu_run()
    ref1 = oracle.solve(po, cfg.gammas, its, jacobi=True, stage_x=True)
    pg.set_c(c2.cuda())
    lam2, xs2 = gpu_run()
    po2 = oracle.Problem(po.I, po.J, po.m, po.row_ptr, po.item_idx, c2.numpy(), po.a, po.b, po.proj_kind, po.p0, po.p1)
    ref2 = oracle.solve(po2, cfg.gammas, its, jacobi=True, stage_x=True)
    assert (ref1.lam > 0).sum() >= 5
    for s, gam in enumerate(cfg.gammas):
        assert np.abs(xs1[s] - ref1.stage_x[s]).max() <= 1e-5, f"stage {s} x"
        assert np.abs(xs2[s] - ref2.stage_x[s]).max() <= 1e-5, f"stage {s} x (perturbed)"
        drift_gpu = np.linalg.norm(xs1[s] - xs2[s])
        drift_ref = np.linalg.norm(ref1.stage_x[s] - ref2.stage_x[s])
        assert abs(drift_gpu - drift_ref) <= 1e-5 * np.sqrt(inst.nnz) + 1e-6 * drift_ref, f"gamma={gam}: {drift_gpu} vs {drift_ref}"
    assert np.abs(lam1 - ref1.lam).max() <= 1e-6 * np.abs(ref1.lam).max() + 1e-12
    assert np.abs(lam2 - ref2.lam).max() <= 1e-6 * np.abs(ref2.lam).max() + 1e-12
    pg.destroy()


def test_pipeline_geometry_does_not_change_a_bit():
    """Streaming kernel: 2 / 3 / 4 stages, small tiles, odd grids -- the round-robin deal of row-steps to warps changes,
    the 64-bit fixed-point sums do not: grad g, g and x are bit-identical (numerics)."""
    inst = synth.generate(synth.get_config("cfg3-tight", I=30_000))
    lam = synth.probe_lambda(inst, 1, 0.05).numpy()
    outs = []
    for stages, tile, grid in ((0, 0, 0), (2, 0, 0), (4, 0, 0), (3, 512, 0), (4, 1024, 29), (2, 256, 148)):
        po, pg = from_instance(inst, stages=stages, tile_units=tile, grid_ctas=grid)
        info = pg.info()
        assert info.streaming == 1 and (stages == 0 or info.stages == stages) and (tile == 0 or info.tile_units <= tile)
        sc, grad, x = gpu_grad(pg, lam, 1e-3)
        outs.append((sc.g, sc.obj, sc.reg, grad.copy(), x.copy()))
        pg.destroy()
    for o in outs[1:]:
        assert o[:3] == outs[0][:3] and np.array_equal(o[3], outs[0][3]) and np.array_equal(o[4], outs[0][4])
    assert_grad_parity(*from_instance(inst, stages=4, tile_units=256), lam, 1e-3, tag="small tiles")


@pytest.mark.parametrize("J,m", [(40_000, 1), (60_000, 1), (300_000, 1), (30_000, 2), (150_000, 2)])
def test_many_items_lambda_beyond_shared_memory(J, m):
    """J*m from just inside the streaming kernel's shared-memory budget (fp32 lambda only, small stages) to far beyond
    any on-chip copy of lambda (direct-load kernel, duals gathered through L2): same parity bar; the atomics-free CSC
    reduction (fp64 column sums) gives the same x bit for bit and the same gradient to fp32 product rounding."""
    rng = np.random.default_rng(J + m)
    I = 20_000
    d = _ragged(rng, I, J, m, [3, 12, 40, 0, 7, 90, 25])
    d["b"] = (d["b"] * 0.2).astype(np.float32)
    po, pg = both(d)
    info = pg.info()
    if 4 * J * m + 32 * 1024 + 256 <= 227 * 1024:
        assert info.streaming == 1
    else:
        assert info.streaming == 0
    lam = rng.random(J * m) * 0.3
    for gamma in (1e-1, 1e-3):
        assert_grad_parity(po, pg, lam, gamma, tag=f"J={J} m={m} g={gamma}")
    sc0, g0, x0 = gpu_grad(pg, lam, 1e-2)
    _, pc = both(d, reduction=pkg.RED_CSC)
    sc1, g1, x1 = gpu_grad(pc, lam, 1e-2)
    assert np.array_equal(x0, x1) and rel_l2(g1, g0) < 1e-7
    assert_trajectory_parity(po, pg, [1e-1, 1e-2], [12, 12], tag=f"J={J} m={m} solve", jacobi=False)
    _, pj = both(d, jacobi=True)
    assert_trajectory_parity(po, pj, [1e-1], [12], tag=f"J={J} m={m} jacobi", jacobi=True)
    for h in (pg, pc, pj):
        h.destroy()


def test_very_long_rows_and_no_users():
    """Rows longer than any stage (20,000 and 9,000 items: the streaming plan refuses, the direct-load kernel's whole-warp
    path takes them) next to short ones; and the degenerate I = 0 problem (grad g = -b, g = -lambda'b)."""
    rng = np.random.default_rng(123)
    J = 25_000
    d = _ragged(rng, 60, J, 1, [20_000, 5, 9_000, 33, 0, 400, 1])
    d["b"] = (d["b"] * 0.05).astype(np.float32)
    for kind, p0, p1 in (("simplex", 1.0, 0.0), ("boxcut", 0.001, 1.0), ("simplex_eq", 1.0, 0.0)):
        po, pg = both(d, kind, p0, p1)
        info = pg.info()
        assert info.max_row_len == 20_000
        if kind == "boxcut":            # genuine box-cut (ub < z): long rows stay on the direct-load kernel's whole-warp path
            assert info.streaming == 0 and info.long_rows == 0
        else:                           # simplex kinds: the long rows get a CTA each (k_grad_long), the rest streams
            assert info.streaming == 1 and info.long_rows >= 10 and 256 <= info.long_row_threshold < 9000
        for gamma, ls in ((1.0, 0.0), (1e-2, 0.5), (1e-4, 0.5)):
            assert_grad_parity(po, pg, rng.random(J) * ls, gamma, tag=f"long/{kind}/g={gamma}")
        pg.destroy()
    # the same rows on the direct-load plan: rows beyond 4096 nonzeros go to k_grad_long there as well
    po, pg = both(d, direct_kernel=True)
    assert pg.info().streaming == 0 and pg.info().long_row_threshold == 4096 and pg.info().long_rows >= 10
    assert_grad_parity(po, pg, rng.random(J) * 0.5, 1e-2, tag="long/direct")
    assert_trajectory_parity(po, pg, [1e-1, 1e-2], [10, 10], tag="long/direct/solve")
    pg.destroy()
    e = dict(I=0, J=4, m=1, row_ptr=np.zeros(1, dtype=np.int64), item_idx=np.zeros(0, dtype=np.int32),
             c=np.zeros(0, dtype=np.float32), a=np.zeros(0, dtype=np.float32), b=np.array([1, 2, 3, 4], dtype=np.float32))
    po, pg = both(e)
    lam = np.array([0.5, 0.0, 1.5, 2.0])
    sc, grad, x = gpu_grad(pg, lam, 0.1)
    assert np.array_equal(grad, -e["b"].astype(np.float64)) and sc.g == -(lam @ e["b"]) and x.size == 0 and sc.r_inf == 0.0
    out = gpu_solve(pg, [0.1], [5], lam0=lam, want_trace=False)
    assert np.all(out["lam"] <= lam) and np.all(out["lam"] >= 0)
    pg.destroy()
