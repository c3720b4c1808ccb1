"""The input generator: determinism, chunk independence, the stated shapes/distributions, no method
arithmetic needed.  CPU only (scaled-down user counts; recipes per DESIGN.md "Input recipe")."""
import numpy as np
import torch

import synth


def _rows_ok(d, J):
    rp, idx = d["row_ptr"], d["item_idx"]
    assert rp[0] == 0 and rp[-1] == idx.size and (np.diff(rp) >= 0).all()
    assert idx.min() >= 0 and idx.max() < J
    same_row = np.repeat(np.arange(rp.size - 1), np.diff(rp))
    inc = np.diff(idx) > 0
    assert inc[same_row[1:] == same_row[:-1]].all()        # strictly ascending => distinct within a row


def test_cfg1_verbatim_shape_and_determinism():
    a, b = synth.generate("cfg1"), synth.generate("cfg1")
    d = a.numpy()
    assert a.I == 1000 and a.J == 50 and a.nnz == 10_000 and a.short_rows == 0
    assert (np.diff(d["row_ptr"]) == 10).all()
    _rows_ok(d, 50)
    for k in ("row_ptr", "item_idx", "c", "a", "b"):
        assert np.array_equal(d[k], b.numpy()[k])
    assert d["c"].dtype == np.float32 and d["item_idx"].dtype == np.int32 and d["row_ptr"].dtype == np.int64
    assert (d["c"] <= 0).all() and (d["c"] > -1).all() and (d["a"] >= 0.5).all() and (d["a"] <= 1.5).all()
    col = np.zeros(50); np.add.at(col, d["item_idx"], d["a"].astype(np.float64))
    np.testing.assert_allclose(d["b"], 0.2 * col, rtol=1e-6)


def test_chunking_does_not_change_the_instance():
    cfg = synth.get_config("cfg3", I=3000)
    x, y = synth.generate(cfg, chunk_users=3000).numpy(), synth.generate(cfg, chunk_users=700).numpy()
    for k in ("row_ptr", "item_idx", "c", "a"):
        assert np.array_equal(x[k], y[k]), k
    np.testing.assert_allclose(x["b"], y["b"], rtol=1e-6)


def test_degree_distributions():
    d2 = synth.generate(synth.get_config("cfg2", I=30000)).numpy()
    deg = np.diff(d2["row_ptr"])
    assert deg.min() == 5 and deg.max() == 35 and abs(deg.mean() - 20) < 0.3
    assert np.bincount(deg)[5:36].min() > 0.7 * 30000 / 31
    d3 = synth.generate(synth.get_config("cfg3", I=30000)).numpy()
    deg = np.diff(d3["row_ptr"])
    assert abs(deg.mean() - 50) < 0.3 and abs(deg.var() - 50) < 3 and deg.min() >= 1 and deg.max() <= 400
    _rows_ok(d3, 10_000)
    np.testing.assert_array_equal(d3["a"], -d3["c"])                       # spend proportional to value
    lc = np.log(-d3["c"].astype(np.float64))
    assert abs(lc.mean()) < 0.02 and abs(lc.std() - 1) < 0.02              # LogNormal(0,1)


def test_zipf_popularity_is_skewed_and_permuted():
    inst = synth.generate(synth.get_config("cfg5", I=20000))
    cnt = np.sort(np.bincount(inst.numpy()["item_idx"], minlength=20000))[::-1]
    # Zipf(1.0) over 20000 items: p_1 = 1/H ~ 0.0954; with ~30 distinct draws the top item is in most rows
    assert cnt[0] > 0.8 * 20000 and cnt[0] / max(cnt[100], 1) > 20
    hot = np.argsort(np.bincount(inst.numpy()["item_idx"], minlength=20000))[::-1][:8]
    assert not np.array_equal(np.sort(hot), np.arange(8))                   # hot ids are scattered


def test_two_families_layout():
    inst = synth.generate(synth.get_config("cfg4", I=2000))
    d = inst.numpy()
    a = d["a"].reshape(-1, 2)
    assert inst.m == 2 and (a[:, 1] == 1).all() and (a[:, 0] >= 0.5).all()
    cnt = np.bincount(d["item_idx"], minlength=5000)
    col = np.zeros(5000); np.add.at(col, d["item_idx"], a[:, 0].astype(np.float64))
    b = d["b"].reshape(-1, 2)
    np.testing.assert_allclose(b[:, 0], 0.3 * col, rtol=1e-6)
    np.testing.assert_allclose(b[:, 1], 0.2 * cnt, rtol=1e-6)
    deg = np.diff(d["row_ptr"])
    assert deg.min() >= 50 and deg.max() <= 150


def test_tight_companion_rhs_is_the_greedy_load_rule():
    inst = synth.generate("cfg1-tight")
    d = inst.numpy()
    load = np.zeros(50)
    for i in range(1000):
        lo, hi = d["row_ptr"][i], d["row_ptr"][i + 1]
        p = lo + int(np.argmax(d["a"][lo:hi]))
        load[d["item_idx"][p]] += float(d["a"][p])
    rho = d["b"] / (load + 1e-6)
    assert (rho >= 0.5 - 1e-6).all() and (rho <= 1 + 1e-6).all() and rho.std() > 0.05
    base = synth.generate("cfg1").numpy()
    for k in ("row_ptr", "item_idx", "c", "a"):
        assert np.array_equal(d[k], base[k])


def test_probe_and_perturbation_are_seeded():
    inst = synth.generate("cfg1")
    l0, l1 = synth.probe_lambda(inst, 0, 0.5), synth.probe_lambda(inst, 1, 0.5)
    assert l0.dtype == torch.float64 and l0.min() >= 0 and l0.max() <= 0.5 and not torch.equal(l0, l1)
    assert torch.equal(l0, synth.probe_lambda(inst, 0, 0.5))
    c2 = synth.perturb_c(inst)
    rel = ((c2 - inst.c) / inst.c).double()
    assert abs(rel.std().item() - 0.01) < 1e-3 and abs(rel.mean().item()) < 1e-3
