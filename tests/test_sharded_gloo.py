"""Host logic of the user-sharded path (paper_2606_07777_b200/sharded.py) on CPU: two processes over gloo.  The CUDA handle is
replaced by a stand-in that holds integer arrays, so what is checked is the exchange pattern: global extents by SUM / MAX, the
fixed-point column sums and the per-evaluation accumulators by int64 SUM, identical results on both ranks."""
import json
import os
import socket
import subprocess
import sys
import textwrap

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, {root!r})
    import torch
    import torch.distributed as dist
    from paper_2606_07777_b200.binding import ShardExtents
    from paper_2606_07777_b200.sharded import ShardedProblem
    dist.init_process_group(backend="gloo")
    rank = dist.get_rank()

    class FakeLocal:                      # the calls ShardedProblem makes on a Problem, on CPU tensors
        J, m = 3, 2
        acc_words = 3 * 2 + 3
        def __init__(self):
            self.acc = torch.arange(self.acc_words, dtype=torch.int64) * (10 ** rank) + rank
            self.constants = None
        def shard_extents(self):
            return ShardExtents(100 + rank, 1000 * (rank + 1), 1.5 + rank, 0.25 * (2 - rank))
        def column_stats(self, g, out):
            assert (g.I, g.nnz, g.max_abs_a, g.max_abs_c) == (201, 3000, 2.5, 0.5)
            out.copy_(torch.arange(out.numel(), dtype=torch.int64) + 7 * rank)
            return out
        def set_shard_constants(self, g, summed):
            self.constants = summed.clone()
            self.agreed = getattr(self, "agreed", 0) + 1
        def set_c(self, c_new, stream=None):
            self.c = c_new
        def set_reduce_hook(self, fn):
            self.hook = fn
        def export_accumulators(self, out, clear=True):
            out.copy_(self.acc)
        def import_accumulators(self, acc, accumulate=False):
            self.acc = acc.clone()
        def destroy(self):
            pass

    loc = FakeLocal()
    sp = ShardedProblem(loc, dist=dist, device=torch.device("cpu"))
    loc.hook(0, loc.acc_words, 0, 1e-3, 0)            # what the library does between the gradient kernel and the epilogue
    acc = loc.acc.tolist()
    sp.set_c("c2")                                    # a new c: the constants must be agreed on again, on every rank
    print(json.dumps({{"rank": rank, "constants": loc.constants.tolist(), "acc": acc, "calls": sp.allreduce_calls,
                      "agreed": loc.agreed, "c": loc.c}}), flush=True)
    dist.destroy_process_group()
""")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_shards_exchange_integers_and_end_identical(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=180)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    n = 2 * 6 + 1
    want_const = (2 * np.arange(n) + 7).tolist()
    want_acc = (np.arange(9) * 1 + 0 + np.arange(9) * 10 + 1).tolist()
    for o in outs:
        assert o["constants"] == want_const and o["acc"] == want_acc and o["calls"] == 1
        assert o["agreed"] == 2 and o["c"] == "c2"        # ShardedProblem.set_c: local set_c, then the a0 exchange once more


def test_split_users_balances_nonzeros():
    from paper_2606_07777_b200.sharded import split_users
    rng = np.random.default_rng(0)
    deg = rng.integers(0, 400, size=5000)
    rp = np.concatenate([[0], np.cumsum(deg)]).astype(np.int64)
    for world in (1, 2, 3, 8):
        cuts = split_users(rp, world)
        assert cuts[0] == 0 and cuts[-1] == 5000 and all(a <= b for a, b in zip(cuts, cuts[1:]))
        per = [rp[b] - rp[a] for a, b in zip(cuts, cuts[1:])]
        assert max(per) - min(per) <= 40 * 400
        assert all(c % 2 == 0 and rp[c] % 4 == 0 for c in cuts[1:-1])        # 16-byte aligned slices
        raw = split_users(rp, world, align=False)
        assert max(rp[b] - rp[a] for a, b in zip(raw, raw[1:])) - min(rp[b] - rp[a] for a, b in zip(raw, raw[1:])) <= 2 * 400
