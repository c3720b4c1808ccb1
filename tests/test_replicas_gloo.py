"""N > 1 host logic on CPU: two processes over gloo (the GPU box has one GPU; the path is replicas-only, DESIGN.md
section 6).  Checks the barrier, the max-over-ranks timing rule and the aggregate the bench line reports."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys, time
    sys.path.insert(0, {root!r})
    from paper_2606_07777_b200.replicas import Replicas
    r = Replicas(backend="gloo")
    assert r.world == 2 and r.rank in (0, 1)
    r.barrier()
    mine = 0.25 if r.rank == 0 else 0.5            # rank 1 is the slow replica
    worst = r.max_over_ranks(mine)
    agg = r.aggregate_throughput(1000.0, mine)
    r.barrier()
    print(json.dumps({{"rank": r.rank, "worst": worst, "agg": agg}}), flush=True)
    r.close()
""")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_replicas_report_the_slowest_time(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    import json
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=120)
        assert p.returncode == 0, err[-2000:]
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["worst"] == 0.5                   # every rank sees the max, not its own time
        assert o["agg"] == 2 * 1000.0 / 0.5        # all replicas' units over the slowest replica's time


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    from paper_2606_07777_b200.replicas import Replicas
    env = {k: os.environ.pop(k) for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK") if k in os.environ}
    try:
        r = Replicas(backend="gloo")
        assert r.world == 1 and r.dist is None
        assert r.max_over_ranks(0.125) == 0.125 and r.aggregate_throughput(10.0, 0.5) == 20.0
        r.barrier(); r.close()
    finally:
        os.environ.update(env)
