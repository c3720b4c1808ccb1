#!/usr/bin/env python
"""bench.py -- measures the dual-ascent hot path on B200 (contract: see the task statement / DESIGN.md section 8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg3]

A "step" is ONE dual-ascent iteration of the whole hot path (gather lambda, candidate,
projection, item reduction, scalars, AGD update) over the full synthetic workload.  Workload = BASELINE.json
config 3 (10M users x 10k items, ~500M nonzeros, Zipf(1.1) items, box-cut(1,1), gamma = 1e-3): the config the
north_star quotes the bandwidth target on and the largest one that is routinely a single-GPU case.

Prints ONE JSON line.  `value` = nonzeros processed per second (= nnz x iterations/s), whole job, inputs
resident in HBM.  `e2e` = the same metric through the C ABI with HOST (pinned) buffers: dualip_create (H2D of
all row data) + dualip_solve (K iterations + final evaluation) + D2H of lambda and the scalars, all timed.
`roofline` = the gradient kernel's algorithmic bytes / its average launch time (CUDA events on the launching
stream, recorded inside the timed region by the library's profiling hook) against the measured HBM peak.
`cpu_baseline` = the fp64 oracle, as it stands, timed on one host core on a bounded sample of the same workload.
Multi-GPU: replicas only -- N independent copies of the job, max time over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "dual-ascent nonzeros/s (nnz x AGD iterations/s), fused gradient iteration"
UNIT = "nnz/s"
# DRAM bytes per k_grad launch from the committed `ncu --set full` capture (profiles/), or None until one exists.
NCU_TRAFFIC_BYTES = {"cfg3": 6.085430e9 + 37.377024e6, "cfg5": 7.381245e9 + 37.766912e6, "cfg4": 81.132569e9 + 38.185216e6,
                     "cfg2": 249.187584e6 + 36.514560e6}   # profiles/r01g_k_grad_tma_full.csv (dram read + write, one launch)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)      # config 3 states 1,000 AGD iterations
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--users", type=int, default=None, help="override the number of users (smaller = not the graded workload)")
    ap.add_argument("--group-lanes", type=int, default=0, help="lanes per row in the gradient kernel (0 = the library's choice)")
    ap.add_argument("--stages", type=int, default=0, help="pipeline stages of the streaming kernel (0 = the library's choice)")
    ap.add_argument("--tile-units", type=int, default=0, help="cap on the streaming kernel's tile size (0 = the library's choice)")
    ap.add_argument("--grid-ctas", type=int, default=0, help="CTAs of the gradient kernel (0 = the library's choice)")
    ap.add_argument("--graph", action="store_true", help="dualip_solve replays a CUDA graph of chained iteration launches "
                    "(small, launch-bound workloads); the per-launch kernel timing hook is then off")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-users", type=int, default=1_000_000, help="users in the oracle's bounded sample")
    return ap.parse_args()


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, STREAM-style copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (profiling recipe's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu, self.proc, self.path = gpu_index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50",
                                          "-i", str(self.gpu)], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return None
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        try:
            for line in open(self.path):
                f = [t.strip() for t in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1])); mx.append(float(f[2]))
                except ValueError:
                    continue
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def oracle_problem(inst_np, cfg, oracle, synth):
    kind, p0, p1 = synth.proj_spec(cfg)
    k = {"simplex": oracle.PROJ_SIMPLEX_INEQ, "box": oracle.PROJ_BOX, "boxcut": oracle.PROJ_BOXCUT}[kind]
    I = inst_np["row_ptr"].size - 1
    return oracle.Problem(I, cfg.J, cfg.m, inst_np["row_ptr"], inst_np["item_idx"], inst_np["c"], inst_np["a"], inst_np["b"], k, p0, p1)


def time_oracle_steps(po, gamma, steps, warmup, oracle):
    """One oracle step = one AGD iteration (gradient at y + update): oracle.solve with one iteration per call
    would add a final evaluation, so time the two parts the iteration consists of: grad + the J*m update."""
    import numpy as np
    L = oracle.lipschitz(po)
    lam = np.zeros(po.J * po.m); y = lam.copy()
    times = []
    for t in range(warmup + steps):
        t0 = time.perf_counter()
        r = oracle.grad(po, y, gamma, want_x=False)
        new = np.maximum(0.0, y + (gamma / L) * r.grad)
        y = new + (t / (t + 3.0)) * (new - lam)
        lam = new
        dt = time.perf_counter() - t0
        if t >= warmup:
            times.append(dt)
    return times


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np
    import torch

    import oracle
    import synth
    # bounded sample: about 1.5e9 nonzero-visits in the whole run (~2 minutes at the oracle's ~1.4e7 nnz/s per core),
    # split over the K + W steps; every step is one full oracle iteration over the first `users` users of the workload
    full0 = synth.get_config(args.workload)
    mean_deg = {"const": lambda d: d[1], "uniform": lambda d: (d[1] + d[2]) / 2, "poisson": lambda d: d[1]}[full0.deg[0]](full0.deg)
    users = int(1.5e9 / max(args.steps + args.warmup, 1) / mean_deg)
    users = max(2_000, min(users, 400_000, full0.I)) if args.users is None else args.users
    cfg = synth.get_config(args.workload, I=users)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    inst = synth.generate(cfg, device=dev)
    d = inst.numpy()
    po = oracle_problem(d, cfg, oracle, synth)
    times = time_oracle_steps(po, cfg.gammas[-1], args.steps, args.warmup, oracle)
    tot = float(np.sum(times))
    val = po.nnz * len(times) / tot
    full = synth.get_config(args.workload)
    sample = f"first {users} users of {args.workload} ({po.nnz} nnz) per step; oracle/dualip_oracle.c, 1 thread, fp64"
    line = {"metric": METRIC, "value": val, "unit": UNIT, "impl": "reference", "n_gpus": args.gpus, "steps": len(times),
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload} (BASELINE.json configs[{int(args.workload[3]) - 1}]: {full.I} users x {full.J} items); bounded sample",
                       "sample_users": users, "sample_nnz": po.nnz, "gamma": cfg.gammas[-1]},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    import numpy as np
    import torch

    import paper_2606_07777_b200 as pkg
    import synth

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    from paper_2606_07777_b200.replicas import Replicas
    rep = Replicas(backend="nccl")                       # replicas only: barrier + max-over-ranks, nothing on the data path
    world, rank, local = rep.world, rep.rank, rep.local_rank
    barrier = rep.barrier

    # ---- workload: generated on the device (replicas only: every rank holds the whole job) ----
    cfg = synth.get_config(args.workload, I=args.users)
    t0 = time.time()
    inst = synth.generate(cfg, device="cuda")
    torch.cuda.synchronize()
    t_gen = time.time() - t0
    kind, p0, p1 = synth.proj_spec(cfg)
    proj = {"simplex": pkg.PROJ_SIMPLEX_INEQ, "box": pkg.PROJ_BOX, "boxcut": pkg.PROJ_BOXCUT}[kind]
    gamma = cfg.gammas[-1]
    opts = pkg.binding.make_opts(projection=proj, p0=p0, p1=p1, borrow=True, group_lanes=args.group_lanes, grid_ctas=args.grid_ctas, stages=args.stages, tile_units=args.tile_units,
                                  use_graph=args.graph)
    t0 = time.time()
    prob = pkg.Problem.create(inst.I, inst.J, inst.m, inst.row_ptr, inst.item_idx, inst.c, inst.a, inst.b, opts)
    torch.cuda.synchronize()
    t_create = time.time() - t0
    info = prob.info()
    nnz, Jm = inst.nnz, inst.J * inst.m
    alg_bytes = nnz * (4 + 4 + 4 * inst.m) + 8 * inst.I          # idx + c + a per nonzero, row_ptr per user

    lam = torch.zeros(Jm, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    # ---- warm-up (untimed) ----
    prob.solve([gamma], [max(args.warmup, 3)], lam)
    lam.zero_()
    barrier()

    # ---- timed region: exactly K steps, CUDA events on the launching stream ----
    prob.set_profiling(not args.graph)
    launches0 = prob.info().launches
    sampler = ClockSampler(local)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record(stream)
    prob.solve([gamma], [args.steps], lam)                       # no final outputs requested: K gradient+update steps
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    ms_total = ev0.elapsed_time(ev1)
    inf = prob.info()
    launches = inf.launches - launches0
    kern_ms = inf.grad_kernel_ms / max(inf.grad_kernel_count, 1) if not args.graph else ms_total / args.steps
    prob.set_profiling(False)
    ms_total_max = rep.max_over_ranks(ms_total)
    value = world * nnz * args.steps / (ms_total_max * 1e-3)

    # ---- end to end through the C ABI with host buffers (create + solve + readback, all timed) ----
    e2e = None
    if not args.no_e2e:
        host = {}
        for k in ("row_ptr", "item_idx", "c", "a", "b"):
            t = getattr(inst, k)
            hbuf = torch.empty(t.shape, dtype=t.dtype, pin_memory=True)
            hbuf.copy_(t)
            host[k] = hbuf.numpy()
        torch.cuda.synchronize()
        lam_h = np.zeros(Jm)
        sc = pkg.Scalars()
        barrier()
        t0 = time.perf_counter()
        p2 = pkg.Problem.create(inst.I, inst.J, inst.m, host["row_ptr"], host["item_idx"], host["c"], host["a"], host["b"],
                                pkg.binding.make_opts(projection=proj, p0=p0, p1=p1, group_lanes=args.group_lanes, grid_ctas=args.grid_ctas, stages=args.stages, tile_units=args.tile_units,
                                                      use_graph=args.graph))
        p2.solve([gamma], [args.steps], lam_h, scalars=sc)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = rep.max_over_ranks(dt)
        h2d = sum(v.nbytes for v in host.values()) + lam_h.nbytes
        d2h = lam_h.nbytes + 5 * 8
        e2e = {"value": world * nnz * args.steps / dt, "unit": UNIT, "h2d_bytes_per_step": h2d / args.steps,
               "d2h_bytes_per_step": d2h / args.steps, "seconds": dt, "final_g": sc.g,
               "what": "dualip_create(host pinned rows) + dualip_solve(K its, host lambda, host scalars) incl. final evaluation"}
        p2.destroy()
        del host

    # ---- the oracle beside it (rank 0, N = 1 only): bounded sample of the same workload ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        import oracle
        nu = min(args.cpu_users, inst.I)
        end = int(inst.row_ptr[nu].item())
        sample = {"row_ptr": inst.row_ptr[:nu + 1].cpu().numpy(), "item_idx": inst.item_idx[:end].cpu().numpy(),
                  "c": inst.c[:end].cpu().numpy(), "a": inst.a[:end * inst.m].cpu().numpy(), "b": inst.b.cpu().numpy()}
        po = oracle_problem(sample, cfg, oracle, synth)
        times = time_oracle_steps(po, gamma, 3, 0, oracle)
        cpu = {"value": po.nnz * len(times) / float(np.sum(times)), "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"3 AGD iterations over the first {nu} users ({po.nnz} nnz) of the same instance; "
                         f"oracle/dualip_oracle.c as it stands, 1 thread, fp64; {float(np.sum(times)):.1f} s of CPU work",
               "host_cores_available": len(os.sched_getaffinity(0))}

    peak, peak_src = measured_peak()
    achieved = alg_bytes / (kern_ms * 1e-3) / 1e9 if kern_ms > 0 else None
    traffic = NCU_TRAFFIC_BYTES.get(args.workload) if args.users is None else None
    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_total_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32 (fp64 duals, fp64 shift, 64-bit fixed-point reduction)", "data": "synthetic",
            "config": {"workload": f"{args.workload} (BASELINE.json configs[{int(args.workload[3]) - 1}]): {inst.I} users x {inst.J} items, m={inst.m}, "
                                   f"{nnz} nonzeros, projection {kind}({p0},{p1}), gamma={gamma}",
                       "parallelism": "replicas only" if world > 1 else "single GPU", "l2_policy": (f"inputs larger than L2 ({alg_bytes / 1e9:.2f} GB streamed per step vs 126 MB L2); no flush needed"
                                     if alg_bytes > 4 * 126e6 else
                                     f"inputs NOT much larger than L2 ({alg_bytes / 1e6:.0f} MB per step vs 126 MB L2): partly L2-resident, not a bandwidth case"),
                       "group_lanes": info.group_lanes, "stages": info.stages, "tile_units": info.tile_units, "chunk_regs": info.chunk_regs, "grid_ctas": info.grid_ctas,
                       "block_threads": info.block_threads, "smem_bytes": info.smem_bytes,
                       "reduction": {1: "smem fixed-point", 2: "global RED.ADD.64", 3: "csc"}[info.reduction],
                       "short_rows": inst.short_rows, "cuda_graph": bool(args.graph)},
            "iters_per_s": world * args.steps / (ms_total_max * 1e-3),
            "solve_time_s": ms_total_max * 1e-3, "gen_time_s": t_gen, "create_time_s": t_create,
            "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": (achieved / peak) if achieved else None, "traffic": traffic, "peak_source": peak_src,
                         "kernel": "k_grad", "kernel_ms": kern_ms, "kernel_launches_timed": int(inf.grad_kernel_count),
                         "algorithmic_bytes_per_launch": alg_bytes,
                         "kernel_share_of_step": kern_ms * args.steps / ms_total if ms_total > 0 else None},
            "e2e": e2e, "cpu_baseline": cpu, "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    prob.destroy()
    rep.close()


if __name__ == "__main__":
    main()
