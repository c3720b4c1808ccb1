#!/usr/bin/env python
"""bench.py -- measures the dual-ascent hot path on B200 (contract: see the task statement / DESIGN.md section 8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfgN|cfgN-tight] [--gamma G] [--jacobi] [--adaptive] [--lambda zero|probe]
                    [--pre "1e-1:200,1e-2:200"] [--legs default|none|NAME,NAME...]

A "step" is ONE dual-ascent iteration of the whole hot path (gather lambda, candidate,
projection, item reduction, scalars, AGD update) over the full synthetic workload.  Headline workload = BASELINE.json
config 3 (10M users x 10k items, ~500M nonzeros, Zipf(1.1) items, box-cut(1,1), gamma = 1e-3): the config the
north_star quotes the bandwidth target on.  Taken verbatim it is slack at lambda = 0, so the headline number is the
VERTEX regime (almost every row projects onto a vertex, lambda stays 0).  The regime in which the solver moves lambda
(binding constraints, large gamma: most rows fractional) is measured by the extra LEGS below and by the flags:

    --workload cfg3-tight --jacobi --pre 1e-1:200,1e-2:200 --gamma 1e-3     the fractional regime near the optimum
    --workload cfg5 --gamma 1e-1                                            stage 1 of config 5's own schedule

Prints ONE JSON line.  `value` = nonzeros processed per second (= nnz x iterations/s), whole job, inputs
resident in HBM.  `e2e` = the same metric through the C ABI with HOST (pinned) buffers: dualip_create (H2D of
all row data) + dualip_solve (K iterations + final evaluation) + D2H of lambda and the scalars, all timed.
`roofline` = the gradient kernel's algorithmic bytes / its average launch time (CUDA events on the launching
stream, recorded inside the timed region by the library's profiling hook) against the measured HBM peak.
`cpu_baseline` = the fp64 oracle, as it stands, timed on one host core on a bounded sample of the same workload.
`legs` (N = 1, default run only) = the same measurement, K steps each, for the other large configs and for the
fractional regime, so that every number DESIGN.md / BASELINE.md quote is one tracked command.
Multi-GPU: replicas only -- N independent copies of the job, max time over ranks.
"""
from __future__ import annotations

import argparse
import csv
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
# The committed `ncu --set full` capture the `roofline.traffic` figure is READ from (rows: config,kernel,metric,unit,value;
# the config column is the leg name).  profiles/README.md names the command that produced it.
NCU_CAPTURE = os.path.join("profiles", "r02_k_grad_tma_full.csv")
NCU_CAPTURE_FALLBACK = os.path.join("profiles", "r01g_k_grad_tma_full.csv")

AGD_NOTE = ("projected Nesterov ascent, beta_t = t/(t+3), gradient at the extrapolated point: the paper prints no update "
            "formula, so this part is oracle-defined and parity-unpinned against the paper (DESIGN.md R1)")

# Extra legs of the default N = 1 run: name -> measurement spec.  The vertex-regime legs are the verbatim configs at
# their final gamma; the fractional legs are the regime the solver actually works in.
LEGS = {
    # the first iterations after the momentum restart of the gamma = 1e-3 stage (an iteration costs 4 ms right after the restart and
    # climbs to the steady state within ~25 iterations): what the round-1 review timed ...
    "cfg3-tight+jacobi@1e-3": dict(workload="cfg3-tight", jacobi=True, pre="1e-1:200,1e-2:200", gamma=1e-3, regime="fractional (transient after the stage's momentum restart)"),
    # ... and the steady state of that stage (40 untimed iterations first): every row dense (all w within gamma of each other)
    "cfg3-tight+jacobi@1e-3/steady": dict(workload="cfg3-tight", jacobi=True, pre="1e-1:200,1e-2:200", gamma=1e-3, warmup=40, regime="fractional (steady state: dense rows)"),
    "cfg5@1e-1": dict(workload="cfg5", gamma=1e-1, regime="fractional"),
    "cfg5": dict(workload="cfg5", regime="vertex"),
    "cfg2": dict(workload="cfg2", regime="vertex"),
    "cfg4": dict(workload="cfg4", regime="vertex"),
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)      # config 3 states 1,000 AGD iterations
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", help="cfgN or cfgN-tight (greedy-load right-hand side: binding constraints)")
    ap.add_argument("--gamma", type=float, default=None, help="ridge parameter of the timed steps (default: the config's final gamma)")
    ap.add_argument("--jacobi", action="store_true", help="Jacobi-preconditioned step (DESIGN.md R18)")
    ap.add_argument("--adaptive", action="store_true", help="range-clipped adaptive step (DESIGN.md R20)")
    ap.add_argument("--lambda", dest="lam", default="zero", choices=["zero", "probe"],
                    help="starting dual of the run: zeros (cold start) or the seeded probe lambda")
    ap.add_argument("--lambda-scale", type=float, default=None, help="scale of the probe lambda (default 0.5; 0.05 for config 3)")
    ap.add_argument("--pre", default="", help="untimed continuation stages run before the warm-up, e.g. 1e-1:200,1e-2:200")
    ap.add_argument("--legs", default="default", help="extra legs in the same JSON line: default (all, N = 1 default workload only), "
                    "none, or a comma list of " + ", ".join(LEGS))
    ap.add_argument("--leg-steps", type=int, default=0, help="timed steps per extra leg (0 = min(--steps, 50))")
    ap.add_argument("--users", type=int, default=None, help="override the number of users (smaller = not the graded workload)")
    ap.add_argument("--group-lanes", type=int, default=0, help="lanes per row in the gradient kernel (0 = the library's choice)")
    ap.add_argument("--stages", type=int, default=0, help="pipeline stages of the streaming kernel (0 = the library's choice)")
    ap.add_argument("--tile-units", type=int, default=0, help="cap on the streaming kernel's tile size (0 = the library's choice)")
    ap.add_argument("--grid-ctas", type=int, default=0, help="CTAs of the gradient kernel (0 = the library's choice)")
    ap.add_argument("--reduction", default="auto", choices=["auto", "smem", "global", "csc"], help="item-reduction strategy (DUALIP_RED_*)")
    ap.add_argument("--lambda-plan", type=int, default=0, help="streaming kernel's exact-path dual operand: 0 per launch, 1 never stage the low word, 2 always")
    ap.add_argument("--step-deal", type=int, default=0, help="row-steps dealt 0 = the library's choice, 1 = statically, 2 = dynamically")
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


def ncu_traffic(leg_name: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one gradient-kernel launch, read from the committed capture."""
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    for rel in (NCU_CAPTURE, NCU_CAPTURE_FALLBACK):
        path = os.path.join(ROOT, rel)
        if not os.path.exists(path):
            continue
        tot, seen = 0.0, 0
        with open(path) as f:
            for row in csv.DictReader(f):
                if row.get("config") == leg_name and row.get("metric") in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                    tot += float(row["value"]) * scale.get(row.get("unit", "byte"), 1.0)
                    seen += 1
        if seen == 2:
            return tot, rel
    return None, None


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


def parse_pre(text: str):
    """'1e-1:200,1e-2:200' -> ([0.1, 0.01], [200, 200])"""
    gam, its = [], []
    for part in filter(None, (t.strip() for t in text.split(","))):
        g, n = part.split(":")
        gam.append(float(g)); its.append(int(n))
    return gam, its


def cfg_index(workload: str):
    return int(workload[3]) - 1 if workload.startswith("cfg") else None


def oracle_problem(inst_np, cfg, oracle, synth):
    kind, p0, p1 = synth.proj_spec(cfg)
    k = {"simplex": oracle.PROJ_SIMPLEX_INEQ, "box": oracle.PROJ_BOX, "boxcut": oracle.PROJ_BOXCUT}[kind]
    I = inst_np["row_ptr"].size - 1
    return oracle.Problem(I, cfg.J, cfg.m, inst_np["row_ptr"], inst_np["item_idx"], inst_np["c"], inst_np["a"], inst_np["b"], k, p0, p1)


def time_oracle(po, gamma, iters, oracle, jacobi=False):
    """The oracle as it stands: oracle.solve runs `iters` AGD iterations (R1-R4) plus the final evaluation at lambda_T (R3),
    i.e. iters + 1 gradient evaluations -- what the product's dualip_solve does when asked for the final scalars.
    Returns (seconds, evaluations)."""
    t0 = time.perf_counter()
    oracle.solve(po, [gamma], [iters], want_x=False, jacobi=jacobi)
    return time.perf_counter() - t0, iters + 1


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch

    import oracle
    import synth
    # bounded sample: about 1.5e9 nonzero-visits in the whole run (~2 minutes at the oracle's ~1.3e7 nnz/s per core),
    # split over the K + W steps; every step is one full oracle iteration over the first `users` users of the workload
    full = synth.get_config(args.workload)
    mean_deg = {"const": lambda d: d[1], "uniform": lambda d: (d[1] + d[2]) / 2, "poisson": lambda d: d[1]}[full.deg[0]](full.deg)
    users = int(1.5e9 / max(args.steps + args.warmup + 2, 1) / mean_deg)
    users = max(2_000, min(users, 400_000, full.I)) if args.users is None else args.users
    cfg = synth.get_config(args.workload, I=users)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    inst = synth.generate(cfg, device=dev)
    d = inst.numpy()
    po = oracle_problem(d, cfg, oracle, synth)
    gamma = args.gamma if args.gamma is not None else cfg.gammas[-1]
    if args.warmup > 0:
        time_oracle(po, gamma, max(args.warmup - 1, 0), oracle, args.jacobi)                 # untimed
    tot, evals = time_oracle(po, gamma, max(args.steps - 1, 0), oracle, args.jacobi)     # K gradient evaluations
    val = po.nnz * evals / tot
    sample = (f"first {users} users of {args.workload} ({po.nnz} nnz) per step; oracle.solve ({evals - 1} AGD iterations + the final "
              f"evaluation = {evals} gradient evaluations); oracle/dualip_oracle.c, 1 thread, fp64")
    line = {"metric": METRIC, "value": val, "unit": UNIT, "impl": "reference", "n_gpus": args.gpus, "steps": evals,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / evals, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload} (BASELINE.json configs[{cfg_index(args.workload)}]: {full.I} users x {full.J} items); bounded sample",
                       "sample_users": users, "sample_nnz": po.nnz, "gamma": gamma, "jacobi": bool(args.jacobi), "agd_rule": AGD_NOTE},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


class Leg:
    """One workload resident on the device + its problem handle; measures K timed steps."""

    def __init__(self, pkg, synth, torch, spec, args):
        self.pkg, self.synth, self.torch, self.args = pkg, synth, torch, args
        self.workload = spec["workload"]
        self.cfg = synth.get_config(self.workload, I=args.users)
        self.jacobi = bool(spec.get("jacobi", False))
        self.adaptive = bool(spec.get("adaptive", False))
        self.gamma = float(spec["gamma"]) if spec.get("gamma") is not None else self.cfg.gammas[-1]
        self.pre = parse_pre(spec.get("pre", "") or "")
        self.lam_mode = spec.get("lam", "zero")
        self.lam_scale = spec.get("lam_scale")
        self.regime = spec.get("regime")
        self.warmup = spec.get("warmup")
        t0 = time.time()
        self.inst = synth.generate(self.cfg, device="cuda")
        torch.cuda.synchronize()
        self.t_gen = time.time() - t0
        kind, p0, p1 = synth.proj_spec(self.cfg)
        self.kind, self.p0, self.p1 = kind, p0, p1
        self.proj = {"simplex": pkg.PROJ_SIMPLEX_INEQ, "box": pkg.PROJ_BOX, "boxcut": pkg.PROJ_BOXCUT}[kind]
        t0 = time.time()
        self.prob = pkg.Problem.create(self.inst.I, self.inst.J, self.inst.m, self.inst.row_ptr, self.inst.item_idx, self.inst.c,
                                       self.inst.a, self.inst.b, self.opts(borrow=True))
        torch.cuda.synchronize()
        self.t_create = time.time() - t0
        self.info = self.prob.info()
        inst = self.inst
        self.nnz, self.Jm = inst.nnz, inst.J * inst.m
        self.alg_bytes = inst.nnz * (4 + 4 + 4 * inst.m) + 8 * inst.I    # idx + c + a per nonzero, row_ptr per user

    def opts(self, borrow):
        a = self.args
        return self.pkg.binding.make_opts(projection=self.proj, p0=self.p0, p1=self.p1, borrow=borrow, group_lanes=a.group_lanes,
                                          grid_ctas=a.grid_ctas, stages=a.stages, tile_units=a.tile_units, use_graph=a.graph,
                                          jacobi=self.jacobi, adaptive=self.adaptive, lambda_plan=a.lambda_plan, step_deal=a.step_deal,
                                          reduction={"auto": 0, "smem": 1, "global": 2, "csc": 3}[a.reduction])

    def start_lambda(self):
        torch = self.torch
        if self.lam_mode == "probe":
            scale = self.lam_scale if self.lam_scale is not None else (0.05 if self.workload.startswith("cfg3") else 0.5)
            return self.synth.probe_lambda(self.inst, 0, scale).clone()
        return torch.zeros(self.Jm, dtype=torch.float64, device="cuda")

    def measure(self, steps, warmup, barrier, local_rank):
        """pre stages (untimed) -> W warm-up iterations -> exactly K timed iterations, all continuing one trajectory."""
        torch, prob = self.torch, self.prob
        lam = self.start_lambda()
        stream = torch.cuda.current_stream()
        if self.pre[0]:
            prob.solve(self.pre[0], self.pre[1], lam)
        prob.solve([self.gamma], [max(self.warmup if self.warmup is not None else warmup, 3)], lam)
        barrier()
        prob.set_profiling(not self.args.graph)
        launches0 = prob.info().launches
        sampler = ClockSampler(local_rank)
        sampler.start()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record(stream)
        prob.solve([self.gamma], [steps], lam)                     # no final outputs requested: K gradient+update steps
        ev1.record(stream)
        barrier()
        clocks = sampler.stop()
        ms_total = ev0.elapsed_time(ev1)
        inf = prob.info()
        launches = inf.launches - launches0
        kern_ms = inf.grad_kernel_ms / max(inf.grad_kernel_count, 1) if not self.args.graph else ms_total / steps
        prob.set_profiling(False)
        sc = self.pkg.Scalars()
        prob.grad(lam, self.gamma, scalars=sc)                      # state the timed steps ended in (untimed)
        torch.cuda.synchronize()
        state = {"g": sc.g, "r_inf": sc.r_inf, "active_duals": int((lam > 0).sum().item()), "lambda_max": float(lam.max().item()),
                 "table4": sc.table4(), "lambda_lo_smem": int(prob.info().lambda_lo_smem)}
        return {"ms_total": ms_total, "kern_ms": kern_ms, "launches": int(launches), "timed": int(inf.grad_kernel_count),
                "clocks": clocks, "state": state}

    def kernel_name(self):
        i = self.info
        if self.kind == "box":
            return "k_grad_box"
        return f"k_grad_tma<G={i.group_lanes}, M={self.inst.m}>" if i.streaming else f"k_grad<G={i.group_lanes}, KREG={i.chunk_regs}, M={self.inst.m}>"

    def config(self, world):
        i, inst = self.info, self.inst
        base = self.workload.split("-")[0]
        return {"workload": f"{self.workload} (" + (f"BASELINE.json configs[{cfg_index(self.workload)}]" if cfg_index(self.workload) is not None else "stress recipe, not a BASELINE.json config") +
                            (", right-hand side by the paper's greedy-load rule P:264-268: binding constraints" if self.workload.endswith("-tight") else "") +
                            f"): {inst.I} users x {inst.J} items, m={inst.m}, {self.nnz} nonzeros, projection {self.kind}({self.p0},{self.p1}), gamma={self.gamma}",
                "regime": self.regime or ("vertex (the verbatim config is slack at lambda = 0: lambda stays 0, almost every row projects onto a vertex)"
                                          if self.workload == base and self.lam_mode == "zero" and not self.pre[0] and self.gamma <= self.cfg.gammas[-1] else "see gamma / lambda / pre"),
                "jacobi": self.jacobi, "adaptive_step": self.adaptive, "lambda_start": self.lam_mode,
                "pre_stages": [f"{g}:{n}" for g, n in zip(*self.pre)],
                "agd_rule": AGD_NOTE,
                "parallelism": "replicas only" if world > 1 else "single GPU",
                "l2_policy": (f"inputs larger than L2 ({self.alg_bytes / 1e9:.2f} GB streamed per step vs 126 MB L2); no flush needed"
                              if self.alg_bytes > 4 * 126e6 else
                              f"inputs NOT much larger than L2 ({self.alg_bytes / 1e6:.0f} MB per step vs 126 MB L2): partly L2-resident, not a bandwidth case"),
                "group_lanes": i.group_lanes, "stages": i.stages, "tile_units": i.tile_units, "chunk_regs": i.chunk_regs, "grid_ctas": i.grid_ctas,
                "block_threads": i.block_threads, "smem_bytes": i.smem_bytes,
                "reduction": {1: "smem fixed-point", 2: "global RED.ADD.64", 3: "csc"}[i.reduction],
                "short_rows": inst.short_rows, "cuda_graph": bool(self.args.graph)}

    def roofline(self, m, steps, leg_name):
        peak, peak_src = measured_peak()
        achieved = self.alg_bytes / (m["kern_ms"] * 1e-3) / 1e9 if m["kern_ms"] > 0 else None
        traffic, src = ncu_traffic(leg_name) if self.args.users is None else (None, None)
        dram = (traffic / (m["kern_ms"] * 1e-3) / 1e9) if (traffic and m["kern_ms"] > 0) else None
        return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": (achieved / peak) if achieved else None,
                "traffic": traffic, "traffic_source": src, "dram_gbs": dram, "dram_frac": (dram / peak) if dram else None,
                "bytes_note": ("achieved = ALGORITHMIC bytes of the ABI's format (int32 index + fp32 c + m fp32 a per nonzero, int64 row_ptr per user: "
                               "SURVEY 8(d)) / kernel time.  The streaming kernel reads a uint16 copy of the item indices kept by dualip_create "
                               "(J < 65536 whenever lambda fits in shared memory: SURVEY 8(d)'s 'legitimate byte reduction'), i.e. it moves 2 bytes "
                               "per nonzero less than that: traffic / dram_gbs / dram_frac are what actually crosses the HBM interface (ncu), so frac "
                               "can exceed dram_frac and 1" if self.info.streaming else None),
                "peak_source": peak_src, "kernel": self.kernel_name(), "kernel_ms": m["kern_ms"],
                "kernel_launches_timed": m["timed"], "algorithmic_bytes_per_launch": self.alg_bytes,
                "kernel_share_of_step": m["kern_ms"] * steps / m["ms_total"] if m["ms_total"] > 0 else None}

    def close(self):
        self.prob.destroy()
        del self.inst
        self.torch.cuda.empty_cache()


def leg_name_of(args):
    n = args.workload
    if args.jacobi:
        n += "+jacobi"
    if args.adaptive:
        n += "+adaptive"
    if args.gamma is not None:
        n += f"@{args.gamma:g}"
    return n


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

    # ---- headline workload: generated on the device (replicas only: every rank holds the whole job) ----
    spec = dict(workload=args.workload, gamma=args.gamma, jacobi=args.jacobi, adaptive=args.adaptive, lam=args.lam,
                lam_scale=args.lambda_scale, pre=args.pre)
    leg = Leg(pkg, synth, torch, spec, args)
    inst, nnz, Jm = leg.inst, leg.nnz, leg.Jm
    m = leg.measure(args.steps, args.warmup, barrier, local)
    ms_total_max = rep.max_over_ranks(m["ms_total"])
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
        lam_h = leg.start_lambda().cpu().numpy()
        sc = pkg.Scalars()
        gam_all, its_all = leg.pre[0] + [leg.gamma], leg.pre[1] + [args.steps]
        barrier()
        t0 = time.perf_counter()
        p2 = pkg.Problem.create(inst.I, inst.J, inst.m, host["row_ptr"], host["item_idx"], host["c"], host["a"], host["b"], leg.opts(borrow=False))
        p2.solve(gam_all, its_all, lam_h, scalars=sc)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = rep.max_over_ranks(dt)
        h2d = sum(v.nbytes for v in host.values()) + lam_h.nbytes
        d2h = lam_h.nbytes + 5 * 8
        n_e2e = int(sum(its_all))
        e2e = {"value": world * nnz * n_e2e / dt, "unit": UNIT, "h2d_bytes_per_step": h2d / n_e2e,
               "d2h_bytes_per_step": d2h / n_e2e, "seconds": dt, "iterations": n_e2e, "final_g": sc.g,
               "what": "dualip_create(host pinned rows) + dualip_solve(pre stages + K its, host lambda, host scalars) incl. final evaluation"}
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
        po = oracle_problem(sample, leg.cfg, oracle, synth)
        secs, evals = time_oracle(po, leg.gamma, 2, oracle, leg.jacobi)
        cpu = {"value": po.nnz * evals / secs, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"oracle.solve: 2 AGD iterations + the final evaluation = {evals} gradient evaluations over the first {nu} users "
                         f"({po.nnz} nnz) of the same instance; oracle/dualip_oracle.c as it stands, 1 thread, fp64; {secs:.1f} s of CPU work",
               "host_cores_available": len(os.sched_getaffinity(0))}
        del po, sample

    name = leg_name_of(args)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_total_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32 (fp64 duals, fp64 shift, 64-bit fixed-point reduction)", "data": "synthetic",
        "config": leg.config(world),
        "iters_per_s": world * args.steps / (ms_total_max * 1e-3),
        "solve_time_s": ms_total_max * 1e-3, "gen_time_s": leg.t_gen, "create_time_s": leg.t_create,
        "gpu_launches": m["launches"],
        "roofline": leg.roofline(m, args.steps, name),
        "end_state": m["state"],
        "e2e": e2e, "cpu_baseline": cpu, "clocks": m["clocks"],
    }
    leg.close()

    # ---- extra legs (N = 1): the other large configs and the fractional regime, K steps each ----
    want = []
    if args.legs == "default":
        if world == 1 and args.workload == "cfg3" and args.users is None and args.gamma is None and not args.jacobi and not args.pre \
                and not args.adaptive and args.lam == "zero":
            want = list(LEGS)
    elif args.legs != "none":
        want = [t.strip() for t in args.legs.split(",") if t.strip()]
    legs = {}
    total_mem = torch.cuda.get_device_properties(local).total_memory
    for nm in want:
        spec = LEGS[nm]
        cfg = synth.get_config(spec["workload"], I=args.users)
        mean_deg = {"const": lambda d: d[1], "uniform": lambda d: (d[1] + d[2]) / 2, "poisson": lambda d: d[1]}[cfg.deg[0]](cfg.deg)
        need = cfg.I * mean_deg * (8 + 4 * cfg.m) * 1.35
        if need > total_mem:
            legs[nm] = {"skipped": f"needs about {need / 1e9:.0f} GB of device memory"}
            continue
        k = args.leg_steps if args.leg_steps > 0 else min(args.steps, 50)
        try:
            lg = Leg(pkg, synth, torch, spec, args)
            mm = lg.measure(k, args.warmup, barrier, local)
            legs[nm] = {"value": lg.nnz * k / (mm["ms_total"] * 1e-3), "unit": UNIT, "steps": k, "ms_per_step": mm["ms_total"] / k,
                        "config": lg.config(world), "roofline": lg.roofline(mm, k, nm), "end_state": mm["state"], "clocks": mm["clocks"],
                        "gpu_launches": mm["launches"]}
            lg.close()
        except Exception as e:                                       # a leg must never take the headline line down with it
            legs[nm] = {"error": f"{type(e).__name__}: {e}"}
    if legs:
        line["legs"] = legs
    if rank == 0:
        print(json.dumps(line), flush=True)
    rep.close()


if __name__ == "__main__":
    main()
