#!/usr/bin/env python
"""bench.py -- OPTCC-schedule AllReduce on B200: algbw GB/s, the executor against its HBM roofline, modeled T/T0.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--k -1] [--exec-mode 0] [--impl reference]

One "step" = one pass of the whole hot path over one batch of seeded synthetic input,
all through the C ABI: optcc_plan (classify, bandwidth-weighted chunking, flow / step tables), then optcc_cost (the
alpha-beta model, on a second host thread) beside optcc_prepare + optcc_execute (reduce and copy steps) +
optcc_verify (contributor masks).  `value` = n*sizeof(dtype) / step time (algorithm bandwidth, BASELINE.json's
metric) summed over ranks; `execute_only` gives the same metric for the AllReduce proper (optcc_execute alone).
The executor and k are the library's and the model's: exec_mode 0 = OPTCC_EXEC_AUTO (what a user of optcc_plan
gets), k = the k at which the modelled T/T0 is within the paper's reported gap (BENCH_K).

`roofline.frac` is an HBM fraction: for the column / dataflow executors the compulsory DRAM bytes 2 p n sizeof
(inputs read once, outputs written once) over the kernel's CUDA-event time against the measured copy peak -- their
partial sums live in L1 / L2, so the schedule's 5 (p-1) n sizeof bytes never reach HBM (`schedule_over_peak` keeps
that ratio); `roofline_stepwise` times the step-ordered persistent executor on the same workload in the same run and
reports SURVEY 8(d)'s literal number, schedule bytes / time.  `other_configs` carries C1, C3, C4 and the whole C5
sweep (execute ms, verify ms, both fractions, k, modelled T/T0, a parity spot check each).
Inputs are restored from a pristine device copy between steps, outside the timed events (the AllReduce is in place);
that restore also flushes L2 (footprint >> 126 MB).

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
--gpus N: N independent replicas, one per GPU -- the path shards along the element axis with no data-path collective
(SURVEY 8(e)); under torchrun each rank is one replica, without it bench.py starts the N workers itself; NCCL is used
for the barrier and the max over ranks of the device times only; scaling is "weak".
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "OPTCC-schedule AllReduce algbw"
UNIT = "GB/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs index (default 1 = C2, the metric's config)")
    ap.add_argument("--ell", type=float, default=1.6, help="ell for config 4 (the C5 sweep)")
    ap.add_argument("--k", type=int, default=-1,
                    help="segments (PAPER.md:124); -1 = bench default per config (BENCH_K: the modelled-gap k), 0 = planner's auto rule")
    ap.add_argument("--exec-mode", type=int, default=0,
                    help="OPTCC_EXEC_*: 0 = auto (the library chooses from the plan's shape; what a user of optcc_plan gets), "
                         "1 persistent kernel with grid barriers, 2 one launch per step, 3 dataflow kernel, 4 column kernel")
    ap.add_argument("--tile-units", type=int, default=0, help="opts.tile_units (0 = the library's choice)")
    ap.add_argument("--col-order", type=int, default=0, help="opts.col_order (column executor: 0 chain by chain, 1 table order)")
    ap.add_argument("--no-forward", type=int, default=0, help="opts.no_forward (column executor, f32: 1 = every reduce flow loads both operands)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--e2e-shards", type=int, default=16,
                    help="element shards of the end-to-end leg (optcc_execute_host_sharded: H2D, execute and D2H of "
                         "neighbouring shards overlap); 1 = optcc_execute_host, one plan for the whole n")
    ap.add_argument("--cpu-sample-log2", type=int, default=0,
                    help="log2 of n per rank for the CPU-oracle sample (0 = 24 for the cpu_baseline leg, 22 per --impl reference step)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--only-main", action="store_true", help="skip roofline_stepwise and other_configs (profiling runs)")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


# k per config: free in BASELINE.json's configs; the k at which the modelled T/T0 is within the paper's
# reported gap (<= 1.06 single straggler, <= 1.085 multi-straggler, <= 1.06 multi-GPU) -- the column
# executor's time does not depend on k, so the timed k is the modelled-gap k
BENCH_K = {0: 20, 1: 16, 2: 20, 3: 32, 4: 24}


EXEC_KERNEL = {1: "optcc_exec_kernel", 2: "optcc_exec_kernel", 3: "optcc_dataflow_kernel", 4: "optcc_column_kernel"}


def bench_k(args):
    return BENCH_K[args.config] if args.k < 0 else args.k


def workload_name(w, k):
    return f"{w.name}: {w.note}; k={k}"


# ------------------------------------------------------------------------------------------------------------
# CPU oracle legs (the only place bench.py executes oracle/)
# ------------------------------------------------------------------------------------------------------------
def oracle_step(w, k):
    """One pass of the whole path by the oracle as it stands, on workload w (a bounded sample of the config):
    plan, cost simulation, plan-order execution, masks, fp64 reference sum.  Returns seconds."""
    import numpy as np
    from paper_2606_01680_b200 import workloads as W
    from oracle import planner as OP, interpreter as OI, cost_sim, reference as OR
    x = W.all_inputs(w)
    t0 = time.perf_counter()
    plan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=k)
    cost_sim.simulate(plan)
    if w.dtype == W.F32:
        y = OI.run_f32(plan, x)
        ok = OR.check_f32(y[0], x).all()
    else:
        y = OI.run_bf16(plan, x)
        ok = OR.check_bf16(OI.bf16_bits_to_f32(y[0]), OI.bf16_bits_to_f32(x)).all()
    masks, overlaps = OI.element_masks(plan)
    ok = ok and overlaps == 0 and bool((masks == OI.full_mask_words(w.p)[None, None, :]).all())
    dt = time.perf_counter() - t0
    if not ok:
        raise RuntimeError("oracle self-check failed")
    return dt


def oracle_walk_compiled(w, k):
    """The oracle's flow walk restated in C (oracle/walk.c: same table, same order, one IEEE add per element of a
    reduce flow, the independent flows of a step spread over the host threads), on workload w (fp32).  Only the walk is
    timed -- no planning, cost simulation, masks or fp64 check.  Returns (seconds, threads)."""
    from paper_2606_01680_b200 import workloads as W
    from oracle import planner as OP, cwalk
    plan = OP.build_plan(w.p, w.g, list(w.ell), w.n, w.dtype, k=k)
    x = W.all_inputs(w)
    t0 = time.perf_counter()
    y = cwalk.run_f32(plan, x, copy=False)
    dt = time.perf_counter() - t0
    if not all(y[r, :4096].tobytes() == y[0, :4096].tobytes() for r in range(1, w.p)):
        raise RuntimeError("compiled oracle walk: outputs differ between ranks")
    return dt, cwalk.threads()


def cpu_threads_used():
    """Threads the oracle actually uses: its numpy work is elementwise slicing/adding (no BLAS), one thread."""
    return 1


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric / config, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2606_01680_b200 import workloads as W
    w_full = W.config(args.config, args.ell) if args.config == 4 else W.config(args.config)
    lg = args.cpu_sample_log2 or 22
    w = w_full.scaled(min(w_full.n, 2 ** lg))
    from oracle import planner as OP
    k = OP.build_plan(w_full.p, w_full.g, list(w_full.ell), w_full.n, w_full.dtype, k=bench_k(args)).k
    for _ in range(min(args.warmup, 1)):
        oracle_step(w, k)
    ts = [oracle_step(w, k) for _ in range(args.steps)]
    t = sum(ts) / len(ts)
    value = w.n * w.elem_bytes / t / 1e9
    sample = f"n={w.n} elements per rank (2^{lg}) of the config's n={w_full.n}, all p={w.p} ranks, every flow of the plan"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": min(args.warmup, 1), "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32" if w.dtype == W.F32 else "bf16", "data": "synthetic",
        "config": {"workload": workload_name(w_full, k), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cpu_threads_used(), "kind": "oracle", "sample": sample,
                         "host_cores": os.cpu_count()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------------------
# native arm
# ------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons of one GPU while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [c.strip() for c in line.split(",")]))

    def count_since(self, t):
        return sum(1 for ts, _ in self.rows if ts >= t)

    def stop(self, t_begin=0.0):
        """Median SM clock and throttle reasons over the samples taken since t_begin (perf_counter)."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, r in self.rows:
            if ts < t_begin:
                continue
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
            except Exception:
                continue
            for name, val in zip(names, r[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy, burst: the kernel is timed alone)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def ncu_traffic(workload, kernel):
    """(dram bytes per launch, commit the capture was taken at, source) of `kernel` from the committed ncu --set full
    captures (profiles/exec_kernel_traffic.csv), or (None, None, None).  ncu cannot run inside the bench: the line says
    which commit the byte count belongs to."""
    path = os.path.join(ROOT, "profiles", "exec_kernel_traffic.csv")
    if not os.path.exists(path):
        return None, None, None
    for line in open(path):
        if line.startswith("#"):
            continue
        parts = [s.strip() for s in line.split(",")]
        if len(parts) >= 5 and parts[0] == workload and parts[1] == kernel:
            try:
                return float(parts[2]), parts[3], parts[4]
            except ValueError:
                return None, None, None
    return None, None, None


EXEC_NAME = {1: "persistent cooperative kernel, grid barrier per step", 2: "one launch per step",
             3: "dataflow cooperative kernel: tile-ops in table order, per-range completion counters, no grid barrier",
             4: "column kernel: a tile is taken through its region's whole flow list in dependency order, partial sums "
                "forwarded in registers between consecutive flows, no synchronisation between CTAs (every dependency lies "
                "inside one element column)"}


def roofline_of(kernel, exec_mode, p, n, esize, t_ms, peak, peak_src):
    """HBM roofline of one executor launch.  Step-ordered executors (persistent, per-step): SURVEY 8(d)'s schedule
    bytes 5 (p-1) n sizeof -- every flow's operands travel through HBM / L2 in global step order.  Column and dataflow
    executors: the partial sums of a tile stay in L1 / L2, so what HBM must carry is the compulsory 2 p n sizeof
    (every input read once, every output written once); the schedule-bytes ratio is kept beside it."""
    sched = 5 * (p - 1) * n * esize
    comp = 2 * p * n * esize
    stepwise = exec_mode in (1, 2)
    nbytes = sched if stepwise else comp
    return {"bound": "hbm", "kernel": kernel, "achieved": nbytes / t_ms / 1e6, "peak": peak, "peak_source": peak_src, "unit": "GB/s",
            "frac": nbytes / t_ms / 1e6 / peak,
            "definition": ("schedule bytes 5 (p-1) n sizeof / kernel time (SURVEY 8(d)): this executor keeps global step order, "
                           "every flow's operands go through HBM / L2") if stepwise else
                          ("compulsory DRAM bytes 2 p n sizeof (every input read once, every output written once) / kernel time: "
                           "this executor takes a tile through its whole flow list, partial sums travel between consecutive flows "
                           "in registers (column executor) or through L1 / L2, so the schedule's 5 (p-1) n sizeof bytes never reach "
                           "HBM (see schedule_over_peak; roofline_every_load_and_store: the same with opts.no_forward = 1)"),
            "algorithmic_bytes_per_launch": nbytes, "schedule_bytes_per_launch": sched,
            "schedule_over_peak": sched / t_ms / 1e6 / peak, "ms": t_ms}


class Bench:
    """Device state shared by the measurements of one bench run."""

    def __init__(self, args):
        import torch
        from paper_2606_01680_b200 import binding as B, workloads as W
        from paper_2606_01680_b200 import build as optcc_build
        from paper_2606_01680_b200.device import Session
        from paper_2606_01680_b200.replicas import Replicas
        self.torch, self.B, self.W, self.Session = torch, B, W, Session
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: liboptcc has no CPU fallback (use --impl reference for the oracle)")
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        torch.cuda.set_device(self.local)
        self.dev = torch.device("cuda", self.local)
        self.rep = Replicas(backend="nccl", device=self.dev)
        if self.rep.rank == 0:
            optcc_build.build()
        self.rep.barrier()
        B.load()
        self.stream = torch.cuda.current_stream(self.dev)
        self.args = args
        self.peak, self.peak_src = measured_peak()
        import queue
        self.cost_in, self.cost_out = queue.SimpleQueue(), queue.SimpleQueue()
        threading.Thread(target=self._cost_worker, daemon=True).start()

    def _cost_worker(self):
        """The second host thread: optcc_cost of every plan it is handed (started once: creating a Python thread per
        step costs 50-100 us of the step)."""
        while True:
            plan = self.cost_in.get()
            if plan is None:
                return
            tc = time.perf_counter()
            c = self.B.optcc_cost(plan)
            self.cost_out.put((c, (time.perf_counter() - tc) * 1e3))
            del plan

    def ev(self):
        return self.torch.cuda.Event(enable_timing=True)

    def measure(self, w, k, steps, warmup, x=None, sampler=None, keep=False, exec_mode=None, execute_only=False, no_forward=None):
        """`steps` timed passes of the whole hot path on workload w (inputs resident in HBM, restored from a pristine
        device copy between passes, untimed: the AllReduce is in place and the restore flushes L2).  One pass =
        optcc_plan -> {optcc_cost on a second host thread} || {optcc_prepare, optcc_execute, optcc_verify} -> join."""
        torch, B, W, args = self.torch, self.B, self.W, self.args
        import numpy as np
        esize = w.elem_bytes
        mode = args.exec_mode if exec_mode is None else exec_mode
        nf = args.no_forward if no_forward is None else no_forward
        mk = lambda: B.optcc_plan(w.p, w.g, w.ell, w.n, w.dtype, k=k, exec_mode=mode, tile_units=args.tile_units,
                                  col_order=args.col_order, no_forward=nf)
        plan0 = mk()
        info = plan0.info
        cost0 = B.optcc_cost(plan0)
        sess = self.Session(plan0, device=self.dev, verify=not execute_only)
        if x is None:
            x = W.all_inputs(w)
        sess.upload(x)
        pristine = [b.clone() for b in sess.bufs]
        restore = lambda: [b.copy_(s) for b, s in zip(sess.bufs, pristine)]
        stream = self.stream

        def one_pass():
            e = [self.ev() for _ in range(5)]
            box = {}
            e[0].record(stream)
            t0 = time.perf_counter()
            plan = mk()                                   # a1-a3: classify, chunk, flow / step tables
            t1 = time.perf_counter()

            if not execute_only:
                self.cost_in.put(plan)                    # a4 on a second host thread (ctypes releases the GIL)
            old = sess.plan
            sess.plan = plan
            sess.prepare()                                # the executor's tables, built on the host and uploaded
            e[1].record(stream)                           # (in stream order after the upload: plan_to_launch ends here)
            sess.execute()                                # a5-a7
            e[2].record(stream)
            del old                                       # the previous step's plan is destroyed while the GPU works
            res = None if execute_only else sess.verify() # a8 (synchronises the stream once to read the counters)
            e[3].record(stream)
            if not execute_only:
                box["cost"], box["cost_ms"] = self.cost_out.get()
            e[4].record(stream)
            torch.cuda.synchronize(self.dev)
            if res is not None and (res["bad_elements"] or res["overlap_elements"]):
                raise RuntimeError(f"verification failed: {res}")
            return {"total": e[0].elapsed_time(e[4]), "plan_host": (t1 - t0) * 1e3, "cost_host": box.get("cost_ms", 0.0),
                    "plan_to_launch": e[0].elapsed_time(e[1]), "execute": e[1].elapsed_time(e[2]),
                    "verify": e[2].elapsed_time(e[3]), "cost_not_hidden": e[3].elapsed_time(e[4])}

        for _ in range(warmup):
            restore()
            one_pass()
        if sampler is not None:
            for _ in range(200):         # nvidia-smi takes longer to start than a short timed region lasts
                if sampler.count_since(0.0) or not sampler.proc:
                    break
                restore()
                one_pass()
        self.rep.barrier()
        torch.cuda.synchronize(self.dev)
        recs = []
        wall0 = time.perf_counter()
        for _ in range(steps):
            restore()
            torch.cuda.synchronize(self.dev)
            recs.append(one_pass())
        torch.cuda.synchronize(self.dev)
        wall = time.perf_counter() - wall0
        clocks = None
        if sampler is not None:
            in_region = sampler.count_since(wall0)
            extra = 0
            while sampler.proc and sampler.count_since(wall0) < 3 and extra < 400:
                restore()                # region shorter than three sampling periods: keep the same load running, untimed
                one_pass()
                extra += 1
            clocks = sampler.stop(wall0)
            clocks["samples_in_timed_region"] = in_region
            clocks["untimed_steps_of_the_same_load_added_for_sampling"] = extra
        self.rep.barrier()
        mean = lambda key: sum(r[key] for r in recs) / len(recs)
        t_step, t_exec, t_ver = self.rep.max_over_ranks([mean("total"), mean("execute"), mean("verify")])
        # parity spot-check of the last timed pass against the fp64 sum on sampled elements (cheap, outside timing)
        idx = W.sample_indices(w, 4096)
        y0 = sess.bufs[0][torch.from_numpy(idx).to(self.dev)].float().cpu().numpy().astype(np.float64)
        if w.dtype == W.F32:
            xs = x[:, idx].astype(np.float64)
            tol = w.p * 2.0 ** -23 * np.abs(xs).sum(0)
        else:
            xs = (x[:, idx].astype(np.uint32) << 16).view(np.float32).astype(np.float64)
            tol = 2.0 ** -7 * np.abs(xs.sum(0)) + w.p * 2.0 ** -23 * np.abs(xs).sum(0)
        parity_ok = bool((np.abs(y0 - xs.sum(0)) <= tol).all())
        ranks_equal = all(torch.equal(sess.bufs[0].view(torch.int16 if w.dtype == W.BF16 else torch.int32),
                                      b.view(torch.int16 if w.dtype == W.BF16 else torch.int32)) for b in sess.bufs[1:])
        parity_ok = self.rep.all_true(parity_ok and ranks_equal)
        out = {"w": w, "k": info["k"], "info": info, "cost": cost0, "t_step": t_step, "t_exec": t_exec, "t_ver": t_ver,
               "breakdown_ms": {"plan_host": mean("plan_host"), "plan_to_launch": mean("plan_to_launch"), "execute": t_exec,
                                "verify": t_ver, "cost_host_on_second_thread": mean("cost_host"),
                                "cost_host_not_hidden": mean("cost_not_hidden")},
               "parity_ok": parity_ok, "idx": idx, "xs": xs, "tol": tol, "wall": wall, "clocks": clocks, "steps": steps}
        if keep:
            out["sess"], out["x"] = sess, x
        else:
            del sess, pristine
            torch.cuda.empty_cache()
        return out

    def summary(self, m):
        """The per-config object of `other_configs` (and the pieces of the headline line)."""
        w, info, c = m["w"], m["info"], m["cost"]
        esize = w.elem_bytes
        mode = info["exec_mode"]
        kern = EXEC_KERNEL[mode] + ("<MODE_F32>" if w.dtype == self.W.F32 else "<MODE_BF16>")
        roof = roofline_of(kern, mode, w.p, w.n, esize, m["t_exec"], self.peak, self.peak_src)
        mask_final = w.p * w.n * info["mask_bytes"]
        lb = c["lb_table1"] / c["T0"]
        return {"workload": workload_name(w, m["k"]), "k": m["k"], "executor": EXEC_NAME[mode], "step_ms": m["t_step"],
                "algbw_GBs": self.rep.world * w.n * esize / m["t_step"] / 1e6,
                "execute_ms": m["t_exec"], "execute_algbw_GBs": self.rep.world * w.n * esize / m["t_exec"] / 1e6,
                "verify_ms": m["t_ver"], "breakdown_ms": m["breakdown_ms"], "plan_steps": info["n_steps"], "plan_flows": info["n_flows"],
                "roofline_frac": roof["frac"], "schedule_over_peak": roof["schedule_over_peak"],
                "roofline_verify_frac": mask_final / m["t_ver"] / 1e6 / self.peak,
                "model": {"T_over_T0": c["T_over_T0"], "lb_table1_over_T0": lb, "T_over_lb_table1": c["T_over_T0"] / lb,
                          "lb_tight_over_T0": (c["lb_tight"] / c["T0"]) if c["lb_tight"] == c["lb_tight"] else None},
                "parity_spot_check": {"sampled_elements": int(len(m["idx"])), "within_tolerance_and_all_ranks_identical": m["parity_ok"]}}


def run_native(args):
    import numpy as np
    bench = Bench(args)
    torch, B, W, rep = bench.torch, bench.B, bench.W, bench.rep
    rank, world, dev, stream = rep.rank, rep.world, bench.dev, bench.stream
    w = rep.shard(W.config(args.config, args.ell) if args.config == 4 else W.config(args.config))
    esize = w.elem_bytes
    sampler = ClockSampler(bench.local)
    sampler.start()
    m = bench.measure(w, bench_k(args), args.steps, max(args.warmup, 3), sampler=sampler, keep=True)
    sess, x, info, cost0, k = m["sess"], m["x"], m["info"], m["cost"], m["k"]
    t_step, t_exec, t_ver = m["t_step"], m["t_exec"], m["t_ver"]
    idx, xs, tol = m["idx"], m["xs"], m["tol"]
    exec_mode = info["exec_mode"]          # what OPTCC_EXEC_AUTO resolved to
    launches_per_step = (info["n_steps"] if exec_mode == 2 else 1) * 2 + (0 if info["lazy_verify"] else 2)

    # e2e: the same step through the C-ABI call with HOST buffers, H2D + D2H inside the timed region.  The path shards
    # along the element axis, so the host call pipelines S element shards, each an AllReduce with the
    # plan for n / S: copy-in of shard c+1, execution of shard c and copy-out of shard c-1 overlap.
    e2e = None
    if not args.no_e2e:
        S = max(1, args.e2e_shards)
        while S > 1 and (w.n % S or (w.n // S) % 8):
            S //= 2
        mk_e = lambda: B.optcc_plan(w.p, w.g, w.ell, w.n // S, w.dtype, k=bench_k(args), exec_mode=args.exec_mode,
                                    tile_units=args.tile_units, col_order=args.col_order, no_forward=args.no_forward)
        se = bench.Session(mk_e(), device=dev, verify=True, alloc_bufs=False, shards=S)
        se.bufs = sess.bufs
        hin = [torch.from_numpy(x[r]).pin_memory() if w.dtype == W.F32 else
               torch.from_numpy(x[r].view(np.int16)).pin_memory() for r in range(w.p)]
        hout = [torch.empty_like(t).pin_memory() for t in hin]
        ts = []
        for i in range(1 + args.e2e_steps):
            a, b_ = bench.ev(), bench.ev()
            torch.cuda.synchronize(dev)
            a.record(stream)
            plan = mk_e()
            se.plan = plan
            if S > 1:
                se.execute_host_sharded(hin, hout)
            else:
                se.execute_host(hin, hout)
            B.optcc_cost(plan)       # on the host while the copies and the plan run
            se.verify()
            b_.record(stream)
            torch.cuda.synchronize(dev)
            if i:
                ts.append(a.elapsed_time(b_))
        t_e2e = rep.max_over_ranks([sum(ts) / len(ts)])[0]
        ok = all(torch.equal(hout[0], h) for h in hout[1:])
        y_e = hout[0].numpy()[idx].astype(np.float64) if w.dtype == W.F32 else \
            (hout[0].numpy().view(np.uint16)[idx].astype(np.uint32) << 16).view(np.float32).astype(np.float64)
        ok = ok and bool((np.abs(y_e - xs.sum(0)) <= tol).all())           # the pipelined result against the fp64 sum
        e2e = {"value": world * w.n * esize / t_e2e / 1e6, "unit": UNIT, "h2d_bytes_per_step": w.p * w.n * esize,
               "d2h_bytes_per_step": w.p * w.n * esize, "ms_per_step": t_e2e, "steps": len(ts),
               "call": ("optcc_execute_host_sharded: %d element shards of n/%d, one plan, H2D / execute / D2H overlapped" % (S, S))
                       if S > 1 else "optcc_execute_host",
               "all_ranks_identical_and_within_tolerance": bool(ok)}
        del hin, hout, se

    # the number SURVEY 8(d) literally defines: a step-ordered executor (global step order, every intermediate state
    # of the p buffers in HBM / L2) at its best k, on the same workload in the same run
    stepwise = None
    stepwise_extra = None
    if not args.only_main and args.config == 1 and rank == 0 and world == 1:
        del sess
        m.pop("sess")
        torch.cuda.empty_cache()
        ms = bench.measure(w, 4, 5, 3, x=x, exec_mode=B.OPTCC_EXEC_PERSISTENT, execute_only=True)
        kern = "optcc_exec_kernel<MODE_F32>"
        stepwise = roofline_of(kern, 1, w.p, w.n, esize, ms["t_exec"], bench.peak, bench.peak_src)
        stepwise["k"] = ms["k"]
        stepwise["executor"] = EXEC_NAME[1]
        tr, sha, src = ncu_traffic("C2", kern)
        stepwise["traffic"] = tr
        stepwise["traffic_captured_at_commit"] = sha
        # ... and the column executor with every load and store of every flow issued (opts.no_forward = 1): what the
        # register forwarding of partial sums is worth, measured in the same run
        if exec_mode == B.OPTCC_EXEC_COLUMN and not args.no_forward:
            mn = bench.measure(w, k, 5, 3, x=x, execute_only=True, no_forward=1)
            every = roofline_of(EXEC_KERNEL[exec_mode] + "<MODE_F32>, opts.no_forward = 1", exec_mode, w.p, w.n, esize, mn["t_exec"],
                                bench.peak, bench.peak_src)
            every["definition"] = ("the same executor with every flow's two loads and its store issued (no partial sum kept in "
                                   "registers between flows); compulsory DRAM bytes 2 p n sizeof / kernel time")
            stepwise_extra = every
        else:
            stepwise_extra = None

    others = None
    if not args.only_main and world == 1 and args.config == 1:
        m.pop("sess", None)
        sess = None
        del x
        torch.cuda.empty_cache()
        others = {}
        for ci in (0, 2, 3):
            wo = W.config(ci)
            others[wo.name] = bench.summary(bench.measure(wo, BENCH_K[ci], 3, 3))
        x5 = None
        for ell in W.C5_ELLS:      # the whole sweep of configs[4]; the inputs do not depend on ell
            wo = W.config(4, ell)
            if x5 is None:
                x5 = W.all_inputs(wo)
            others[wo.name] = bench.summary(bench.measure(wo, BENCH_K[4], 3, 3, x=x5))
        del x5

    if rank != 0:
        rep.close()
        return 0

    peak, peak_src = bench.peak, bench.peak_src
    kern = EXEC_KERNEL[exec_mode] + ("<MODE_F32>" if w.dtype == W.F32 else "<MODE_BF16>")
    roof = roofline_of(kern, exec_mode, w.p, w.n, esize, t_exec, peak, peak_src)
    traffic, sha, src = ncu_traffic(w.name.split("[")[0], kern)
    roof.update({"traffic": traffic, "traffic_captured_at_commit": sha, "traffic_source": src,
                 "traffic_frac_of_peak": (traffic / t_exec / 1e6 / peak) if traffic else None,
                 "share_of_step": t_exec / t_step})
    mask_final = w.p * w.n * info["mask_bytes"]
    lb = cost0["lb_table1"] / cost0["T0"]
    line = {
        "metric": METRIC, "value": world * w.n * esize / t_step / 1e6, "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": t_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32" if w.dtype == W.F32 else "bf16(f32 accumulate)",
        "data": "synthetic",
        "config": {"workload": workload_name(w, k),
                   "step": "optcc_plan -> {optcc_cost on a second host thread} || {optcc_prepare, optcc_execute, optcc_verify} "
                           "(SURVEY 8(a) a1-a8, all through the C ABI)",
                   "exec_mode": ("auto -> " if args.exec_mode == 0 else "") + EXEC_NAME[exec_mode],
                   "k": "%d: the k at which the modelled T/T0 is within the paper's reported gap of the Table-1 bound" % k,
                   "plan_steps": info["n_steps"], "plan_flows": info["n_flows"],
                   "parallelism": f"replicas x{world} (element-axis shards, no collective)",
                   "l2": "inputs larger than L2 (footprint %.2f GB) and restored from a pristine copy between steps, untimed" % (w.p * w.n * esize / 1e9)},
        "execute_only": {"algbw": world * w.n * esize / t_exec / 1e6, "unit": UNIT, "ms": t_exec},
        "breakdown_ms": m["breakdown_ms"],
        "model": {"T_over_T0": cost0["T_over_T0"], "lb_table1_over_T0": lb, "T_over_lb_table1": cost0["T_over_T0"] / lb,
                  "lb_tight_over_T0": (cost0["lb_tight"] / cost0["T0"]) if cost0["lb_tight"] == cost0["lb_tight"] else None,
                  "paper_closed_form_over_T0": cost0["T_closed_form"] / cost0["T0"], "limit_over_T0": cost0["T_limit"] / cost0["T0"],
                  "bodies": cost0["bodies"], "k": k,
                  "with_14pct_fixed_overhead": 0.14 + 0.86 * cost0["T_over_T0"],   # how the paper plots it (PAPER.md:201 fn.5)
                  "ring_on_degraded_topology_over_T0": cost0["T_ring_degraded"] / cost0["T0"],
                  "r2ccl_closed_form_over_T0": (cost0["T_r2ccl"] / cost0["T0"]) if cost0["T_r2ccl"] == cost0["T_r2ccl"] else None,
                  "paper_context": "SimAI: OPTCC within 2-6% of fault-free NCCL ring at <=50% bandwidth loss; prior work up to 57% (PAPER.md:7)"},
        "roofline": roof,
        "roofline_verify": {"bound": "hbm", "kernel": "%s<masks of %d bits>%s" % (EXEC_KERNEL[exec_mode], 8 * info["mask_bytes"],
                                                                  " (lazy: initial masks are constants, partial sets forwarded in registers, "
                                                                  "final masks checked by their last writer)"
                                                                  if info["lazy_verify"] else " (+init, check)"),
                            "achieved": mask_final / t_ver / 1e6, "peak": peak, "unit": "GB/s", "frac": mask_final / t_ver / 1e6 / peak,
                            "definition": "compulsory DRAM bytes p n mask_bytes (every final mask written once) / kernel time",
                            "ms": t_ver, "share_of_step": t_ver / t_step},
        "parity_spot_check": {"sampled_elements": int(len(idx)), "within_tolerance_and_all_ranks_identical": m["parity_ok"]},
        "clocks": m["clocks"], "gpu_launches": launches_per_step * args.steps, "wall_s_timed_region": m["wall"],
    }
    if stepwise:
        line["roofline_stepwise"] = stepwise
    if stepwise_extra:
        line["roofline_every_load_and_store"] = stepwise_extra
    if others:
        line["other_configs"] = others
    if e2e:
        line["e2e"] = e2e
    if world == 1 and not args.no_cpu_baseline:
        ws = w.scaled(min(w.n, 2 ** (args.cpu_sample_log2 or 24)))
        t = oracle_step(ws, k)
        line["cpu_baseline"] = {"value": ws.n * esize / t / 1e9, "unit": UNIT, "cores": cpu_threads_used(), "kind": "oracle",
                                "sample": f"n={ws.n} elements per rank of the config's n={w.n}, all p={w.p} ranks, every flow; {t:.1f} s",
                                "host_cores": os.cpu_count()}
        if w.dtype == W.F32:      # the same walk compiled (the numpy figure is an interpreter number)
            tc, nthreads = oracle_walk_compiled(ws, k)
            line["cpu_baseline"]["compiled_walk"] = {
                "value": ws.n * esize / tc / 1e9, "unit": UNIT, "cores": nthreads, "kind": "oracle/walk.c",
                "what": "flow walk only (no planning, cost model, masks or fp64 check), gcc -O2 -fopenmp, same sample", "s": tc}
    ok = m["parity_ok"] and (not others or all(o["parity_spot_check"]["within_tolerance_and_all_ranks_identical"] for o in others.values()))
    if not ok:
        line["error"] = "parity spot check failed"
    print(json.dumps(line), flush=True)
    rep.close()
    return 0 if ok else 1


def launch_replicas(args):
    """`bench.py --gpus N` without torchrun: start N workers of this script (one per GPU, NCCL barrier + max over ranks
    as in replicas.py) and hand their output through; rank 0 prints the line with n_gpus = N."""
    from paper_2606_01680_b200.replicas import launch
    return launch(args.gpus, os.path.abspath(__file__), sys.argv[1:])


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        sys.exit(run_reference(a))
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(launch_replicas(a))
    sys.exit(run_native(a))
