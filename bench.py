#!/usr/bin/env python
"""bench.py -- throughput of the batched interior-point hot path (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl jipm|reference]

A "step" is one pass of the whole hot path over one batch of synthetic problems: one jipm_solve_batch call
(Step I for every problem, then fused IPM iterations with iteration-level batching until every problem of the
batch has a final status).  Default workload: BASELINE.json configs[1] (single-quadrotor tracking, batch 4096,
fp64, tol 1e-8).  `value` = SOLVED problems per second with inputs resident in HBM; `e2e` = the same through
jipm_solve_batch_host (pinned host buffers, H2D/D2H inside the timed region).

N > 1 (torchrun): the problem queue is sharded, every rank solves its own batch of the same size (weak scaling),
no collective on the data path; time = max over ranks.

--impl reference times the ORACLE (oracle/, plain numpy fp64) on the host cores on a bounded sample of the same
workload; it is a deliberately slow checker, reported as a baseline, not a target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_26341_b200 import workloads as wl  # noqa: E402

METRIC = "converged NLPs/sec (fp64, tol 1e-8)"
UNIT = "NLPs/s"
WORKLOAD_NAMES = {0: "C0 2-D point-mass NMPC N=10, batch 256",
                  1: "C1 single-quadrotor tracking RK4 N=20 3 obstacles, batch 4096",
                  2: "C2 4-quadrotor collision-free navigation N=20, batch 2048",
                  3: "C3 quadrotor in clutter N=30 32 obstacles, batch 8192",
                  5: "N3 the paper's own vehicle (PAPER.md:174-180): 13-state quaternion quadrotor, dt 0.1, 30 knots, "
                     "sector navigation with 3 obstacles, batch 2000"}


# ---------------------------------------------------------------------------------------------------------
# algorithmic FP64 work per operation of the structured algorithm (flops = 2 per FMA)
# ---------------------------------------------------------------------------------------------------------
def algorithmic_flops(d: wl.Dims) -> dict:
    N, nx, nu, ng, na = d.horizon_N, d.nx, d.nu, d.ng, d.n_agents
    nz, n, m = nx + nu, d.n, d.m
    pd = 2 if d.family == wl.FAM_POINTMASS2D else 3
    # stage-block LDL^T: per stage  T*[A B] (2 nx^2 nz), [A B]^T (T [A B]) (2 nx nz^2,
    # symmetric half counted: nx nz^2), control-block elimination (nu pivots, rank-1 updates of an nz x nz tile:
    # ~ nu nz^2), condensation of the (slack, multiplier) pairs (ng * pd^2 * 2)
    fact = N * (2 * nx * nx * nz + nx * nz * nz + nu * nz * nz + 2 * ng * pd * pd * na)
    # one solve: backward + forward sweeps: T (2 nx^2), [A B] twice (4 nx nz), X/L (2 nx nu + nu^2), x2 passes
    solve = N * 2 * (2 * nx * nx + 4 * nx * nz + 2 * nx * nu + nu * nu) + 8 * (n + m)
    if d.family == wl.FAM_POINTMASS2D:
        fc = N * 12 + (N + 1) * 6 + N * ng * 8
        deriv = fc + 4 * n
    elif d.family == wl.FAM_QUAT_NAV:
        ode = 90   # flops of one evaluation of the polynomial quaternion dynamics
        fc = N * (4 * ode + 13 * 10) + (N + 1) * 9 + N * ng * 10
        # matrix-free chain: 4 RK points x (ode + adjoint product 110) and 17 columns x 4 points x (Jacobian-vector
        # product 100 + contracted-Hessian-vector product 150 + the 17 x 17 accumulation 578)
        deriv = N * (4 * (ode + 110) + 17 * 4 * (100 + 150 + 578)) + 6 * n
    else:
        ode = 110  # flops of one continuous-dynamics evaluation (sincos counted as 2 x 20)
        fc = N * na * (4 * ode + 12 * 10) + (N + 1) * na * 9 + N * ng * 10
        # analytic chain: 4 RK points x (Df entries ~120 + contracted 7x7 Hessian ~250 + adjoint 60) and the 16
        # columns x 4 points x (Df column 60 + Hq v 45 + 7x16 accumulation 224)
        deriv = N * na * (4 * (ode + 120 + 250 + 60) + 16 * 4 * (60 + 45 + 224)) + 6 * n
    resid = 2 * (N * (nz * nz + 2 * nx * nz)) + 12 * (n + m)  # one residual of the unreduced system (6)
    return dict(fact=fact, solve=solve, deriv=deriv, fc=fc, resid=resid)


def flops_from_stats(d: wl.Dims, st: dict) -> float:
    a = algorithmic_flops(d)
    # every KKT solve inside solve_full is paired with one residual evaluation of (6)
    return (st["factorisations"] * a["fact"] + st["kkt_solves"] * (a["solve"] + a["resid"])
            + st["deriv_evals"] * a["deriv"] + st["fc_evals"] * a["fc"])


# ---------------------------------------------------------------------------------------------------------
class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        super().__init__(daemon=True)
        self.gpu, self.rows, self.stop_flag, self.proc = gpu_index, [], False, None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.gpu)], stdout=subprocess.PIPE, text=True)
            for line in self.proc.stdout:
                if self.stop_flag:
                    break
                self.rows.append([c.strip() for c in line.split(",")])
        except Exception:
            pass

    def finish(self) -> dict:
        self.stop_flag = True
        if self.proc is not None:
            self.proc.terminate()
        sm, smax, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[1])); smax.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, col in (("hw_slowdown", 5), ("hw_thermal_slowdown", 6), ("sw_thermal_slowdown", 7),
                              ("sw_power_cap", 8)):
                if len(r) > col and r[col].lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm)}


def _oracle_worker(args):
    cfg, idx, budget_s = args
    os.environ["OMP_NUM_THREADS"] = "1"
    from oracle import families as ofam, ipm as oipm
    d, theta, x0 = wl.generate(cfg, 1, first_id=idx)
    xL, xU = wl.bounds(d)
    prob = ofam.Problem(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt)
    s = oipm.Solver(prob, xL, xU)
    t_end = time.perf_counter() + budget_s
    st = s.initialise(x0[0], theta[0])
    while st.status == oipm.ST_NOT_RUN and time.perf_counter() < t_end:
        s.iterate(st, theta[0])
    return int(st.status), int(st.k)


def time_oracle(cfg: int, first: int, count: int, cores: int, budget_s: float):
    """The oracle as it stands, one problem per process over `cores` host cores.  A problem still running after
    budget_s seconds is cut (status -1: not counted as solved, its iterations are).  Returns (seconds, solved,
    iterations, problems cut)."""
    from multiprocessing import get_context
    t0 = time.perf_counter()
    with get_context("fork").Pool(cores) as pool:
        res = pool.map(_oracle_worker, [(cfg, first + i, budget_s) for i in range(count)], chunksize=1)
    dt = time.perf_counter() - t0
    return dt, sum(1 for s, _ in res if s == 0), sum(k for _, k in res), sum(1 for s, _ in res if s == -1)


# ncu's dram__bytes_read.sum + dram__bytes_write.sum of ONE launch is not measured inside bench.py (it needs the
# profiler): `traffic` is null in the JSON line and `traffic_source` names the committed capture that holds it.
TRAFFIC_SOURCE = {1: "profiles/r2_ncu_full_c1.md"}

# Oracle sample: problems per timed sample and the per-problem time budget, sized for about 20-30 s of wall-clock on the
# box's cores.  C0 / C1 problems finish (1 ms / ~8 s each); a C2 / C3 problem needs minutes (dense 2576 / 2784-row KKT
# factorisations in numpy), so its sample measures ITERATIONS per second and converts with the iterations per converged
# NLP that the GPU arm measured on the same workload (the line says so).
def oracle_sample(cfg: int, cores: int):
    return {0: (256, 30.0), 1: (cores, 25.0), 2: (cores, 20.0), 3: (cores, 20.0), 5: (cores, 25.0)}[cfg]


def golden_iterations_per_solved(cfg: int):
    """tests/golden/full_size_c{cfg}.json (written by the oracle): iterations per converged NLP of the sample."""
    fn = os.path.join(ROOT, "tests", "golden", f"full_size_c{cfg}.json")
    if not os.path.exists(fn):
        return None
    rows = json.load(open(fn))["problems"]
    solved = sum(1 for r in rows if r["status"] == 0)
    return sum(r["iters"] for r in rows) / solved if solved else None


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    cores = os.cpu_count() or 1
    count, budget = oracle_sample(cfg, cores)
    for _ in range(min(args.warmup, 1)):
        time_oracle(cfg, 0, min(count, cores), cores, min(budget, 5.0))
    tot_t, tot_solved, tot_it, tot_cut = 0.0, 0, 0, 0
    for s in range(args.steps):
        dt, solved, its, cut = time_oracle(cfg, 0, count, cores, budget)   # the same ids the GPU arm's sample uses
        tot_t += dt; tot_solved += solved; tot_it += its; tot_cut += cut
    val = tot_solved / tot_t
    sample = (f"first {count} problems of {WORKLOAD_NAMES[cfg]} per step, one process per problem, each cut after "
              f"{budget:.0f} s ({tot_cut} of {count * args.steps} cut)")
    per_solved = golden_iterations_per_solved(cfg)
    if tot_solved == 0 and per_solved:
        val = (tot_it / tot_t) / per_solved
        sample += (f"; no problem finishes inside the budget: value = measured oracle iterations/s / {per_solved:.1f} "
                   "iterations per converged NLP (tests/golden, the oracle's own full solves)")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAMES[cfg], "sample": sample},
            "iterations_per_s": tot_it / tot_t,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def shard_first_id(rank: int, batch_per_gpu: int) -> int:
    """Queue sharding over ranks: rank r owns problem ids [r*P, (r+1)*P) (disjoint; no data-path collective)."""
    return rank * batch_per_gpu


def reduce_over_ranks(times, counts, world: int):
    """Step times: max over ranks; solved / iteration / problem counts: sum over ranks (whole-job aggregate)."""
    import torch.distributed as dist
    if world > 1:
        dist.all_reduce(times, op=dist.ReduceOp.MAX)
        dist.all_reduce(counts, op=dist.ReduceOp.SUM)
    return times, counts


def run_jipm(args):
    import torch
    import torch.distributed as dist
    from paper_2606_26341_b200 import jipm

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (jipm has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = args.config
    P = args.batch or wl.CONFIG_BATCH[cfg]
    d, theta, x0 = wl.generate(cfg, P, first_id=shard_first_id(rank, P))  # queue sharded by rank
    xL, xU = wl.bounds(d)
    opts = None
    if args.max_iter > 0 or args.opt:
        opts = jipm.default_options()
        if args.max_iter > 0:
            opts.max_iter = args.max_iter
        for kv in args.opt:   # option sweeps: not the bench configuration
            key, val = kv.split("=", 1)
            setattr(opts, key, type(getattr(opts, key))(float(val)))
    s = jipm.Solver(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt, xL, xU, opts, resident_slots=args.slots)
    dev = torch.device("cuda", local)
    x0_d = torch.as_tensor(x0, device=dev)
    th_d = torch.as_tensor(theta, device=dev)
    out = dict(x=torch.empty((P, d.n), dtype=torch.float64, device=dev),
               lam=torch.empty((P, d.m), dtype=torch.float64, device=dev),
               zL=torch.empty((P, d.n), dtype=torch.float64, device=dev),
               zU=torch.empty((P, d.n), dtype=torch.float64, device=dev),
               status=torch.empty((P,), dtype=torch.int32, device=dev),
               iters=torch.empty((P,), dtype=torch.int32, device=dev))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2
    # pinned host buffers of the end-to-end leg
    hx0 = torch.as_tensor(x0).pin_memory(); hth = torch.as_tensor(theta).pin_memory()
    hout = dict(x=torch.empty((P, d.n), dtype=torch.float64).pin_memory(),
                lam=torch.empty((P, d.m), dtype=torch.float64).pin_memory(),
                zL=torch.empty((P, d.n), dtype=torch.float64).pin_memory(),
                zU=torch.empty((P, d.n), dtype=torch.float64).pin_memory(),
                status=torch.empty((P,), dtype=torch.int32).pin_memory(),
                iters=torch.empty((P,), dtype=torch.int32).pin_memory())
    hnp = {k: v.numpy() for k, v in hout.items()}
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        s.solve_batch_into(x0_d, th_d, out)
    peak_fp64 = jipm.fp64_peak_tflops()  # roofline denominator measured on this GPU, outside the timed region
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    # ---- timed region: K steps, device-resident inputs, CUDA events on the launching stream -------------
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    stats_sum = {}
    t_wall0 = time.perf_counter()
    for a, b in ev:
        flush.fill_(1)  # L2 flush between timed iterations (not inside an event pair)
        a.record(stream)
        s.solve_batch_into(x0_d, th_d, out)
        b.record(stream)
        for k, v in s.stats().items():
            stats_sum[k] = stats_sum.get(k, 0) + v
    barrier()
    t_wall = time.perf_counter() - t_wall0
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)
    clocks = sampler.finish() if rank == 0 else None
    status = out["status"].cpu().numpy()
    iters = out["iters"].cpu().numpy()
    solved = int((status == 0).sum())
    # ---- end-to-end leg: host buffers through jipm_solve_batch_host -------------------------------------
    s.solve_batch_host(hx0.numpy(), hth.numpy(), hnp)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        s.solve_batch_host(hx0.numpy(), hth.numpy(), hnp)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_solved = int((hnp["status"] == 0).sum())
    # ---- reduce over ranks ---------------------------------------------------------------------------------
    red = torch.tensor([dev_ms, e2e_s, t_wall], dtype=torch.float64, device=dev)
    cnt = torch.tensor([solved, e2e_solved, int(iters.sum()), P], dtype=torch.float64, device=dev)
    reduce_over_ranks(red, cnt, world)
    dev_ms, e2e_s, t_wall = red.tolist()
    solved_all, e2e_solved_all, iters_all, P_all = cnt.tolist()
    if rank == 0:
        K = args.steps
        secs = dev_ms * 1e-3
        value = solved_all * K / secs
        flops = flops_from_stats(d, stats_sum)  # rank 0's launches
        cyc_it = max(stats_sum.get("cyc_iterations", 0), 1)
        phase_share = {k[4:]: round(stats_sum[k] / cyc_it, 4) for k in
                       ("cyc_derivs", "cyc_factor", "cyc_solve", "cyc_residual", "cyc_trial_eval")}
        phase_share.update({"factor/" + k[5:]: round(stats_sum[k] / cyc_it, 4) for k in stats_sum if k.startswith("cycf_")
                            and stats_sum[k] > 0})
        # overlapping views: whole blocks of the iteration (they contain the solves / evaluations counted above)
        phase_share.update({"block/" + k[5:]: round(stats_sum[k] / cyc_it, 4) for k in stats_sum if k.startswith("cycx_")})
        phase_share["block/speculative_trials"] = round(stats_sum.get("cyc_speculative_trials", 0) / cyc_it, 4)
        us_per_iter = cyc_it / max(stats_sum["iterations"], 1) / (clocks["sm_mhz"] or 1965.0) if clocks else None
        my_secs = sum(a.elapsed_time(b) for a, b in ev) * 1e-3
        achieved = flops / my_secs / 1e12
        hist = {int(k): int((status == k).sum()) for k in np.unique(status)}
        h2d = (x0.nbytes + theta.nbytes)
        d2h = sum(v.nbytes for v in hnp.values())
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": dev_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_NAMES[cfg], "batch_per_gpu": P, "n": d.n, "m": d.m,
                       "resident_slots": s.stats()["slots"], "l2": "flushed between timed steps (256 MiB fill)",
                       **({"max_iter_cap": args.max_iter, "note": "profiling run, not a bench value"}
                          if args.max_iter > 0 else {}),
                       **({"option_overrides": list(args.opt), "note": "option sweep, not a bench value"} if args.opt else {}),
                       "parallelism": f"queue sharded over {world} GPU(s), no collective"},
            "iterations_per_s": iters_all * K / secs,
            "slot_us_per_iteration": us_per_iter,
            "converged_fraction": solved_all / P_all,
            "iters_mean": float(iters.mean()), "iters_max": int(iters.max()),
            "iters_percentiles_50_90_99": [float(v) for v in np.percentile(iters, [50, 90, 99])],
            "status_hist_rank0": hist,
            "wall_s_timed_region": t_wall,
            "e2e": {"value": e2e_solved_all * K / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h},
            "gpu_launches": int(stats_sum["launches"]),
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_fp64, "unit": "TFLOP/s",
                         "frac": achieved / peak_fp64,
                         "traffic": None,
                         "traffic_source": TRAFFIC_SOURCE.get(cfg, "not captured for this config"),
                         "algorithmic_bytes_per_launch": h2d + d2h,
                         "kernel": "jipm_slot_kernel (persistent, one launch per step)",
                         "peak_source": "DFMA microbenchmark jipm_bench_fp64_peak measured in this run "
                                        "(MEASURED_PEAKS.json has no FP64 entry); nominal 148 SM x 64 DFMA/clk x 2 x "
                                        "1.965 GHz = 37.2",
                         "algorithmic_flops_per_step": flops / K,
                         "counts_per_step": {k: v / K for k, v in stats_sum.items() if not k.startswith("cyc")},
                         "phase_share_of_iteration_cycles": phase_share,
                         "slot_us_per_iteration": us_per_iter},
            "clocks": clocks,
        }
        if not args.no_cpu_baseline and world == 1:
            cores = os.cpu_count() or 1
            cnt_o, budget = oracle_sample(cfg, cores)
            dt, so, it, cut = time_oracle(cfg, 0, cnt_o, cores, budget)
            sample = (f"first {cnt_o} problems of the same workload, one process per problem, each cut after "
                      f"{budget:.0f} s ({cut} cut); bounded to about {budget:.0f} s of wall-clock on {cores} cores "
                      "(SURVEY 8(d)'s 512 / 64 problems would take minutes per line)")
            val = so / dt
            if so == 0 and solved_all > 0:
                per_solved = iters_all / solved_all
                val = (it / dt) / per_solved
                sample += (f"; no problem finishes inside the budget: value = measured oracle iterations/s / "
                           f"{per_solved:.1f} iterations per converged NLP measured by the GPU arm on this workload")
            line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "iterations_per_s": it / dt, "sample": sample}
        print(json.dumps(line))
    s.close()
    if world > 1:
        dist.destroy_process_group()


def run_c4(args):
    """BASELINE.json configs[4]: iteration-level batching sweep on "the config-2 problem family" -- ambiguous (reading
    D-2): --c4-family 1 = the single-quadrotor family of configs[1] (1-based reading), --c4-family 2 = the four-quadrotor
    family of configs[2] (0-based reading).  A queue of seeded problems is solved with R = 1024, 4096, 16384, 65536
    problem slots.  A slot is a CTA: R CTAs are launched, the SMs hold as many as fit (co_resident_slots below) and every
    CTA pops problems until the queue is empty, so a finished problem is replaced at once whatever R is; the global
    scratch is sized for the co-resident CTAs only."""
    import torch
    from paper_2606_26341_b200 import jipm
    torch.cuda.set_device(0)
    fam = args.c4_family
    P = args.queue or (100000 if fam == 1 else 20000)
    d, theta, x0 = wl.generate(fam, P)
    xL, xU = wl.bounds(d)
    dev = torch.device("cuda", 0)
    x0_d, th_d = torch.as_tensor(x0, device=dev), torch.as_tensor(theta, device=dev)
    out = dict(x=torch.empty((P, d.n), dtype=torch.float64, device=dev),
               lam=torch.empty((P, d.m), dtype=torch.float64, device=dev),
               status=torch.empty((P,), dtype=torch.int32, device=dev),
               iters=torch.empty((P,), dtype=torch.int32, device=dev))
    peak = jipm.fp64_peak_tflops()
    sm_count = torch.cuda.get_device_properties(0).multi_processor_count
    sweep, ref_iters, co_res = [], None, None
    for R in [int(r) for r in args.slots_list.split(",")]:
        s = jipm.Solver(d.family, d.horizon_N, d.n_agents, d.n_obstacles, d.dt, xL, xU, resident_slots=R)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); s.solve_batch_into(x0_d, th_d, out); b.record(); torch.cuda.synchronize()
        ms = a.elapsed_time(b)
        st = s.stats()
        co_res = st["co_resident_slots"]
        iters = out["iters"].cpu().numpy(); status = out["status"].cpu().numpy()
        if ref_iters is None:
            ref_iters = iters.copy()
        busy = (st["cyc_iterations"] + st["cyc_init"]) / 1.965e9
        pct = np.percentile(iters, [50, 90, 99, 99.9]).tolist()
        hist_it = np.bincount(np.minimum(iters, 3000) // 25, minlength=121).tolist()
        sweep.append({"R": R, "ms": ms, "nlps_per_s": float((status == 0).sum()) / (ms * 1e-3),
                      "iterations_per_s": float(iters.sum()) / (ms * 1e-3),
                      "slot_occupancy": busy / (min(R, co_res) * ms * 1e-3),
                      "fp64_frac": flops_from_stats(d, st) / (ms * 1e-3) / 1e12 / peak,
                      "iters_identical_to_first_R": bool(np.array_equal(iters, ref_iters)),
                      "iters_p50_p90_p99_p999": pct, "iters_max": int(iters.max()),
                      "iters_histogram_bins_of_25": hist_it,
                      "status_hist": {int(k): int((status == k).sum()) for k in np.unique(status)}})
        s.close()
    best = max(sweep, key=lambda r: r["nlps_per_s"])
    print(json.dumps({"metric": METRIC, "value": best["nlps_per_s"], "unit": UNIT, "n_gpus": 1, "steps": 1, "warmup": 0,
                      "ms_per_step": best["ms"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                      "dtype": "f64", "data": "synthetic",
                      "config": {"workload": f"C4 iteration-level batching sweep, queue of {P} problems of the "
                                             f"C{fam} family ({WORKLOAD_NAMES[fam].split(',')[0]})",
                                 "co_resident_slots": co_res, "sm_count": sm_count}, "sweep": sweep}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3, 4, 5])
    ap.add_argument("--queue", type=int, default=0, help="config 4: problems in the queue (default 100000 for the C1 "
                                                         "family, 20000 for the C2 family)")
    ap.add_argument("--c4-family", type=int, default=1, choices=[1, 2], help="config 4: which reading of 'the config-2 "
                                                                            "problem family' (D-2)")
    ap.add_argument("--slots-list", default="1024,4096,16384,65536", help="config 4: resident slot counts")
    ap.add_argument("--batch", type=int, default=0, help="problems per GPU per step (default: the config's batch)")
    ap.add_argument("--slots", type=int, default=0, help="resident slots (0: library picks)")
    ap.add_argument("--impl", default="jipm", choices=["jipm", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="override one solver option (repeatable), e.g. --opt watchdog_trigger=0: option sweeps only")
    ap.add_argument("--max-iter", type=int, default=0,
                    help="cap IPM iterations per problem (profiling runs only: keeps the kernel short under ncu; "
                         "a line produced with this flag says so in config and is not a bench value)")
    args = ap.parse_args()
    if args.config == 4:
        run_c4(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_jipm(args)


if __name__ == "__main__":
    main()
