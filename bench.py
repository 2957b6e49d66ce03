#!/usr/bin/env python
"""bench.py -- the treecode BEM matvec of Eq. (5) on seeded synthetic input, timed on the
configuration BASELINE.json's metric belongs to: configs[4] (C4: 20,000 atoms, ~1.04 M panels, K = 7,
theta = 0.5, P = 6), the largest single-GPU configuration.

  step     = one pass of the matvec hot path over one vector x resident in HBM:
             k_weights -> {k_p2p2  ||  k_upward (P2M, M2M, M->F) -> k_m2p2} -> k_combine.
  value    = interactions evaluated per second over the timed steps, SURVEY section 8(d)'s unit: one P2P
             interaction = one (target collocation point, source Gauss point) pair producing all four kernels of
             Eq. (3)-(4); one M2P interaction = one (target, cell) pair producing all four order-P sums.  Both
             counts come from the stored lists (pb_get_stats) and are reported separately under "evaluated";
             "direct_equivalent_per_s" = N * N_s / time (the pairs the dense operator accounts for) is a side key.
             The count depends on the lists: with pb_params.list_split = 1 (default; the two 32-target halves of a group
             decided separately) one C4 matvec evaluates 25 % fewer interactions than with one decision per group and
             takes 8 % less time, so `value` falls while ms_per_step and direct_equivalent_per_s improve; --list-split 0
             gives the other lists.
  e2e      = the same step through pb_matvec_host: x copied from pinned host memory, y copied back, every step.
  roofline = both hot kernels, FP64 ALU bound.  Per kernel: (i) algorithmic flop (80 per P2P pair;
             4 N_T + N_k + 6 P + 30 per M2P pair at the order it is evaluated at) / CUDA-event time / measured
             DFMA peak, and (ii) executed FP64-pipe instructions (ncu, profiles/r02_counters.csv) / time /
             (148 SM x 64 lanes x SM clock).  "frac" is (i) for the kernel with the larger share of the step.
  solve    = one full polarizable solve (vacuum SCF, RHS, GCR / flexible GMRES, reaction field, SOR to 1e-7 D, energies),
             timed after the matvec steps on its second call (the first, also reported, builds the site-side lists); "configs" = the solve times of C1, C2 and the C3 binding triple.
  cpu_baseline = the oracle's direct O(N^2 K) sum on this box's host cores on sampled target rows.

python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl reference]
N > 1 (torchrun): target-leaf sharding of ONE matvec across the ranks: every rank owns a
contiguous Morton range of target groups, x is all-gathered (NCCL) before the step's kernels and the owned rows of y
after them; "scaling": "strong".
"""
import argparse
import csv
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "treecode_matvec_interactions_per_s"
UNIT = "interactions/s"
# Algorithmic FP64 work per unit: one P2P pair = the four kernels of
# Eq. (3)-(4) for one (target, Gauss point) pair; one M2P pair at order P = 4*NT + Nk + 6P + 30.
P2P_FLOP_PER_PAIR = 80.0
FP64_LANES = 148 * 64                                  # SMs x FP64 FMA lanes (B200_PROFILING.md unit counts)
FP64_NOMINAL_TFLOPS = FP64_LANES * 2 * 1.965e9 / 1e12  # x 2 flop x max SM clock
COUNTERS_CSV = os.path.join(ROOT, "profiles", "r02_counters.csv")


def n_terms_of(P):
    return sum((P - a - b - c) // 2 + 1 for a in range(P + 1) for b in range(P + 1 - a) for c in range(P + 1 - a - b))


def m2p_flop_per_pair(P, n_terms=None):
    nk = (P + 1) * (P + 2) * (P + 3) // 6
    return 4.0 * (n_terms if n_terms is not None else n_terms_of(P)) + nk + 6.0 * P + 30.0


def m2p_flop(P, st):
    """Algorithmic flop of one M2P launch: every pair at the order it is evaluated at -- P, or P - 1 / P - 2 for the pairs
    the list build flagged (R-30)."""
    low, mid = st.get("m2p_pairs_low", 0), st.get("m2p_pairs_mid", 0)
    return (m2p_flop_per_pair(P, st["n_terms"]) * (st["m2p_pairs"] - low - mid) + (m2p_flop_per_pair(P - 2) * low if low else 0.0)
            + (m2p_flop_per_pair(P - 1) * mid if mid else 0.0))


def load_counters(workload, theta, P, ncrit):
    """Per-launch ncu counters of the hot kernels for this workload and launch configuration, from the committed
    capture profiles/r02_counters.csv (written from `ncu --set full`, command in profiles/r02_counters.md):
    kernel -> dict(dram_bytes, fp64_thread_inst, pairs).  Missing file or row -> empty; a row whose pair count
    differs from this run's lists is ignored by the caller (the counters belong to another list build)."""
    out = {}
    try:
        with open(COUNTERS_CSV) as fh:
            for row in csv.DictReader(r for r in fh if not r.startswith("#")):
                if (row["workload"] == workload and abs(float(row["theta"]) - theta) < 1e-12 and int(row["order_P"]) == P
                        and int(row["ncrit"]) == ncrit):
                    out[row["kernel"]] = dict(dram_bytes=float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]),
                                              fp64_thread_inst=32.0 * float(row["fp64_warp_inst"]), pairs=int(row["pairs"]),
                                              source=row["source"])
    except (OSError, KeyError, ValueError):
        pass
    return out


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.samples = []
        self.stop_flag = threading.Event()

    def run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i",
                                      str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
                f = [s.strip() for s in out.split(",")]
                if len(f) >= 6:
                    self.samples.append(f)
            except Exception:
                pass
            self.stop_flag.wait(0.1)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(float(s[0]) for s in self.samples)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(s[2 + k].lower().startswith("active") for s in self.samples)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.samples[0][1]), "reasons": reasons,
                "samples": len(sm)}


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def max_over_ranks(value, world, device=None):
    """Max of a python float over ranks (identity when world == 1).  gloo or nccl."""
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, world, device=None):
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def load_workload(name):
    from paper_1810_03698_b200.workloads import make_config
    if name.startswith("C3-"):
        return make_config("C3", which=name[3:])
    return make_config(name)


# ---- the oracle on the host cores (cpu_baseline, --impl reference) ----------------------------------------------
def oracle_rows(n, count, seed=8):
    import numpy as np
    return np.sort(np.random.Generator(np.random.PCG64(seed)).choice(n, size=min(count, n), replace=False))


def oracle_setup(w, rows_per_call):
    import numpy as np
    from oracle import pb_oracle as po
    po.build()
    orc = po.Oracle(w.verts, w.tris, po.Params(K_far=w.params["K_far"]))
    n = orc.nt
    x = np.random.Generator(np.random.PCG64(7)).normal(size=2 * n)
    rows = None if rows_per_call >= n else oracle_rows(n, rows_per_call)
    nrows = n if rows is None else int(rows.size)
    pairs = float(nrows) * n * w.params["K_far"]          # (target, Gauss point) pairs of one call, all four kernels each
    what = (f"the oracle's direct O(N^2 K) sum of Eq. (5) on {w.name}: "
            + (f"{nrows} seeded sampled target rows against all {n * w.params['K_far']} source points"
               if rows is not None else f"all {n} target rows"))
    return po, orc, x, rows, pairs, what


def oracle_matvec_rate(w, rows_per_call=256, budget_s=12.0):
    """The oracle as it stands, timed for about `budget_s` seconds."""
    po, orc, x, rows, pairs, what = oracle_setup(w, rows_per_call)
    orc.matvec(x, rows)                            # warm-up (thread pool, page faults)
    t0 = time.perf_counter()
    reps = 0
    while True:
        orc.matvec(x, rows)
        reps += 1
        el = time.perf_counter() - t0
        if el > budget_s or reps >= 50:
            break
    n = orc.nt
    rate = pairs * reps / el
    return dict(value=rate, unit=UNIT, cores=po.num_threads(), kind="oracle",
                sample=f"{reps} x {what}, {el:.1f} s; P2P interactions only (the oracle has no far field)",
                ms_per_call=1e3 * el / reps,
                full_matvec_seconds_extrapolated=float(n) * n * w.params["K_far"] / rate)


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    w = load_workload(args.workload)
    po, orc, x, rows, pairs, what = oracle_setup(w, args.ref_rows)
    for _ in range(args.warmup):
        orc.matvec(x, rows)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.matvec(x, rows)
    el = time.perf_counter() - t0
    val = pairs * args.steps / el
    sample = f"each step = {what}"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "panels": int(orc.nt), "K_far": int(w.params["K_far"]), "what": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": po.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ---- our arm ---------------------------------------------------------------------------------------------------------
def timed_solve(pb, torch, name, dev_index, repeats=1, warm=0):
    """One polarizable solve of a workload on resident inputs (mesh, sites, tree already built): seconds, result."""
    w = load_workload(name)
    ctx = pb.from_workload(w, dev_index)
    ctx.tree_build()
    for _ in range(warm):
        ctx.solve()
    torch.cuda.synchronize()
    best, res = None, None
    for _ in range(repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _, _, res = ctx.solve()
        e1.record()
        e1.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None or ms < best else best
    st = ctx.stats()
    ctx.close()
    return best, res, st


def run_ours(args):
    import numpy as np
    import torch
    rank, local_rank, world = dist_env()
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    from paper_1810_03698_b200 import pb
    pb.lib()                                       # fails loudly if the CUDA library is missing

    if args.workload == "C3-triple":               # the binding triple's three independent problems, one per rank (replicas)
        args.replicas = True
        args.workload = ("C3-complex", "C3-receptor", "C3-ligand")[rank % 3]
    w = load_workload(args.workload)
    names = {k for k, _ in pb.Params._fields_}
    prm = {k: v for k, v in w.params.items() if k in names}
    if args.theta is not None:
        prm["theta"] = args.theta
    if args.order is not None:
        prm["order_P"] = args.order
    if args.ncrit is not None:
        prm["ncrit"] = args.ncrit
    if args.list_split is not None:
        prm["list_split"] = args.list_split
    if args.scf_recycle is not None:
        prm["scf_recycle"] = args.scf_recycle
    if args.scf_eta is not None:
        prm["scf_eta"] = args.scf_eta
    ctx = pb.PB(local_rank, **prm)
    s = w.sites
    ctx.mesh_load(w.verts, w.tris)
    ctx.sites_load(s["pos"], s["q"], s["dip"], s["quad"], s["alpha"], s["group"])
    if world > 1 and not args.replicas:
        ctx.set_shard(rank, world)                 # owned Morton range of target groups; all-gather of y's owned rows per matvec
    ctx.tree_build()
    nt, na = int(w.tris.shape[0]), int(s["pos"].shape[0])
    f64 = torch.float64
    x_np = np.random.Generator(np.random.PCG64(7)).normal(size=2 * nt)
    x_host = torch.from_numpy(x_np).pin_memory()
    y_host = torch.empty(2 * nt, dtype=f64).pin_memory()
    x = x_host.to(dev)
    y = torch.empty_like(x)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def step_resident():
        ctx.matvec(x, out=y)                       # sharded: owned rows, then one all-gather of them (NCCL) and the un-permute

    def step_e2e():
        ctx.matvec_host(x_host, y_host)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps):
        tot_ms = 0.0
        for _ in range(steps):
            flush.zero_()                          # L2 flush, outside the event pair
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            e1.synchronize()
            tot_ms += e0.elapsed_time(e1)
        return tot_ms

    sharded = world > 1 and not args.replicas
    W = max(args.warmup, 3)
    for _ in range(W):
        step_resident()
    if world == 1:
        step_e2e()
    sampler = ClockSampler(local_rank)
    sampler.start()
    st0 = ctx.stats()
    barrier()
    if args.profiler_range:                        # ncu --profile-from-start off captures exactly the timed steps
        torch.cuda.profiler.start()
    ms_total = timed(step_resident, args.steps)
    if args.profiler_range:
        torch.cuda.synchronize()
        torch.cuda.profiler.stop()
    barrier()
    st1 = ctx.stats()
    ms_e2e = timed(step_e2e, args.steps) if world == 1 else 0.0
    barrier()
    # Kernel durations for the roofline: the SAME steps once more with a CUDA-event pair around every P2P and M2P
    # launch on the stream they are launched on.  In this mode the library runs the matvec's two branches back to
    # back on one stream (in the timed steps above the far-field branch overlaps P2P on a second stream), so each
    # pair brackets exactly one kernel; grids, blocks and data are identical.
    ctx.set_profiling(True)
    ms_prof = timed(step_resident, args.steps)
    stp = ctx.stats()
    ctx.set_profiling(False)
    barrier()
    sampler.stop_flag.set()
    sampler.join(timeout=2)
    clocks = sampler.summary()

    ms_total = max_over_ranks(ms_total, world, dev)
    P = int(ctx.get_params().order_P)
    theta = float(ctx.get_params().theta)
    # sharded: pb_stats counts the owned groups' pairs, the job's are the sum over ranks; replicas: every rank does all of them
    p2p_pairs = sum_over_ranks(float(st1["p2p_pairs"]), world, dev)
    m2p_pairs = sum_over_ranks(float(st1["m2p_pairs"]), world, dev)
    evald_per_mv = p2p_pairs + m2p_pairs
    inter_per_mv = float(nt) * float(st1["n_sources"])          # the N x N_s pairs one matvec accounts for
    value = evald_per_mv * args.steps / (ms_total * 1e-3)
    launches = st1["kernel_launches"] - st0["kernel_launches"]

    # ---- roofline of both hot kernels
    peak_probe = ctx.fp64_peak_probe()                          # measured DFMA throughput of this GPU, TFLOP/s
    sm_hz = (clocks["sm_mhz"] or 1965.0) * 1e6
    inst_peak = FP64_LANES * sm_hz                              # FP64 lane-instructions per second at the sampled clock
    counters = load_counters(w.name, theta, P, int(st1["ncrit_used"]))
    p2p_kernel = "k_p2p2" if nt >= 30000 else "k_p2p"
    m2p_kernel = "k_m2p2" if P <= 8 else "k_m2p"
    p2p_ms = stp["prof_p2p_ms"] / max(stp["prof_p2p_launches"], 1)
    m2p_ms = stp["prof_m2p_ms"] / max(stp["prof_m2p_launches"], 1)

    def kernel_entry(kname, ms, nlaunch, pairs, flop):
        c = counters.get(kname, {})
        if c and c["pairs"] != int(pairs):
            c = {}                                 # counters of another list build: not this run's kernel
        e = {"kernel": kname, "ms_per_launch": ms, "launches": int(nlaunch), "pairs_per_launch": int(pairs),
             "algorithmic_tflops": flop / (ms * 1e-3) / 1e12 if ms > 0 else 0.0,
             "share_of_step": ms * nlaunch / ms_prof if ms_prof > 0 else None}
        e["frac_algorithmic"] = e["algorithmic_tflops"] / peak_probe if peak_probe > 0 else None
        if c and ms > 0:
            e["fp64_inst_per_pair"] = c["fp64_thread_inst"] / pairs if pairs else None
            e["frac_inst"] = c["fp64_thread_inst"] / (ms * 1e-3) / inst_peak
            e["dram_bytes_per_launch"] = c["dram_bytes"]
            e["counters_source"] = c["source"]
        else:
            e["fp64_inst_per_pair"] = e["frac_inst"] = e["dram_bytes_per_launch"] = None
        return e

    e_p2p = kernel_entry(p2p_kernel, p2p_ms, stp["prof_p2p_launches"], st1["p2p_pairs"], P2P_FLOP_PER_PAIR * st1["p2p_pairs"])
    e_m2p = kernel_entry(m2p_kernel, m2p_ms, stp["prof_m2p_launches"], st1["m2p_pairs"], m2p_flop(P, st1))
    dom = e_p2p if stp["prof_p2p_ms"] >= stp["prof_m2p_ms"] else e_m2p
    roofline = {"bound": "alu", "kernel": dom["kernel"], "achieved": dom["algorithmic_tflops"], "peak": peak_probe,
                "unit": "TFLOP/s", "frac": dom["frac_algorithmic"], "frac_inst": dom["frac_inst"],
                "traffic": dom["dram_bytes_per_launch"],
                "peak_source": "pb_fp64_peak_probe, measured in this run (independent DFMA chains); nominal "
                               "148 SM x 64 lanes x 2 x 1.965 GHz = %.1f TFLOP/s (MEASURED_PEAKS.json has no FP64 "
                               "figure); frac_inst = executed FP64-pipe lane-instructions (ncu) / time / "
                               "(148 x 64 x sampled SM clock)" % FP64_NOMINAL_TFLOPS,
                "timed_in": "a repeat of the timed steps with a CUDA-event pair around every P2P and M2P launch on the "
                            "launching stream (branches serialised): %.3f ms per step against %.3f ms with the far-field "
                            "branch overlapped" % (ms_prof / args.steps, ms_total / args.steps),
                "p2p": e_p2p, "m2p": e_m2p}
    if rank != 0:
        ctx.close()
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()
        return

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong" if sharded else "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "panels": nt, "gauss_points": int(st1["n_sources"]), "sites": na,
                   "theta": theta, "order_P": P, "ncrit": int(st1["ncrit_used"]), "K_far": int(w.params["K_far"]),
                   "list_split": int(ctx.get_params().list_split),
                   "step": "one treecode matvec of Eq. (5) on a resident vector",
                   "l2": "flushed between steps (256 MiB device write, outside the event pairs); the step's own "
                         "inputs (0.46 GB source records, 1.3 GB near table at C4) exceed the 126 MB L2",
                   "parallelism": "1 GPU" if world == 1 else (f"target groups of one matvec sharded over {world} GPUs, one NCCL all-gather "
                                                                 f"of y's owned rows per step" if sharded else f"{world} replicas")},
        "evaluated": {"p2p_pairs_per_matvec": int(p2p_pairs), "m2p_pairs_per_matvec": int(m2p_pairs),
                      "m2p_pairs_at_order_P_minus_2": int(sum_over_ranks(float(st1["m2p_pairs_low"]), world, dev)) if world == 1 else None,
                      "m2p_pairs_at_order_P_minus_1": int(st1["m2p_pairs_mid"]) if world == 1 else None,
                      "p2p_pairs_for_one_half_of_a_group": int(st1["p2p_pairs_half"]) if world == 1 else None,
                      "m2p_pairs_for_one_half_of_a_group": int(st1["m2p_pairs_half"]) if world == 1 else None,
                      "covered_pairs": int(st1["covered_pairs"]), "covered_equals_N_x_Ns": bool(st1["covered_pairs"] == int(inter_per_mv)) if world == 1 else None,
                      "direct_equivalent_per_s": inter_per_mv * (1 if sharded or world == 1 else world) * args.steps / (ms_total * 1e-3)},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "clocks": clocks,
    }
    if world == 1:
        line["e2e"] = {"value": evald_per_mv * args.steps / (ms_e2e * 1e-3), "unit": UNIT,
                       "h2d_bytes_per_step": int(x_host.numel() * 8), "d2h_bytes_per_step": int(y_host.numel() * 8),
                       "ms_per_step": ms_e2e / args.steps, "api": "pb_matvec_host"}
    else:
        line["e2e"] = None
    # ---- the second half of the metric: time per polarizable PB solve
    if world == 1 and not args.no_solve:
        # like the C1-C3 solves below: one untimed call first (it also builds, once, the site-side lists of the RHS and
        # reaction-field treecodes and allocates the solver workspace), then the timed one; both are reported
        times = []
        for _ in range(2):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            _, _, res = ctx.solve()
            e1.record()
            e1.synchronize()
            times.append(e0.elapsed_time(e1) * 1e-3)
        line["solve"] = {"workload": w.name, "time_per_polarizable_solve_s": times[1], "first_call_s": times[0], "runs": 2,
                         "dG_solv_kcal_mol": res["dG_solv"], "scf_iters": res["scf_iters"], "gmres_iters": res["gmres_iters_total"],
                         "matvecs": res["matvecs_total"], "final_gmres_relres": res["final_gmres_relres"],
                         "final_scf_delta_debye": res["final_scf_delta_debye"], "status": res["status"],
                         "scf_recycle": int(ctx.get_params().scf_recycle), "scf_eta": float(ctx.get_params().scf_eta)}
    ctx.close()
    if world == 1 and not args.no_configs:
        cfgs = {}
        for name in ("C1", "C2", "C3-complex", "C3-receptor", "C3-ligand"):
            ms, res, st = timed_solve(pb, torch, name, local_rank, repeats=3 if name in ("C1", "C2") else 1, warm=1)
            cfgs[name] = {"panels": int(st["n_panels"]), "sites": int(st["n_sites"]), "solve_ms": ms, "dG_solv_kcal_mol": res["dG_solv"],
                          "scf_iters": res["scf_iters"], "matvecs": res["matvecs_total"], "status": res["status"]}
        cfgs["C3-ddG_bind_kcal_mol"] = (cfgs["C3-complex"]["dG_solv_kcal_mol"] - cfgs["C3-receptor"]["dG_solv_kcal_mol"]
                                         - cfgs["C3-ligand"]["dG_solv_kcal_mol"])
        line["configs"] = cfgs
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = oracle_matvec_rate(w, rows_per_call=args.ref_rows)
    print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def run_sweep(args):
    """BASELINE configs[4]: matvec throughput over theta x P on one workload (default C4), each with its
    error on seeded sampled rows against the oracle's direct sum, then one full polarizable solve at the
    workload's own theta, P.  One JSON line per case; not the driver's bench line."""
    import numpy as np
    import torch
    from paper_1810_03698_b200 import pb
    from oracle import pb_oracle as po
    torch.cuda.set_device(0)
    w = load_workload(args.workload)
    nt = int(w.tris.shape[0])
    x = np.random.Generator(np.random.PCG64(7)).normal(size=2 * nt)
    rows = np.sort(np.random.Generator(np.random.PCG64(8)).choice(nt, size=min(args.sweep_rows, nt), replace=False))
    po.build()
    orc = po.Oracle(w.verts, w.tris, po.Params(K_far=w.params["K_far"]))
    t0 = time.perf_counter()
    y1, y2 = orc.matvec(x, rows)
    t_or = time.perf_counter() - t0
    yref = np.concatenate([y1, y2])
    print(json.dumps({"case": "oracle", "workload": w.name, "panels": nt, "rows": int(rows.size), "seconds": t_or,
                      "cores": po.num_threads(), "pairs_per_s": float(rows.size) * nt * w.params["K_far"] / t_or}), flush=True)
    ctx = pb.from_workload(w)
    xd = torch.from_numpy(x).cuda()
    y = torch.empty_like(xd)
    idx = torch.from_numpy(np.concatenate([rows, nt + rows])).cuda()
    cases = set(args.sweep_cases.split(","))
    peak = None
    for theta in (0.3, 0.5, 0.7):
        for P in (4, 6, 8):
            if "matvec" not in cases:
                break
            ctx.set_params(theta=theta, order_P=P)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); ctx.tree_build(); e1.record(); e1.synchronize()
            t_build = e0.elapsed_time(e1)
            if peak is None:
                peak = ctx.fp64_peak_probe()
            for _ in range(3):
                ctx.matvec(xd, out=y)
            ts = []
            for _ in range(5):
                e0.record(); ctx.matvec(xd, out=y); e1.record(); e1.synchronize()
                ts.append(e0.elapsed_time(e1))
            ms = sorted(ts)[len(ts) // 2]
            ctx.matvec(xd, out=y, timed=True)
            st = ctx.stats()
            lm = st["last_matvec_ms"]
            got = y[idx].cpu().numpy()
            err = float(np.linalg.norm(got - yref) / np.linalg.norm(yref))
            print(json.dumps({
                "case": "matvec", "workload": w.name, "theta": theta, "order_P": P, "ncrit": int(st["ncrit_used"]),
                "ms_per_matvec": ms, "tree_build_ms": t_build,
                "interactions_per_s": (st["p2p_pairs"] + st["m2p_pairs"]) / (ms * 1e-3),
                "direct_equivalent_per_s": float(nt) * st["n_sources"] / (ms * 1e-3),
                "p2p_pairs": int(st["p2p_pairs"]), "m2p_pairs": int(st["m2p_pairs"]),
                "covered_equals_N_x_Ns": bool(st["covered_pairs"] == nt * st["n_sources"]),
                "serial_ms": {k: lm[k] for k in ("weights", "p2m_m2m", "m2p", "p2p", "near_combine")},
                "p2p_tflops": P2P_FLOP_PER_PAIR * st["p2p_pairs"] / (lm["p2p"] * 1e-3) / 1e12,
                "m2p_pairs_low_order": int(st["m2p_pairs_low"]), "m2p_pairs_mid_order": int(st["m2p_pairs_mid"]),
                "m2p_tflops": m2p_flop(P, st) / (lm["m2p"] * 1e-3) / 1e12 if lm["m2p"] > 0 else 0.0,
                "fp64_peak_tflops_measured": peak, "rel_l2_vs_oracle_rows": err, "device_gb": st["device_bytes"] / 1e9}), flush=True)
    ctx.set_params(**{k: v for k, v in w.params.items() if k in ("theta", "order_P")})
    ctx.tree_build()
    if "gmres" in cases:
        # the Krylov vector kernels at this size (HBM-bound: the basis does not fit in L2): a capped GMRES run
        iters = args.gmres_iters
        ctx.set_params(gmres_maxit=iters, gmres_tol=1e-30)
        b = ctx.rhs_multipole()
        ctx.gmres(b)                                   # warm-up: workspace allocation
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); _, info = ctx.gmres(b); e1.record(); e1.synchronize()
        ms_g = e0.elapsed_time(e1)
        e0.record()
        for _ in range(5):
            ctx.matvec(xd, out=y)
        e1.record(); e1.synchronize()
        ms_mv = e0.elapsed_time(e1) / 5
        n2 = 2 * nt
        # per iteration j (nv = j+1 basis vectors): two dot passes read nv+1 vectors, two updates read nv+1 and write 1 (+1 for v_next)
        byts = sum((2 * (j + 2) + 2 * (j + 2) + 3) * n2 * 8 for j in range(info["iters"]))
        ms_vec = ms_g - (info["iters"] + 2) * ms_mv
        print(json.dumps({"case": "gmres_vectors", "workload": w.name, "iters": info["iters"], "ms_total": ms_g, "ms_per_matvec": ms_mv,
                          "ms_vector_kernels": ms_vec, "algorithmic_gb": byts / 1e9, "gb_per_s": byts / 1e9 / (ms_vec * 1e-3),
                          "hbm_peak_gb_per_s_measured": 6551.0}), flush=True)
        ctx.set_params(gmres_maxit=1000, gmres_tol=float(w.params["gmres_tol"]))
    if "solve" not in cases:
        ctx.close()
        return
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    _, _, res = ctx.solve()
    torch.cuda.synchronize()
    print(json.dumps({"case": "solve", "workload": w.name, "sites": int(w.sites["pos"].shape[0]), "seconds": time.perf_counter() - t0,
                      **{k: res[k] for k in ("dG_solv", "scf_iters", "scf_iters_vac", "gmres_iters_total", "matvecs_total",
                                             "final_scf_delta_debye", "final_gmres_relres", "status")}}), flush=True)
    ctx.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4", help="C4 (BASELINE configs[4], default), C1, C2, C3-complex, C3-receptor, C3-ligand")
    ap.add_argument("--theta", type=float, default=None)
    ap.add_argument("--order", type=int, default=None)
    ap.add_argument("--ncrit", type=int, default=None)
    ap.add_argument("--list-split", type=int, default=None, choices=(0, 1),
                    help="pb_params.list_split: 1 (library default) = the two 32-target halves of a group take the MAC decisions "
                         "separately, 0 = one decision per 64-target group")
    ap.add_argument("--scf-recycle", type=int, default=None, choices=(0, 1, 2), help="pb_params.scf_recycle (library default 2)")
    ap.add_argument("--scf-eta", type=float, default=None, help="pb_params.scf_eta (library default 0.03)")
    ap.add_argument("--ref-rows", type=int, default=256,
                    help="target rows per oracle call (cpu_baseline and --impl reference): about 2 s per call at C4 on 16 cores")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--replicas", action="store_true",
                    help="N > 1: independent replicas of the whole matvec on every rank (weak scaling) instead of target sharding")
    ap.add_argument("--no-solve", action="store_true", help="skip the timed full polarizable solve")
    ap.add_argument("--no-configs", action="store_true", help="skip the C1-C3 solve times")
    ap.add_argument("--profiler-range", action="store_true",
                    help="bracket the timed resident steps with cudaProfilerStart/Stop (for ncu --profile-from-start off)")
    ap.add_argument("--sweep", action="store_true",
                    help="theta x P matvec sweep with sampled-row accuracy and one full solve (BASELINE configs[4])")
    ap.add_argument("--sweep-rows", type=int, default=1024)
    ap.add_argument("--sweep-cases", default="matvec,solve", help="comma list of matvec, gmres, solve")
    ap.add_argument("--gmres-iters", type=int, default=40)
    args = ap.parse_args()
    if args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
