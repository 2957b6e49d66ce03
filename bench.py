#!/usr/bin/env python
"""bench.py -- one polarizable Poisson-Boltzmann solve per step on seeded synthetic input.

A step is one pass of the whole hot path over one workload:
pb_mesh_load -> pb_sites_load -> pb_tree_build (Morton octree, lists, near/singular table) ->
pb_solve (vacuum SCF, then {RHS -> GMRES with one treecode matvec per iteration -> reaction
field -> multipole field -> SOR update} to 1e-7 Debye, then the energies).

  metric  = treecode matvec interactions per second over the whole step.  One interaction = one
            (collocation point, source Gauss point) pair of the N x N_s pairs the operator of
            Eq. (5) accounts for in a matvec, whether it is summed directly (P2P) or through a
            cell expansion (M2P): value = N * N_s * matvecs / time.  This is the unit the oracle's
            direct sum is timed in (cpu_baseline, --impl reference), and it does not reward
            evaluating more pairs than the MAC requires.  The pairs actually evaluated per second
            (P2P pairs, M2P (target, cell) pairs) are reported beside it under "evaluated".
  ms_per_step = time per polarizable PB solve (the second half of BASELINE.json's metric)
  e2e     = the same through the host-buffer C-ABI calls (inputs in pinned host memory copied in
            every step, x and mu copied out)
  roofline = the dominant kernel (P2P), FP64 ALU bound, CUDA-event timed inside the step
  cpu_baseline = the oracle's direct O(N^2 K) matvec on this box's host cores

python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C1] [--impl reference]
N > 1 (torchrun): the path has no data-path exchange on one GPU; ranks run independent
replicas of the workload ("weak" scaling), timed as the max over ranks.
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

METRIC = "treecode_matvec_interactions_per_s"
UNIT = "interactions/s"
# Algorithmic FP64 work per unit: one P2P pair = the four kernels of
# Eq. (3)-(4) for one (target, Gauss point) pair; one M2P pair at order P = 4*NT + Nk + 6P + 30.
P2P_FLOP_PER_PAIR = 80.0
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12     # SMs x FP64 FMA lanes x 2 x max SM clock


def n_terms_of(P):
    return sum((P - a - b - c) // 2 + 1 for a in range(P + 1) for b in range(P + 1 - a) for c in range(P + 1 - a - b))


def m2p_flop_per_pair(P, n_terms=None):
    nk = (P + 1) * (P + 2) * (P + 3) // 6
    return 4.0 * (n_terms if n_terms is not None else n_terms_of(P)) + nk + 6.0 * P + 30.0


def m2p_flop(P, st):
    """Algorithmic flop of one M2P launch: pairs at order P plus the pairs the list build flagged for order P - 2."""
    low = st.get("m2p_pairs_low", 0)
    return m2p_flop_per_pair(P, st["n_terms"]) * (st["m2p_pairs"] - low) + (m2p_flop_per_pair(P - 2) * low if low else 0.0)


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
            self.stop_flag.wait(0.2)

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
    return make_config(name)


def oracle_matvec_rate(w, budget_s=12.0):
    """The oracle as it stands: direct O(N^2 K) matvec over all host cores."""
    import numpy as np
    from oracle import pb_oracle as po
    po.build()
    orc = po.Oracle(w.verts, w.tris, po.Params(K_far=w.params["K_far"]))
    n = orc.nt
    x = np.random.Generator(np.random.PCG64(7)).normal(size=2 * n)
    rows = None
    pairs_per_call = float(n) * n * w.params["K_far"]
    if pairs_per_call > 2e9:                      # bounded sample of target rows on big meshes
        rows = np.random.Generator(np.random.PCG64(8)).choice(n, size=4096, replace=False)
        pairs_per_call = 4096.0 * n * w.params["K_far"]
    orc.matvec(x, rows)                            # warm-up (thread pool, page faults)
    t0 = time.perf_counter()
    reps = 0
    while True:
        orc.matvec(x, rows)
        reps += 1
        el = time.perf_counter() - t0
        if el > budget_s or reps >= 50:
            break
    return dict(value=pairs_per_call * reps / el, unit=UNIT, cores=po.num_threads(), kind="oracle",
                sample=f"{reps} direct O(N^2 K) oracle matvecs of {w.name}"
                       + (" on 4096 sampled target rows" if rows is not None else " (all rows)")
                       + f", {el:.1f} s", ms_per_call=1e3 * el / reps)


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    w = load_workload(args.workload)
    import numpy as np
    from oracle import pb_oracle as po
    po.build()
    orc = po.Oracle(w.verts, w.tris, po.Params(K_far=w.params["K_far"]))
    n = orc.nt
    x = np.random.Generator(np.random.PCG64(7)).normal(size=2 * n)
    rows = None
    pairs = float(n) * n * w.params["K_far"]
    if pairs > 2e9:
        rows = np.random.Generator(np.random.PCG64(8)).choice(n, size=4096, replace=False)
        pairs = 4096.0 * n * w.params["K_far"]
    for _ in range(args.warmup):
        orc.matvec(x, rows)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.matvec(x, rows)
    el = time.perf_counter() - t0
    val = pairs * args.steps / el
    sample = (f"each step = one direct O(N^2 K) oracle matvec of {w.name}"
              + (" on 4096 sampled target rows" if rows is not None else " (all rows)"))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "panels": int(n), "K_far": int(w.params["K_far"]), "what": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": po.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


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

    w = load_workload(args.workload)               # every rank: its own replica of the workload
    names = {k for k, _ in pb.Params._fields_}
    prm = {k: v for k, v in w.params.items() if k in names}
    if args.theta is not None:
        prm["theta"] = args.theta
    if args.order is not None:
        prm["order_P"] = args.order
    if args.ncrit is not None:
        prm["ncrit"] = args.ncrit
    ctx = pb.PB(local_rank, **prm)
    s = w.sites
    f64, i32 = torch.float64, torch.int32
    host = dict(verts=torch.from_numpy(np.ascontiguousarray(w.verts)).pin_memory(),
                tris=torch.from_numpy(np.ascontiguousarray(w.tris, dtype=np.int32)).pin_memory(),
                pos=torch.from_numpy(np.ascontiguousarray(s["pos"])).pin_memory(),
                q=torch.from_numpy(np.ascontiguousarray(s["q"])).pin_memory(),
                dip=torch.from_numpy(np.ascontiguousarray(s["dip"])).pin_memory(),
                quad=torch.from_numpy(np.ascontiguousarray(s["quad"])).pin_memory(),
                alpha=torch.from_numpy(np.ascontiguousarray(s["alpha"])).pin_memory(),
                group=torch.from_numpy(np.ascontiguousarray(s["group"], dtype=np.int32)).pin_memory())
    resident = {k: v.to(dev) for k, v in host.items()}
    nt, na = int(w.tris.shape[0]), int(s["pos"].shape[0])
    x_host = torch.empty(2 * nt, dtype=f64).pin_memory()
    mu_host = torch.empty(na, 3, dtype=f64).pin_memory()
    h2d = sum(v.numel() * v.element_size() for v in host.values())
    d2h = x_host.numel() * 8 + mu_host.numel() * 8
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def step_resident():
        d = resident
        ctx.mesh_load(d["verts"], d["tris"])
        ctx.sites_load(d["pos"], d["q"], d["dip"], d["quad"], d["alpha"], d["group"])
        ctx.tree_build()
        return ctx.solve()[2]

    def step_e2e():
        d = {k: v.to(dev, non_blocking=True) for k, v in host.items()}
        ctx.mesh_load(d["verts"], d["tris"])
        ctx.sites_load(d["pos"], d["q"], d["dip"], d["quad"], d["alpha"], d["group"])
        ctx.tree_build()
        return ctx.solve_host(x_host, mu_host)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps):
        tot_ms, last = 0.0, None
        for _ in range(steps):
            flush.zero_()                          # L2 flush, outside the event pair
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            last = fn()
            e1.record()
            e1.synchronize()
            tot_ms += e0.elapsed_time(e1)
        return tot_ms, last

    for _ in range(max(args.warmup, 3)):
        res = step_resident()
    step_e2e()
    sampler = ClockSampler(local_rank)
    sampler.start()
    st0 = ctx.stats()
    barrier()
    if args.profiler_range:                        # ncu --profile-from-start off captures exactly the timed steps
        torch.cuda.profiler.start()
    ms_total, res = timed(step_resident, args.steps)
    if args.profiler_range:
        torch.cuda.synchronize()
        torch.cuda.profiler.stop()
    barrier()
    st1 = ctx.stats()
    barrier()
    ms_e2e, res_e2e = timed(step_e2e, args.steps)
    barrier()
    # Kernel durations for the roofline: the SAME steps once more with a CUDA-event pair around every
    # P2P and M2P launch.  In this mode the library runs the matvec's two branches back to back on one
    # stream (in the timed steps above the far-field branch overlaps P2P on a second stream), so each
    # pair brackets exactly one kernel; grids, blocks and data are identical.
    ctx.set_profiling(True)
    ms_prof, _ = timed(step_resident, args.steps)
    stp = ctx.stats()
    ctx.set_profiling(False)
    barrier()
    sampler.stop_flag.set()
    sampler.join(timeout=2)

    ms_total = max_over_ranks(ms_total, world, dev)
    ms_e2e = max_over_ranks(ms_e2e, world, dev)
    inter_per_mv = float(nt) * float(st1["n_sources"])          # the N x N_s pairs one matvec accounts for
    evald_per_mv = st1["p2p_pairs"] + st1["m2p_pairs"]
    mv_timed = st1["matvec_calls"] - st0["matvec_calls"]
    units = sum_over_ranks(float(inter_per_mv) * mv_timed, world, dev)
    units_e2e = sum_over_ranks(float(inter_per_mv) * res_e2e["matvecs_total"] * args.steps, world, dev)
    value = units / (ms_total * 1e-3)
    value_e2e = units_e2e / (ms_e2e * 1e-3)
    launches = st1["kernel_launches"] - st0["kernel_launches"]

    # roofline of the dominant kernel, from the CUDA-event pairs recorded inside the timed steps
    P = int(ctx.get_params().order_P)
    p2p_ms = stp["prof_p2p_ms"] / max(stp["prof_p2p_launches"], 1)
    m2p_ms = stp["prof_m2p_ms"] / max(stp["prof_m2p_launches"], 1)
    p2p_tf = P2P_FLOP_PER_PAIR * st1["p2p_pairs"] / (p2p_ms * 1e-3) / 1e12 if p2p_ms > 0 else 0.0
    m2p_tf = (m2p_flop(P, st1) / (m2p_ms * 1e-3) / 1e12) if m2p_ms > 0 else 0.0
    dominant = "k_p2p" if stp["prof_p2p_ms"] >= stp["prof_m2p_ms"] else "k_m2p"
    ach = p2p_tf if dominant == "k_p2p" else m2p_tf
    # DRAM bytes per launch of the dominant kernel from the committed ncu --set full captures (per workload)
    traffic = {("C1", "k_p2p"): (2.517e6, "profiles/r01c_ncu_full_C1.md"),
               ("C4", "k_m2p"): (7.68e8, "profiles/r01b_ncu_full_C4.md")}.get((w.name, dominant), (None, None))
    roofline = {"bound": "alu", "kernel": dominant, "achieved": ach, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                "frac": ach / FP64_PEAK_TFLOPS, "traffic": traffic[0], "traffic_source": traffic[1],
                "peak_source": "148 SM x 64 FP64 FMA lanes x 2 x 1.965 GHz (DESIGN.md section 7); "
                               "pb_fp64_peak_probe measured %.1f TFLOP/s on this GPU" % ctx.fp64_peak_probe(),
                "timed_in": "a repeat of the timed steps with per-kernel CUDA events (branches serialised on one "
                            "stream): %.3f ms per step against %.3f ms with the far-field branch overlapped" % (
                                ms_prof / args.steps, ms_total / args.steps),
                "p2p": {"ms_per_launch": p2p_ms, "launches": stp["prof_p2p_launches"], "pairs": st1["p2p_pairs"],
                        "tflops": p2p_tf, "share_of_step": stp["prof_p2p_ms"] / ms_prof},
                "m2p": {"ms_per_launch": m2p_ms, "launches": stp["prof_m2p_launches"], "pairs": st1["m2p_pairs"],
                        "tflops": m2p_tf, "share_of_step": stp["prof_m2p_ms"] / ms_prof}}
    if rank != 0:
        return
    cpu = oracle_matvec_rate(w) if world == 1 and not args.no_cpu_baseline else None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "panels": nt, "gauss_points": int(st1["n_sources"]), "sites": na,
                   "theta": float(ctx.get_params().theta), "order_P": P, "ncrit": int(st1["ncrit_used"]),
                   "K_far": int(w.params["K_far"]), "gmres_tol": float(ctx.get_params().gmres_tol),
                   "scf_tol_debye": float(ctx.get_params().scf_tol_debye),
                   "l2": "flushed between steps (256 MiB device write, outside the event pairs)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "solve": {"time_per_polarizable_solve_ms": ms_total / args.steps, "dG_solv_kcal_mol": res["dG_solv"],
                  "scf_iters": res["scf_iters"], "gmres_iters": res["gmres_iters_total"], "matvecs": res["matvecs_total"],
                  "interactions_per_matvec": int(inter_per_mv), "status": res["status"]},
        "evaluated": {"p2p_pairs_per_matvec": int(st1["p2p_pairs"]), "m2p_pairs_per_matvec": int(st1["m2p_pairs"]),
                      "m2p_pairs_at_order_P_minus_2": int(st1["m2p_pairs_low"]),
                      "pairs_per_s": float(evald_per_mv) * mv_timed / (ms_total * 1e-3) * (world if world > 1 else 1)},
        "e2e": {"value": value_e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "ms_per_step": ms_e2e / args.steps},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "clocks": sampler.summary(),
    }
    if cpu is not None:
        line["cpu_baseline"] = cpu
    print(json.dumps(line))
    ctx.close()
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
    for theta in (0.3, 0.5, 0.7):
        for P in (4, 6, 8):
            if "matvec" not in cases:
                break
            ctx.set_params(theta=theta, order_P=P)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); ctx.tree_build(); e1.record(); e1.synchronize()
            t_build = e0.elapsed_time(e1)
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
            fl_m = m2p_flop_per_pair(P, st["n_terms"])
            print(json.dumps({
                "case": "matvec", "workload": w.name, "theta": theta, "order_P": P, "ncrit": int(st["ncrit_used"]),
                "ms_per_matvec": ms, "tree_build_ms": t_build,
                "interactions_per_s": float(nt) * st["n_sources"] / (ms * 1e-3),
                "p2p_pairs": int(st["p2p_pairs"]), "m2p_pairs": int(st["m2p_pairs"]),
                "serial_ms": {k: lm[k] for k in ("weights", "p2m_m2m", "m2p", "p2p", "near_combine")},
                "p2p_tflops": P2P_FLOP_PER_PAIR * st["p2p_pairs"] / (lm["p2p"] * 1e-3) / 1e12,
                "m2p_pairs_low_order": int(st["m2p_pairs_low"]),
                "m2p_tflops": m2p_flop(P, st) / (lm["m2p"] * 1e-3) / 1e12 if lm["m2p"] > 0 else 0.0,
                "fp64_peak_tflops": FP64_PEAK_TFLOPS, "rel_l2_vs_oracle_rows": err, "device_gb": st["device_bytes"] / 1e9}), flush=True)
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
                          "hbm_peak_gb_per_s_measured": 6548.2}), flush=True)
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
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C1", help="C1 (BASELINE configs[1], default), C0, C2, C3, C4")
    ap.add_argument("--theta", type=float, default=None)
    ap.add_argument("--order", type=int, default=None)
    ap.add_argument("--ncrit", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--profiler-range", action="store_true",
                    help="bracket the timed resident steps with cudaProfilerStart/Stop (for ncu --profile-from-start off)")
    ap.add_argument("--sweep", action="store_true",
                    help="theta x P matvec sweep with sampled-row accuracy and one full solve (BASELINE configs[4]); use with --workload C4")
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
