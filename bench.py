"""bench.py — H_eff·ψ / Davidson-step benchmark of the dmrgk library (contract: see DESIGN.md §Measurement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4|3|2|4rs] [--impl ours|reference]

One "step" is one pass of the whole hot path: one Davidson step (Rayleigh–Ritz, residual, diagonal
preconditioner, 2× Gram–Schmidt, normalise, ONE σ = H_eff ψ apply, Rayleigh-matrix extension) on the
synthetic workload of BASELINE.json configs[3] (6×6 Hubbard, mode-rotated, D = 4096 — the
configuration the metric "H_eff·ψ FP64 TFLOPS … at D=4096" is quoted on; it fits one GPU).
`value` = algorithmic flops of the matvec (dmrgk_heff_query: Σ_tasks min(2m′n(m+n′), 2mn′(n+m′)))
× steps ÷ device time of the steps, i.e. the vector kernels and the host Rayleigh–Ritz are inside the
timed region and count as overhead.  The path does not shard (BASELINE.json: one GPU, no collectives):
with --gpus N every rank runs an independent replica ("replicas only").

The reference arm (--impl reference) times the oracle (oracle/heff.py sigma_blockwise, NumPy/BLAS,
as it stands) on the host cores on a bounded sample of the same workload.
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

METRIC = "heff_apply_fp64_tflops_in_davidson_step"
SAMPLE_EVERY = {"4": 337, "3": 268, "3b": 536, "2": 8, "5": 286, "5r": 286}   # cpu_baseline: every n-th operator pair
UNIT = "TFLOP/s"


def make_workload(name):
    import workloads as wlmod
    if name == "4":
        return wlmod.config4()
    if name == "3":
        return wlmod.config3()
    if name == "3b":
        return wlmod.lattice_workload("spinless", 32, 8192, seed=3, name="shape3b_spinless8x8_rotated_D4096")
    if name in ("5", "5r"):
        return wlmod.config5()      # executed subset; "5": part of it streamed from pinned host memory, "5r": all resident
    if name == "2":
        return wlmod.synthetic_config2()
    raise SystemExit(f"unknown --config {name}")


def sample_terms(wl, every, offset=0):
    """A stratified sample of the operator-pair list: every `every`-th term (h.c. partners are
    adjacent in the list, so families keep their proportions).  Returns (sub-workload, term ids)."""
    import copy
    ids = list(range(offset, len(wl.terms), every))
    sub = copy.copy(wl)
    sub.terms = [wl.terms[i] for i in ids]
    return sub, ids


def host_problem_for_sample(wl, sub):
    """oracle.heff.Problem holding only the operators the sampled terms touch (host generator)."""
    from oracle import heff as oheff
    from workloads import fill_op_host, fill_psi_host
    need = sorted({i for t in sub.terms for i in (t.L, t.R) if i is not None})
    ops = [{"half": s.half, "dq": tuple(s.dq), "parity": s.parity, "blocks": {}} for s in wl.ops]
    for i in need:
        ops[i]["blocks"] = fill_op_host(wl, i)
    terms = [(t.L, t.R, t.coef, t.trans_L, t.trans_R) for t in sub.terms]
    return oheff.Problem(wl.n_charges, list(wl.sectors_A), list(wl.sectors_B), tuple(wl.target), ops, terms,
                         fill_psi_host(wl), wl.name + "_sample")


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else 1
    except Exception:
        return os.cpu_count() or 1


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        def pump():
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        self.thread = threading.Thread(target=pump, daemon=True)
        self.thread.start()

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, smax, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def max_over_ranks(ms, world, device=None):
    """Max of a per-rank duration over all ranks (replicas run independently; the job is as slow
    as its slowest rank).  Works on any initialised backend (nccl on GPUs, gloo in the CPU tests)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_tflops(flops_per_rank_step, world, ms_step):
    """Whole-job throughput of `world` independent replicas ("replicas only", weak scaling)."""
    return world * flops_per_rank_step / ms_step / 1e9


def time_oracle(pb, steps, warmup):
    """Seconds per σ = H_eff ψ of the oracle's blockwise tier on the host cores."""
    from oracle import heff as oheff
    for _ in range(warmup):
        oheff.sigma_blockwise(pb)
    t0 = time.perf_counter()
    for _ in range(steps):
        oheff.sigma_blockwise(pb)
    return (time.perf_counter() - t0) / max(steps, 1)


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step = σ of a bounded
    stratified sample of the workload's operator pairs (the full list would take hours)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import heff as oheff
    wl = make_workload(args.config)
    every = SAMPLE_EVERY[args.config]
    sub, ids = sample_terms(wl, every)
    pb = host_problem_for_sample(wl, sub)
    flops = float(oheff.flops_alg(pb))
    sec = time_oracle(pb, args.steps, args.warmup)
    val = flops / sec / 1e12
    cores = blas_threads()
    sample = f"every {every}th operator pair ({len(ids)} of {len(wl.terms)}), all ψ blocks, {flops:.3e} flop per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    import workloads as wlmod
    from paper_2311_14106_b200 import build as b, dmrgk, problem

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: dmrgk has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if not os.path.exists(dmrgk.LIB_PATH):
        if rank == 0:
            b.build()
        if world > 1:
            dist.barrier()
    dmrgk.load()

    wl = make_workload(args.config)
    t0 = time.perf_counter()
    staged = wlmod.config5_staged_ops(wl) if args.config == "5" else []
    dp = problem.from_workload(wl, device=local, pinned=staged, **({"ring_bytes": 6 << 30} if staged else {}))
    torch.cuda.synchronize()
    setup_s = time.perf_counter() - t0
    h = dp.heff
    n = dp.layout.n_padded
    psi = dp.psi_fill(wl.seed, wlmod.PSI_STREAM)
    dav = dp.davidson(m_max=args.m_max, tol=0.0, max_iter=1 << 30)     # tol 0: never stops early
    dav.start(psi)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- the timed region: K Davidson steps (each exactly one H_eff apply) --------------------
    for _ in range(args.warmup):
        dav.step()
    barrier()
    h.profile(True)
    dmrgk.launch_count(reset=True)
    clocks = ClockSampler(local)
    clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(dp.stream)
    for _ in range(args.steps):
        theta, rho, _ = dav.step()
    e1.record(dp.stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = dmrgk.launch_count()
    prof_ms, prof_n = h.profile_read()
    h.profile(False)
    clk = clocks.stop()
    ms_total = max_over_ranks(ms_total, world, "cuda")
    ms_step = ms_total / args.steps
    value = aggregate_tflops(h.flops_alg, world, ms_step)

    # ---- e2e: the same matvec through the C-ABI call with HOST buffers ---------------------------
    ph = torch.empty(n, dtype=torch.float64).pin_memory()
    sh = torch.empty(n, dtype=torch.float64).pin_memory()
    ph.copy_(psi[:n])
    pdev, sdev = dp.new_vector(), dp.new_vector()
    for _ in range(2):
        h.apply_host(ph, sh, pdev, sdev, dp.workspace, dp.stream, dp.copy_stream)
    barrier()
    clocks_e2e = ClockSampler(local)
    clocks_e2e.start()
    e2, e3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e2.record(dp.stream)
    for _ in range(args.steps):
        h.apply_host(ph, sh, pdev, sdev, dp.workspace, dp.stream, dp.copy_stream)
    e3.record(dp.stream)
    barrier()
    ms_e2e = e2.elapsed_time(e3) / args.steps
    clk_e2e = clocks_e2e.stop()
    ms_e2e = max_over_ranks(ms_e2e, world, "cuda")

    # ---- the FP64 ceiling of this box, live: register-only DMMA loop (burst) -------------------
    sink = torch.zeros(16, dtype=torch.float64, device="cuda")
    dmma_probe = 0.0
    for _ in range(4):      # first call warms up; best of the rest
        pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        pe0.record(dp.stream)
        pf = dmrgk.probe_fp64(dp.ctx, 0, 20000, sink, dp.stream)
        pe1.record(dp.stream)
        torch.cuda.synchronize()
        dmma_probe = max(dmma_probe, pf / pe0.elapsed_time(pe1) / 1e9)
    n_sm = dp.ctx.query()[0]
    sm_max = clk.get("sm_max_mhz") or 1965.0
    peak = n_sm * 128 * sm_max * 1e6 / 1e12     # 64 DFMA-equivalents/clk/SM

    # ---- a8 vector kernels alone: achieved HBM GB/s against MEASURED_PEAKS.json hbm_gbs ------------
    def time_vec(fn, reps=10):
        fn()
        torch.cuda.synchronize()
        v0, v1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        v0.record(dp.stream)
        for _ in range(reps):
            fn()
        v1.record(dp.stream)
        torch.cuda.synchronize()
        return v0.elapsed_time(v1) / reps
    mv = min(8, args.m_max)
    scratch = torch.empty(dmrgk.vec_scratch_bytes(mv + 1), dtype=torch.uint8, device="cuda")
    outv = torch.zeros(64, dtype=torch.float64, device="cuda")
    coefv = torch.full((64,), 0.125, dtype=torch.float64, device="cuda")
    yv = dp.new_vector()
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        hbm_src = "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        hbm_peak, hbm_src = 6650.0, "fallback (B200_PROFILING.md)"
    t_dot = time_vec(lambda: dmrgk.vec_multi_dot(dp.ctx, n, mv, dp.V, n, psi, outv, scratch, dp.stream))
    t_axpy = time_vec(lambda: dmrgk.vec_multi_axpy(dp.ctx, n, mv, dp.V, n, coefv, -1.0, 1.0, yv, dp.stream))
    t_res = time_vec(lambda: dmrgk.vec_residual(dp.ctx, n, mv, dp.V, dp.W, n, coefv, yv, outv, scratch, dp.stream))
    gbs = lambda nvec, ms: nvec * n * 8 / ms / 1e6
    vec = {"n_doubles": int(n), "m": mv, "peak_gbs": hbm_peak, "peak_source": hbm_src,
           "multi_dot": {"ms": t_dot, "gbs": gbs(mv + 1, t_dot), "frac": gbs(mv + 1, t_dot) / hbm_peak},
           "multi_axpy": {"ms": t_axpy, "gbs": gbs(mv + 2, t_axpy), "frac": gbs(mv + 2, t_axpy) / hbm_peak},
           "residual": {"ms": t_res, "gbs": gbs(2 * mv + 1, t_res), "frac": gbs(2 * mv + 1, t_res) / hbm_peak}}

    # dram__bytes_read.sum + dram__bytes_write.sum per GEMM launch from the committed ncu --set full
    # capture of this workload (profiles/r1_v3_summary.md); other workloads have no capture
    traffic = 12.99e9 if args.config == "4" else None

    # device time of the GEMM region of the applies (phase-1/phase-2 launches overlap on two streams, so
    # per-launch durations are not additive; the span from the first to the last launch of each apply
    # is what is timed, and it includes the split-k reduce launches)
    gemm_ms = prof_ms["apply"]
    gemm_n = prof_n["p1"] + prof_n["p2"]
    achieved = h.flops_alg * args.steps / gemm_ms / 1e9 if gemm_ms > 0 else None
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "M_A": wl.M_A, "M_B": wl.M_B, "K_pairs": len(wl.terms), "tasks": h.n_tasks,
                   "flops_alg_per_apply": h.flops_alg, "op_bytes_resident": int(dp.op_arena.numel() * 8),
                   "psi_elems": dp.layout.n_elems, "davidson_m_max": args.m_max, "parallelism": "replicas only",
                   "l2": "operator arena (>> 126 MB L2) is streamed once per step; no flush needed",
                   "setup_s": round(setup_s, 2), "chunks": h.n_chunks,
                   "staged_ops": len(staged), "staged_bytes_per_apply": int(sum(dp.ops[i].n_padded for i in staged) * 8)},
        "davidson_step_ms": ms_step, "theta_last": theta, "resnorm_last": rho,
        "pct_of_fp64_peak": 100.0 * value / world / peak,
        "e2e": {"value": world * h.flops_alg / ms_e2e / 1e9, "unit": UNIT, "ms_per_step": ms_e2e,
                "what": "dmrgk_heff_apply_host: pinned ψ H2D, apply, σ D2H",
                "h2d_bytes_per_step": int(n * 8), "d2h_bytes_per_step": int(n * 8), "clocks": clk_e2e},
        "gpu_launches": int(launches),
        "roofline": {"bound": "tensor", "kernel": "heff_gemm_dmma_kernel (a5 + a6)", "achieved": achieved,
                     "peak": peak, "unit": "TFLOP/s", "frac": (achieved / peak) if achieved else None,
                     "peak_source": f"derived: {n_sm} SMs x 128 FP64 flop/clk x {sm_max:.0f} MHz (no FP64 figure in "
                                    "MEASURED_PEAKS.json); in-run register-only DMMA probe below corroborates",
                     "dmma_probe_tflops": dmma_probe, "launches": int(gemm_n), "avg_launch_ms": gemm_ms / max(gemm_n, 1),
                     "kernel_ms_per_step": gemm_ms / args.steps, "reduce_launches": int(prof_n["reduce"]),
                     "traffic": traffic, "traffic_note": "average over the 48 GEMM launches of one apply (ncu, cold cache); "
                     "algorithmic bytes per launch = 4.2e9 (operators read once per task + psi + sigma); the excess is the T "
                     "round trip and tile re-reads that miss L2 - 0.93 TB/s in total, 14 % of HBM, not the bound"},
        "vector_kernels": vec,
        "clocks": clk,
    }
    if rank == 0 and world == 1 and not args.no_cpu:
        from oracle import heff as oheff
        every = SAMPLE_EVERY[args.config]
        sub, ids = sample_terms(wl, every)
        pb = host_problem_for_sample(wl, sub)
        fl = float(oheff.flops_alg(pb))
        reps = 0
        t0 = time.perf_counter()
        while reps < 3 or (time.perf_counter() - t0 < 10.0 and reps < 200):
            oheff.sigma_blockwise(pb)
            reps += 1
        sec = (time.perf_counter() - t0) / reps
        out["cpu_baseline"] = {"value": fl / sec / 1e12, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                               "sample": f"oracle.heff.sigma_blockwise on every {every}th operator pair ({len(ids)} of "
                                         f"{len(wl.terms)}), all ψ blocks, {fl:.3e} flop x {reps} repeats"}
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_renorm(args):
    """--op renorm: one step = the renormalisation O' = Phi^T O Phi of every enlarged-block operator of
    the left half of the workload to D kept states; not the headline metric."""
    import torch
    import workloads as wlmod
    from paper_2311_14106_b200 import dmrgk, problem
    from oracle import renorm as orenorm
    torch.cuda.set_device(0)
    wl = make_workload(args.config)
    dp = problem.from_workload(wl)
    sectors_new, table = wlmod.renorm_basis(wl)
    rp = problem.RenormProblem(dp, "A", sectors_new)
    rp.fill_phi(wl.seed, wlmod.PHI_STREAM)
    rp.build([(wl.ops[i].dq, wl.ops[i].parity) for i in rp.idx])
    for _ in range(args.warmup):
        rp.apply()
    torch.cuda.synchronize()
    clocks = ClockSampler(0)
    clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dmrgk.launch_count(reset=True)
    e0.record(dp.stream)
    for _ in range(args.steps):
        rp.apply()
    e1.record(dp.stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    launches = dmrgk.launch_count()
    clk = clocks.stop()
    n_sm = dp.ctx.query()[0]
    peak = n_sm * 128 * (clk.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
    val = rp.plan.flops / ms / 1e9
    out = {"metric": "renorm_fp64_tflops", "value": val, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": wl.name + "_renorm_left_half", "operators": len(rp.idx), "blocks": rp.plan.n_tasks,
                      "M_enlarged": wl.M_A, "M_kept": sum(d for _, d in sectors_new), "flops_per_apply": rp.plan.flops,
                      "in_bytes": int(sum(op.n_padded for op in rp.ops_in) * 8),
                      "out_bytes": int(sum(op.n_padded for op in rp.ops_out) * 8),
                      "l2": "operator arenas (>> 126 MB L2) are streamed once per step"},
           "gpu_launches": int(launches),
           "roofline": {"bound": "tensor", "kernel": "heff_gemm_dmma_kernel (renormalisation work lists)", "achieved": val,
                        "peak": peak, "unit": "TFLOP/s", "frac": val / peak, "traffic": None,
                        "launches": int(rp.plan.n_launches * args.steps)},
           "clocks": clk}
    if not args.no_cpu:
        phi = wlmod.fill_phi_host(wl, table)
        ids = rp.idx[::max(1, len(rp.idx) // 12)]
        ops = [{"half": "A", "dq": tuple(wl.ops[i].dq), "parity": wl.ops[i].parity, "blocks": wlmod.fill_op_host(wl, i)} for i in ids]
        fl = float(sum(orenorm.flops(o, phi) for o in ops))
        reps, t0 = 0, time.perf_counter()
        while reps < 2 or (time.perf_counter() - t0 < 10.0 and reps < 100):
            for o in ops:
                orenorm.renormalise_blockwise(o, wl.sectors_A, phi, sectors_new)
            reps += 1
        sec = (time.perf_counter() - t0) / reps
        out["cpu_baseline"] = {"value": fl / sec / 1e12, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                               "sample": f"oracle.renorm.renormalise_blockwise on {len(ids)} of {len(rp.idx)} operators, {fl:.3e} flop x {reps} repeats"}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="4", choices=["2", "3", "3b", "4", "5", "5r"])
    ap.add_argument("--m-max", dest="m_max", type=int, default=16)
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--op", default="davidson", choices=["davidson", "renorm"],
                    help="davidson (default, the headline hot path) or renorm (NEXT-1 row, its own metric)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.op == "renorm":
        run_renorm(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
