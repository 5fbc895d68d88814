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
SAMPLE_EVERY = {"4": 100, "3": 100, "3b": 268, "2": 8, "5": 143, "5r": 143, "4rs": 2, "1": 1}   # --impl reference: every n-th operator pair (host-generated values)
CPU_EVERY = {"4": 20, "3": 20, "3b": 40, "2": 4, "5": 20, "5r": 20, "4rs": 1, "1": 1}              # cpu_baseline leg: ≈ 5 % of the pairs (values read back D2H)
UNIT = "TFLOP/s"


def make_workload(name):
    import workloads as wlmod
    if name == "4":
        return wlmod.config4()
    if name == "4rs":
        return wlmod.config4_realspace()     # configs[3], real-space basis: K = 50 pairs (H_A, H_B and the boundary hoppings)
    if name == "3":
        return wlmod.config3()
    if name == "3b":
        return wlmod.lattice_workload("spinless", 32, 8192, seed=3, name="shape3b_spinless8x8_rotated_D4096")
    if name in ("5", "5r"):
        return wlmod.config5()      # executed subset; "5": part of it streamed from pinned host memory, "5r": all resident
    if name == "2":
        return wlmod.synthetic_config2()
    if name == "1":
        # configs[0]'s SHAPE ("latency only"): 4×4 spinless torus cut 8|8, D = 64 (M = 128), the dense
        # mode-rotated term list (K = 154), seeded values.  The operators of the real bond come out of a DMRG sweep, which
        # only the oracle has (tests/_gpu.config1_problem is that parity case); the timing needs the shape, not the state.
        return wlmod.lattice_workload("spinless", 8, 128, seed=1, name="config1_shape_spinless4x4_rotated_K154_D64")
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


def timed(stream, fn, reps=1):
    """CUDA-event milliseconds of `reps` calls of fn on `stream` (synchronises on both sides)."""
    import torch
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(reps):
        fn()
    b.record(stream)
    torch.cuda.synchronize()
    return a.elapsed_time(b)


def measure_fp64_ceiling(dp, local):
    """The FP64 ceilings of THIS box in THIS run, outside every timed region (two
    denominators).  (i) cuBLAS DGEMM 8192³ through torch.matmul — a library GEMM used only as a
    yardstick — best of 10 (burst) and back to back for ≥ 4 s (sustained); (ii) the library's
    register-only DMMA probe, best of 5 short runs (burst) and one ≥ 1 s run (sustained).  The SM
    clock is sampled during each sustained leg."""
    import torch
    from paper_2311_14106_b200 import dmrgk
    out = {}
    N = 8192
    A = torch.randn(N, N, dtype=torch.float64, device="cuda")
    B = torch.randn(N, N, dtype=torch.float64, device="cuda")
    Cm = torch.empty(N, N, dtype=torch.float64, device="cuda")
    fl = 2.0 * N ** 3
    for _ in range(3):
        torch.matmul(A, B, out=Cm)
    best = min(timed(dp.stream, lambda: torch.matmul(A, B, out=Cm)) for _ in range(10))
    cs = ClockSampler(local)
    cs.start()
    reps, ms = 0, 0.0
    while ms < 4000.0:
        ms += timed(dp.stream, lambda: torch.matmul(A, B, out=Cm), reps=16)
        reps += 16
    clk = cs.stop()
    out["dgemm_8192"] = {"burst_tflops": fl / best / 1e9, "sustained_tflops": fl * reps / ms / 1e9,
                         "sustained_s": ms / 1e3, "clocks": clk, "what": "torch.matmul float64 (cuBLAS), yardstick only"}
    del A, B, Cm
    sink = torch.zeros(16, dtype=torch.float64, device="cuda")
    # the register-only DMMA loop in two shapes: 3 CTAs × 4 warps per SM (the residency of the GEMM kernel) and
    # 4 CTAs × 8 warps per SM (round 1's probe, which reads ≈ 20 % low on this part: too many warps per scheduler)
    out["dmma_probe"] = {"what": "dmrgk_probe_fp64: register-only mma.sync.m8n8k4.f64 loop, full grid"}
    for kind, shape, long_iters in ((4, "3x4_warps_per_sm", 3200000), (0, "4x8_warps_per_sm", 1200000)):
        dmrgk.probe_fp64(dp.ctx, kind, 20000, sink, dp.stream)
        burst = 0.0
        for _ in range(5):
            box = {}
            ms = timed(dp.stream, lambda: box.setdefault("f", dmrgk.probe_fp64(dp.ctx, kind, 20000, sink, dp.stream)))
            burst = max(burst, box["f"] / ms / 1e9)
        cs = ClockSampler(local)
        cs.start()
        box = {}
        ms = timed(dp.stream, lambda: box.setdefault("f", dmrgk.probe_fp64(dp.ctx, kind, long_iters, sink, dp.stream)))
        clk = cs.stop()
        out["dmma_probe"][shape] = {"burst_tflops": burst, "sustained_tflops": box["f"] / ms / 1e9, "sustained_s": ms / 1e3, "clocks": clk}
    box = {}
    ms = timed(dp.stream, lambda: box.setdefault("f", dmrgk.probe_fp64(dp.ctx, 1, 300000, sink, dp.stream)))
    out["dfma_probe"] = {"sustained_tflops": box["f"] / ms / 1e9, "sustained_s": ms / 1e3,
                         "what": "dmrgk_probe_fp64 kind 1: register-only fma.rn.f64 loop"}
    return out


def read_traffic_table(workload, kernel_hash):
    """dram bytes per GEMM launch from the committed ncu capture table (profiles/traffic.csv:
    workload,kernel_hash,traffic_bytes_per_launch,alg_bytes_per_launch,capture).  Only a row taken with the
    SAME kernel sources counts; otherwise traffic is null (never a stale constant)."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        rows = [l.strip().split(",") for l in open(path) if l.strip() and not l.startswith("#")]
    except OSError:
        return None, "no profiles/traffic.csv"
    for r in rows:
        if len(r) >= 5 and r[0] == workload and r[1] == kernel_hash:
            return float(r[2]), f"{r[4]} (kernel sources {kernel_hash}); algorithmic bytes per launch {float(r[3]):.3e}"
    return None, f"no ncu capture of workload {workload} with kernel sources {kernel_hash} in profiles/traffic.csv"


def davidson_bench(dp, wl, args, world, local, steps, warmup, make_davidson=None):
    """W warm-up + K timed Davidson steps (each exactly one H_eff apply) on a built problem."""
    import torch
    import torch.distributed as dist
    import workloads as wlmod
    from paper_2311_14106_b200 import dmrgk
    h = dp.heff
    psi = dp.psi_fill(wl.seed, wlmod.PSI_STREAM)
    make_davidson = make_davidson or dp.davidson
    dav = make_davidson(m_max=args.m_max, tol=0.0, max_iter=1 << 30)     # tol 0: never stops early
    dav.start(psi)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        dav.step()
    barrier()
    h.profile(True)
    dmrgk.launch_count(reset=True)
    clocks = ClockSampler(local)
    clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(dp.stream)
    m_seen = []
    for _ in range(steps):
        m_seen.append(dav.query()[0])
        theta, rho, _ = dav.step()
    e1.record(dp.stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = dmrgk.launch_count()
    prof_ms, prof_n = h.profile_read()
    h.profile(False)
    clk = clocks.stop()
    ms_total = max_over_ranks(ms_total, world, "cuda")
    return {"psi": psi, "ms_step": ms_total / steps, "launches": int(launches), "prof_ms": prof_ms, "prof_n": prof_n,
            "clocks": clk, "theta": theta, "rho": rho, "m_range": [min(m_seen), max(m_seen)] if m_seen else None}


EXTRA_ROWS = [   # (key, bench.py arguments): the other workloads DESIGN.md quotes, each run as its own process
    ("config1", ["--config", "1", "--steps", "20", "--warmup", "5", "--no-extras"]),
    ("config3b", ["--config", "3b", "--steps", "3", "--warmup", "3", "--no-cpu", "--no-extras"]),
    ("config4rs", ["--config", "4rs", "--steps", "5", "--warmup", "3", "--no-cpu", "--no-extras"]),
    ("config5r", ["--config", "5r", "--steps", "3", "--warmup", "3", "--no-cpu", "--no-extras"]),
    ("config5", ["--config", "5", "--steps", "3", "--warmup", "3", "--no-cpu", "--no-extras"]),
    ("su2", ["--op", "su2", "--steps", "3", "--warmup", "3"]),
    ("expect", ["--op", "expect", "--steps", "3", "--warmup", "2"]),
    ("enlarge", ["--op", "enlarge", "--steps", "10", "--warmup", "3"]),
]


def brief(line):
    """The fields of a bench line that an extras row keeps."""
    cfg, roof = line.get("config", {}), line.get("roofline", {})
    row = {"metric": line.get("metric"), "value": line.get("value"), "unit": line.get("unit"), "workload": cfg.get("workload"),
           "ms_per_step": line.get("ms_per_step"), "steps": line.get("steps"), "warmup": line.get("warmup"),
           "gpu_launches": line.get("gpu_launches"),
           "roofline": {k: roof.get(k) for k in ("bound", "achieved", "peak", "unit", "frac", "frac_of_cublas_dgemm") if k in roof},
           "clocks": line.get("clocks")}
    for k in ("apply_burst", "cpu_baseline"):
        if k in line:
            row[k] = line[k]
    if "e2e" in line:
        row["e2e_value"] = line["e2e"].get("value")
    for k in ("K_pairs", "tasks", "flops_alg_per_apply", "staged_ops", "staged_bytes_per_apply", "op_bytes_resident",
              "davidson_m_of_timed_steps", "pairs_per_second", "tiles", "kept_bytes", "formed_bytes"):
        if k in cfg:
            row[k] = cfg[k]
    return row


def extra_rows_in_subprocesses():
    """Every other row the documents quote, measured in the same driver run: one `python bench.py …` process per row,
    started after the headline workload's device memory has been released (the rows need up to 150 GB themselves).
    A row that fails, times out or runs out of memory records its error; it cannot touch the headline numbers."""
    import gc
    import subprocess
    import torch
    gc.collect()
    torch.cuda.empty_cache()
    free, total = torch.cuda.mem_get_info()
    rows = {"device_free_bytes_before_rows": int(free), "how": "python bench.py <args> per row, one process each, one after the other"}
    for key, argv in EXTRA_ROWS:
        t0 = time.perf_counter()
        try:
            p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + argv, cwd=ROOT, capture_output=True,
                               text=True, timeout=900)
            lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
            if p.returncode != 0 or not lines:
                rows[key] = {"error": f"rc {p.returncode}: {(p.stderr or p.stdout)[-300:]}"}
            else:
                rows[key] = brief(json.loads(lines[-1]))
                rows[key]["args"] = " ".join(argv)
        except Exception as exc:
            rows[key] = {"error": repr(exc)[:300]}
        rows[key]["wall_s"] = round(time.perf_counter() - t0, 1)
    a, b_ = rows.get("config5"), rows.get("config5r")
    if a and b_ and "ms_per_step" in a and "ms_per_step" in b_:   # row a3: what the staging costs, and the PCIe rate it sustains
        a["exposed_copy_ms_per_step"] = a["ms_per_step"] - b_["ms_per_step"]
        if a.get("staged_bytes_per_apply"):
            a["h2d_gbs_over_the_step"] = a["staged_bytes_per_apply"] / a["ms_per_step"] / 1e6
    return rows


def run_ours(args):
    import torch
    out = measure_ours(args)      # every device buffer of the headline workload dies with that frame
    if out is None:
        return
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank == 0 and world == 1 and not args.no_extras and args.config == "4":
        try:
            out.setdefault("extras", {}).update(extra_rows_in_subprocesses())
        except Exception as exc:
            out.setdefault("extras", {})["rows_error"] = repr(exc)[:300]
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def measure_ours(args):
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
    if b.built_hash() != b.source_hash():       # missing or stale binary: rank 0 rebuilds, the others wait
        if rank == 0:
            b.build()
        if world > 1:
            dist.barrier()
    dmrgk.load()

    wl = make_workload(args.config)
    if args.shard == "k" and world > 1:
        run_sharded(args, wl, rank, world, local)
        return None
    staged = wlmod.config5_staged_ops(wl) if args.config == "5" else []
    opts = {"ring_bytes": 6 << 30} if staged else {}
    if args.kernel:
        opts["kernel"] = args.kernel
    dp = problem.from_workload(wl, device=local, pinned=staged, **opts)
    torch.cuda.synchronize()
    h = dp.heff
    n = dp.layout.n_padded

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- the timed region: K Davidson steps (each exactly one H_eff apply) --------------------
    r = davidson_bench(dp, wl, args, world, local, args.steps, args.warmup)
    psi, ms_step, clk, prof_ms, prof_n = r["psi"], r["ms_step"], r["clocks"], r["prof_ms"], r["prof_n"]
    value = aggregate_tflops(h.flops_alg, world, ms_step)

    # ---- burst: best of 10 single applies, each timed alone (SURVEY §8(d) timing protocol) --------
    sig = dp.new_vector(zero=False)
    burst_ms = min(timed(dp.stream, lambda: dp.apply(psi, sig)) for _ in range(10))

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
    ms_e2e = timed(dp.stream, lambda: h.apply_host(ph, sh, pdev, sdev, dp.workspace, dp.stream, dp.copy_stream),
                   reps=args.steps) / args.steps
    clk_e2e = clocks_e2e.stop()
    ms_e2e = max_over_ranks(ms_e2e, world, "cuda")
    # ---- the FP64 ceilings of this box, measured live (outside every timed region) ---------------
    ceil = measure_fp64_ceiling(dp, local)
    n_sm = dp.ctx.query()[0]
    sm_max = clk.get("sm_max_mhz") or 1965.0
    peak_derived = n_sm * 128 * sm_max * 1e6 / 1e12     # one DMMA.8x8x4 per 4 clk per SM
    peak_measured = max(ceil["dmma_probe"]["3x4_warps_per_sm"]["sustained_tflops"], ceil["dmma_probe"]["4x8_warps_per_sm"]["sustained_tflops"],
                        ceil["dgemm_8192"]["sustained_tflops"], ceil["dfma_probe"]["sustained_tflops"])
    probe_ratio = ceil["dmma_probe"]["3x4_warps_per_sm"]["sustained_tflops"] / peak_derived

    # ---- a8 vector kernels alone: achieved HBM GB/s against MEASURED_PEAKS.json hbm_gbs ------------
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
    time_vec = lambda fn: (fn(), timed(dp.stream, fn, reps=10) / 10)[1]
    t_dot = time_vec(lambda: dmrgk.vec_multi_dot(dp.ctx, n, mv, dp.V, n, psi, outv, scratch, dp.stream))
    t_axpy = time_vec(lambda: dmrgk.vec_multi_axpy(dp.ctx, n, mv, dp.V, n, coefv, -1.0, 1.0, yv, dp.stream))
    t_res = time_vec(lambda: dmrgk.vec_residual(dp.ctx, n, mv, dp.V, dp.W, n, coefv, yv, outv, scratch, dp.stream))
    gbs = lambda nvec, ms: nvec * n * 8 / ms / 1e6
    vec = {"n_doubles": int(n), "m": mv, "peak_gbs": hbm_peak, "peak_source": hbm_src,
           "multi_dot": {"ms": t_dot, "gbs": gbs(mv + 1, t_dot), "frac": gbs(mv + 1, t_dot) / hbm_peak},
           "multi_axpy": {"ms": t_axpy, "gbs": gbs(mv + 2, t_axpy), "frac": gbs(mv + 2, t_axpy) / hbm_peak},
           "residual": {"ms": t_res, "gbs": gbs(2 * mv + 1, t_res), "frac": gbs(2 * mv + 1, t_res) / hbm_peak}}

    traffic, traffic_note = read_traffic_table(wl.name, b.kernel_hash())

    # device time of the GEMM region of the applies (phase-1/phase-2 launches overlap on two streams, so
    # per-launch durations are not additive; the span from the first to the last launch of each apply
    # is what is timed, and it includes the split-k reduce launches)
    gemm_ms = prof_ms["apply"]
    gemm_n = prof_n["p1"] + prof_n["p2"]
    achieved = h.flops_alg * args.steps / gemm_ms / 1e9 if gemm_ms > 0 else None
    su = dp.setup_seconds
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "M_A": wl.M_A, "M_B": wl.M_B, "K_pairs": len(wl.terms), "tasks": h.n_tasks,
                   "flops_alg_per_apply": h.flops_alg, "flops_exec_over_alg": h.flops_exec / h.flops_alg if h.flops_alg else None,
                   "op_bytes_resident": int(dp.op_arena.numel() * 8),
                   "psi_elems": dp.layout.n_elems, "davidson_m_max": args.m_max,
                   "davidson_m_of_timed_steps": r["m_range"], "davidson_m_what": "subspace size at the start of the timed steps, [min, max]: "
                   "m grows by one per step and collapses to 1 at m_max, so the vector-kernel share of a step varies with it",
                   "parallelism": "replicas only",
                   "l2": "operator arena (>> 126 MB L2) is streamed once per step; no flush needed",
                   "setup_s": {"tables": round(su["structures"] + su["tasklist"], 3), "tables_what": "sector/block tables + "
                               "task-list build and upload (the paper's 'Tables', PAPER.md:142)", "seeded_fill": round(su["fill"], 3),
                               "seeded_fill_what": "harness fill of the operator arena (stands in for operators a sweep already holds)"},
                   "chunks": h.n_chunks, "source_hash": dmrgk.source_hash(), "kernel_variant": args.kernel,
                   "staged_ops": len(staged), "staged_bytes_per_apply": int(sum(dp.ops[i].n_padded for i in staged) * 8)},
        "davidson_step_ms": ms_step, "theta_last": r["theta"], "resnorm_last": r["rho"],
        "apply_burst": {"ms": burst_ms, "tflops": h.flops_alg / burst_ms / 1e9, "what": "best of 10 single applies, each timed alone"},
        "pct_of_fp64_peak": 100.0 * value / world / peak_derived,
        "e2e": {"value": world * h.flops_alg / ms_e2e / 1e9, "unit": UNIT, "ms_per_step": ms_e2e,
                "what": "dmrgk_heff_apply_host: pinned ψ H2D, apply, σ D2H",
                "h2d_bytes_per_step": int(n * 8), "d2h_bytes_per_step": int(n * 8), "clocks": clk_e2e},
        "gpu_launches": r["launches"],
        "roofline": {"bound": "tensor", "kernel": "heff_gemm_dmma_kernel (a5 + a6)", "achieved": achieved,
                     "peak": peak_derived, "unit": "TFLOP/s", "frac": (achieved / peak_derived) if achieved else None,
                     "peak_source": f"of derived: {n_sm} SMs x 128 FP64 flop/clk x {sm_max:.0f} MHz (MEASURED_PEAKS.json has no FP64 "
                                    "figure); the measured ceilings of this run are in fp64_ceilings",
                     "peak_measured": peak_measured,
                     "frac_of_measured": (achieved / peak_measured) if achieved else None,
                     "peak_measured_source": "best sustained ceiling measured in this run: register-only DMMA loop (two shapes), DFMA loop, cuBLAS DGEMM 8192^3",
                     "peak_cublas_dgemm": ceil["dgemm_8192"]["sustained_tflops"],
                     "frac_of_cublas_dgemm": (achieved / ceil["dgemm_8192"]["sustained_tflops"]) if achieved else None,
                     "peak_cublas_dgemm_source": "cuBLAS DGEMM 8192^3 sustained in this run (a library-measured FP64 ceiling, not this repo's kernel)",
                     "probe_over_derived": probe_ratio,
                     "probe_agrees_with_derived": bool(abs(probe_ratio - 1.0) <= 0.03),
                     "launches": int(gemm_n), "avg_launch_ms": gemm_ms / max(gemm_n, 1),
                     "kernel_ms_per_step": gemm_ms / args.steps, "reduce_launches": int(prof_n["reduce"]),
                     "traffic": traffic, "traffic_note": traffic_note},
        "fp64_ceilings": ceil,
        "vector_kernels": vec,
        "clocks": clk,
    }
    # ---- other §8 rows in the same driver-run line (not the headline; each its own workload) ------
    if rank == 0 and world == 1 and not args.no_extras and args.config == "4":
        extras = {}
        try:
            extras["renorm_config4_left_half"], rp_, _, _ = renorm_numbers(dp, wl, steps=5, warmup=3, local=local, peak=peak_derived)
            del rp_
            torch.cuda.empty_cache()
        except Exception as exc:       # an extra must never take the headline line down
            extras["renorm_config4_left_half"] = {"error": repr(exc)[:300]}
        for name in ("3", "2"):
            try:
                wl2 = make_workload(name)
                dp2 = problem.from_workload(wl2, device=local, ctx=dp.ctx)
                r2 = davidson_bench(dp2, wl2, args, 1, local, steps=10, warmup=3)
                sig2 = dp2.new_vector(zero=False)
                b2 = min(timed(dp2.stream, lambda: dp2.apply(r2["psi"], sig2)) for _ in range(10))
                f2 = dp2.heff.flops_alg
                extras["config" + name] = {"workload": wl2.name, "davidson_step_ms": r2["ms_step"], "tflops": f2 / r2["ms_step"] / 1e9,
                                           "frac_of_derived": f2 / r2["ms_step"] / 1e9 / peak_derived,
                                           "apply_burst_ms": b2, "apply_burst_tflops": f2 / b2 / 1e9,
                                           "launches_per_step": r2["launches"] / 10, "flops_alg_per_apply": f2,
                                           "clocks": r2["clocks"]}
                del dp2, r2, sig2
                torch.cuda.empty_cache()
            except Exception as exc:
                extras["config" + name] = {"error": repr(exc)[:300]}
        out["extras"] = extras
    if rank == 0 and world == 1 and not args.no_cpu:
        out["cpu_baseline"] = cpu_baseline_from_device(dp, wl, args)
    return out


def run_sharded(args, wl, rank, world, local):
    """--shard k at N > 1: the operator-pair list is split over the ranks (balanced
    by flops and bytes), ψ is replicated, every apply is followed by ONE NCCL all-reduce (sum) of the
    ψ-sized σ over NVLink, the Davidson iteration runs replicated.  Total work is fixed ⇒ "strong"
    scaling; value = flops of the WHOLE list ÷ max-over-ranks step time.  UNMEASURED on hardware in this
    build (one GPU per call); covered by tests/test_shard.py."""
    import torch
    import torch.distributed as dist
    from paper_2311_14106_b200 import dmrgk, shard
    sp = shard.ShardedProblem(wl, rank, world, device=local)
    torch.cuda.synchronize()
    flops_total = float(shard.term_costs(wl)[0].sum())
    r = davidson_bench(sp.dp, sp.wl, args, world, local, args.steps, args.warmup, make_davidson=sp.davidson)
    ms_step = r["ms_step"]
    n = sp.dp.layout.n_padded
    sm_max = r["clocks"].get("sm_max_mhz") or 1965.0
    peak = sp.dp.ctx.query()[0] * 128 * sm_max * 1e6 / 1e12
    gemm_ms = max_over_ranks(r["prof_ms"]["apply"], world, "cuda")
    out = {"metric": METRIC, "value": flops_total / ms_step / 1e9, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": wl.name, "parallelism": f"k-sharded x{world}: pair list split by flops and bytes, psi replicated, "
                      "one NCCL all-reduce (sum) of sigma per apply", "K_pairs": len(wl.terms),
                      "pairs_per_rank": [len(s) for s in sp.shards], "flops_per_rank": [st["flops"] for st in sp.stats],
                      "op_bytes_per_rank": [st["bytes"] for st in sp.stats], "flops_alg_per_apply": flops_total,
                      "allreduce_bytes_per_apply": int(n * 8), "source_hash": dmrgk.source_hash(),
                      "l2": "operator arenas (>> 126 MB L2) are streamed once per step; no flush needed"},
           "gpu_launches": r["launches"], "theta_last": r["theta"], "resnorm_last": r["rho"],
           "roofline": {"bound": "tensor", "kernel": "heff_gemm_dmma_kernel (a5 + a6), slowest rank", "peak": peak * world,
                        "achieved": flops_total * args.steps / gemm_ms / 1e9 if gemm_ms > 0 else None, "unit": "TFLOP/s",
                        "frac": (flops_total * args.steps / gemm_ms / 1e9) / (peak * world) if gemm_ms > 0 else None,
                        "peak_source": f"of derived: {world} x 148 SMs x 128 FP64 flop/clk x {sm_max:.0f} MHz", "traffic": None},
           "e2e": None, "clocks": r["clocks"]}
    if rank == 0:
        print(json.dumps(out), flush=True)
    dist.destroy_process_group()


def cpu_baseline_from_device(dp, wl, args, budget_s=25.0):
    """The oracle (oracle.heff.sigma_blockwise, NumPy/BLAS, as it stands) on the host cores, on a
    stratified sample of the operator pairs (every CPU_EVERY-th pair ≈ 5 %) with all ψ
    blocks; operator values are read back D2H from the device arena (bit-identical to the host
    recipe, and ~100× faster than regenerating them)."""
    from oracle import heff as oheff
    from workloads import fill_psi_host
    every = CPU_EVERY[args.config]
    sub, ids = sample_terms(wl, every)
    need = sorted({i for t in sub.terms for i in (t.L, t.R) if i is not None})
    ops = [{"half": s.half, "dq": tuple(s.dq), "parity": s.parity, "blocks": {}} for s in wl.ops]
    for i in need:
        ops[i]["blocks"] = dp.read_op_blocks(i) if i in dp.op_views else {}
    terms = [(t.L, t.R, t.coef, t.trans_L, t.trans_R) for t in sub.terms]
    pb = oheff.Problem(wl.n_charges, list(wl.sectors_A), list(wl.sectors_B), tuple(wl.target), ops, terms,
                       fill_psi_host(wl), wl.name + "_sample")
    fl = float(oheff.flops_alg(pb))
    reps, t0 = 0, time.perf_counter()
    while reps < 2 or (time.perf_counter() - t0 < budget_s and reps < 200):
        oheff.sigma_blockwise(pb)
        reps += 1
    sec = (time.perf_counter() - t0) / reps
    tiers = {}
    if args.config == "1":      # the oracle's wall time per σ, both tiers
        t0 = time.perf_counter()
        oheff.sigma_dense(pb)
        tiers = {"oracle_t2_dense_kronecker_s": time.perf_counter() - t0, "oracle_t3_blockwise_s": sec}
    return {**tiers, "value": fl / sec / 1e12, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
            "sample": f"oracle.heff.sigma_blockwise on every {every}th operator pair ({len(ids)} of {len(wl.terms)} = "
                      f"{100.0 * len(ids) / len(wl.terms):.1f} %), all ψ blocks, {fl:.3e} flop x {reps} repeats, "
                      "operator values read back from the device arena"}


def renorm_numbers(dp, wl, steps, warmup, local, peak):
    """Time the renormalisation of every enlarged-block operator of the left half of a built problem
     to D kept states; returns (numbers, RenormProblem, sectors_new, phi table)."""
    import torch
    import workloads as wlmod
    from paper_2311_14106_b200 import dmrgk, problem
    sectors_new, table = wlmod.renorm_basis(wl)
    rp = problem.RenormProblem(dp, "A", sectors_new)
    rp.fill_phi(wl.seed, wlmod.PHI_STREAM)
    rp.build([(wl.ops[i].dq, wl.ops[i].parity) for i in rp.idx])
    for _ in range(warmup):
        rp.apply()
    torch.cuda.synchronize()
    clocks = ClockSampler(local)
    clocks.start()
    dmrgk.launch_count(reset=True)
    ms = timed(dp.stream, rp.apply, reps=steps) / steps
    launches = dmrgk.launch_count()
    clk = clocks.stop()
    burst = min(timed(dp.stream, rp.apply) for _ in range(5))
    val = rp.plan.flops / ms / 1e9
    nums = {"workload": wl.name + "_renorm_left_half", "ms_per_step": ms, "tflops": val, "frac_of_derived": val / peak,
            "burst_ms": burst, "burst_tflops": rp.plan.flops / burst / 1e9,
            "operators": len(rp.idx), "blocks": rp.plan.n_tasks, "M_enlarged": wl.M_A,
            "M_kept": sum(d for _, d in sectors_new), "flops_per_apply": rp.plan.flops,
            "in_bytes": int(sum(op.n_padded for op in rp.ops_in) * 8),
            "out_bytes": int(sum(op.n_padded for op in rp.ops_out) * 8),
            "launches_per_step": launches / steps, "clocks": clk}
    return nums, rp, sectors_new, table


def run_renorm(args):
    """--op renorm: one step = the renormalisation O' = Phi^T O Phi of every enlarged-block operator of
    the left half of the workload to D kept states; not the headline metric."""
    import torch
    import workloads as wlmod
    from paper_2311_14106_b200 import problem
    from oracle import renorm as orenorm
    torch.cuda.set_device(0)
    wl = make_workload(args.config)
    dp = problem.from_workload(wl)
    n_sm = dp.ctx.query()[0]
    peak = n_sm * 128 * 1965.0 * 1e6 / 1e12
    nums, rp, sectors_new, table = renorm_numbers(dp, wl, args.steps, args.warmup, 0, peak)
    clk = nums.pop("clocks")
    val, ms = nums["tflops"], nums["ms_per_step"]
    out = {"metric": "renorm_fp64_tflops", "value": val, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": dict(nums, l2="operator arenas (>> 126 MB L2) are streamed once per step"),
           "gpu_launches": int(nums["launches_per_step"] * args.steps),
           "roofline": {"bound": "tensor", "kernel": "heff_gemm_dmma_kernel (renormalisation work lists)", "achieved": val,
                        "peak": peak, "unit": "TFLOP/s", "frac": val / peak, "traffic": None,
                        "peak_source": f"of derived: {n_sm} SMs x 128 FP64 flop/clk x 1965 MHz",
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


def run_enlarge(args):
    """--op enlarge: one step = forming every operator of the next enlarged left block,
    O_A' = sum_j coef_j (X_j P^pi) (x) y_j (second half), from kept operators with the
    sector structure of config 4 at D = 4096 kept states and a Hubbard site; 4 block sites (8 modes) + 1 site
    + 13 sites to the right, synthetic symmetric t, V (seeded).  HBM-bound: its own metric (GB/s)."""
    import numpy as np
    import torch
    import workloads as wlmod
    from workloads.rng import normal12
    from paper_2311_14106_b200 import dmrgk, blockops
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    wl = make_workload("4")
    sectors_K, _ = wlmod.renorm_basis(wl)
    n_modes, nA = 36, 8
    mc = np.array([(1, 0), (0, 1)] * (n_modes // 2), dtype=np.int64)
    A, S, right = list(range(nA)), [nA, nA + 1], list(range(nA + 2, n_modes))
    g = normal12(11, 1, np.arange(n_modes * n_modes)).reshape(n_modes, n_modes)
    T = 0.5 * (g + g.T)
    G = normal12(11, 2, np.arange(n_modes ** 4)).reshape((n_modes,) * 4) * 0.1
    V = G + G.transpose(3, 2, 1, 0)
    # keep only charge-conserving coefficients (n_up, n_down are conserved by Eq. (1) of the Hubbard-type models)
    up = mc[:, 0]
    T = T * (up[:, None] == up[None, :])
    V = V * ((up[:, None, None, None] + up[None, :, None, None]) == (up[None, None, :, None] + up[None, None, None, :]))
    t0 = time.perf_counter()
    site, lists = blockops.enlarge_left_lists(T, V, mc, A, S, right)
    t_lists = time.perf_counter() - t0
    ctx = dmrgk.Ctx(0)
    st = torch.cuda.current_stream()
    sp_K = dmrgk.Space(ctx, 2, sectors_K)
    sectors_E = blockops.enlarged_sectors(sectors_K, site.charges.tolist())
    sp_E = dmrgk.Space(ctx, 2, sectors_E)
    keys_A, keys_Ap = blockops.left_block_keys(A, S + right), blockops.left_block_keys(A + S, right)

    def alloc(space, keys):
        ops = [dmrgk.Op(ctx, space, *blockops.operator_spec(k, mc)) for k in keys]
        arena = torch.zeros(max(sum(o.n_padded for o in ops), 16), dtype=torch.float64, device=dev)
        o = 0
        for op in ops:
            op.bind_device(arena[o:o + op.n_padded] if op.n_padded else arena[0:16])
            o += op.n_padded
        return ops, arena

    ops_K, arena_K = alloc(sp_K, keys_A)
    o = 0
    for i, op in enumerate(ops_K):
        if op.n_padded:
            op.fill_normal(arena_K[o:o + op.n_padded], 11, 100 + i, 1, 0, st)
        o += op.n_padded
    ops_E, arena_E = alloc(sp_E, keys_Ap)
    index_K = {k: i for i, k in enumerate(keys_A)}
    terms = [(oi, None if k is None else ops_K[index_K[k]], tr, bool(pi), 1.0, y)
             for oi, key in enumerate(keys_Ap) for (k, tr, y, pi) in lists[key]]
    t0 = time.perf_counter()
    enl = dmrgk.Enlarge(ctx, sp_K, sp_E, site.charges, ops_E, terms)
    t_plan = time.perf_counter() - t0
    for _ in range(args.warmup):
        enl.apply(st)
    clocks = ClockSampler(0)
    clocks.start()
    dmrgk.launch_count(reset=True)
    ms = timed(st, lambda: enl.apply(st), reps=args.steps) / args.steps
    launches = dmrgk.launch_count()
    clk = clocks.stop()
    zero_bytes = int(arena_E.numel() * 8)
    # algorithmic HBM bytes: every kept operator read once, every formed operator written once (its zero
    # blocks included).  The gather reads each kept block once PER PRODUCT (enl.bytes_read, served by L2:
    # the kept set is small), so that figure is reported as L2-level traffic, not as HBM work.
    kept_bytes = int(arena_K.numel() * 8)
    moved = kept_bytes + zero_bytes
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        src = "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        hbm_peak, src = 6650.0, "fallback (B200_PROFILING.md)"
    gbs = moved / ms / 1e6
    print(json.dumps({
        "metric": "enlarge_gbs", "value": gbs, "unit": "GB/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "enlarge_left_block_config4_sectors_D4096_hubbard_site", "kept_states": sum(d for _, d in sectors_K),
                   "enlarged_states": sum(d for _, d in sectors_E), "kept_operators": len(ops_K), "formed_operators": len(ops_E),
                   "products": len(terms), "tiles": enl.n_tiles, "sources": enl.n_sources, "kept_bytes": kept_bytes,
                   "formed_bytes": zero_bytes, "gather_reads_l2_bytes": enl.bytes_read, "gather_writes_bytes": enl.bytes_written,
                   "l2_read_gbs": enl.bytes_read / ms / 1e6, "host_lists_s": round(t_lists, 3),
                   "host_plan_s": round(t_plan, 3), "l2": "formed operators (>> 126 MB L2) are written once per step"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "kernel": "enlarge_gather_kernel (+ zero fill)", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                     "frac": gbs / hbm_peak, "peak_source": src, "traffic": None},
        "clocks": clk}), flush=True)


def flat_workload(dim_a, dim_b, n_half=8, seed=11):
    """A lattice-shaped operator-pair list (families F0-F4 of n_half spinless modes per half) over FLAT sectors:
    every A sector has dim_a states, every B sector dim_b — all blocks the same shape, so that the cost of ragged
    tile edges can be read off by comparing shapes (--op ragged)."""
    from workloads.configs import Workload, _family_builder, spinless_term_structure
    sa = [((q,), dim_a) for q in range(n_half + 1)]
    sb = [((q,), dim_b) for q in range(n_half + 1)]
    wl = Workload(f"flat_{dim_a}x{dim_b}", seed, 1, sa, sb, (n_half,))
    sh = spinless_term_structure(n_half, n_half)
    return _family_builder(wl, sh[0], sh[1])


def run_ragged(args):
    """--op ragged: the product kernel on flat-sector workloads — multiples of the 64-wide tile against ragged
    dims — with the phases timed one after the other (dmrgk_heff_profile(2)).  Phase 1 is m' x n with k = m,
    phase 2 m' x n' with k = n (stacked); here m = m' = dim_a, n = n' = dim_b.  Not a product number: it is
    the evidence for the balanced tiling of DESIGN.md §4.1 (profiles/r2_ragged.md)."""
    import torch
    import workloads as wlmod
    from paper_2311_14106_b200 import dmrgk, problem
    torch.cuda.set_device(0)
    dmrgk.load()
    rows = []
    for da, db in ((512, 512), (500, 512), (512, 500), (500, 500), (640, 640), (650, 650), (256, 256), (250, 250), (128, 128), (120, 120)):
        wl = flat_workload(da, db)
        opts = {"kernel": args.kernel} if args.kernel else {}
        dp = problem.from_workload(wl, device=0, **opts)
        psi = dp.psi_fill(wl.seed, wlmod.PSI_STREAM)
        sig = dp.new_vector(zero=False)
        for _ in range(3):
            dp.apply(psi, sig)
        ms = min(timed(dp.stream, lambda: dp.apply(psi, sig)) for _ in range(10))
        h = dp.heff
        h.profile(2)
        for _ in range(5):
            dp.apply(psi, sig)
        torch.cuda.synchronize()
        pm, _ = h.profile_read()
        h.profile(0)
        f1 = 2.0 * da * da * db * h.n_tasks      # identity factors of F0 included: approximate split of flops_alg
        f2 = 2.0 * da * db * db * h.n_tasks
        rows.append({"dim_a": da, "dim_b": db, "tasks": h.n_tasks, "chunks": h.n_chunks, "apply_ms": round(ms, 3),
                     "apply_tflops": round(h.flops_alg / ms / 1e9, 2),
                     "phase1_ms": round(pm["p1"] / 5, 3), "phase2_ms": round(pm["p2"] / 5, 3),
                     "phase1_tflops": round(f1 / (pm["p1"] / 5) / 1e9, 2), "phase2_tflops": round(f2 / (pm["p2"] / 5) / 1e9, 2)})
        del dp, psi, sig
        torch.cuda.empty_cache()
    print(json.dumps({"op": "ragged", "source_hash": dmrgk.source_hash(), "kernel_variant": args.kernel, "rows": rows}), flush=True)


def run_su2(args):
    """--op su2: one step = one apply of the SU(2) spin-adapted singlet H_eff
    on the synthetic spin-adapted workload `workloads.su2_singlet_workload()`: 18 orbitals per half, 190 sectors
    (N, 2S) holding M = 12288 multiplets (D = 4096 kept multiplets × 3 site multiplets), K = 2702 pairs of reduced
    operators, recoupling scalars from paper_2311_14106_b200/su2.py.  Its own metric, not the headline."""
    import torch
    import workloads as wlmod
    from paper_2311_14106_b200 import dmrgk, problem, su2
    torch.cuda.set_device(0)
    dmrgk.load()
    wl = wlmod.su2_singlet_workload()
    terms = [(t.L, t.R, t.coef, t.trans_L, t.trans_R) for t in wl.terms]
    psi_a = [a for (a, _, _, _, _) in wlmod.psi_block_table(wl.sectors_A, wl.sectors_B, wl.target)]
    table = su2.block_coef_table(wl.sectors_A, psi_a, su2.pair_meta(wl.ops, terms, wl.ranks))
    opts = {"kernel": args.kernel} if args.kernel else {}
    dp = problem.from_workload(wl, block_coef=table, **opts)
    h = dp.heff
    psi = dp.psi_fill(wl.seed, wlmod.PSI_STREAM)
    sig = dp.new_vector(zero=False)
    for _ in range(max(args.warmup, 3)):
        dp.apply(psi, sig)
    burst = min(timed(dp.stream, lambda: dp.apply(psi, sig)) for _ in range(5))
    clocks = ClockSampler(0)
    clocks.start()
    dmrgk.launch_count(reset=True)
    ms = timed(dp.stream, lambda: dp.apply(psi, sig), reps=args.steps) / args.steps
    launches = dmrgk.launch_count()
    clk = clocks.stop()
    n_sm = dp.ctx.query()[0]
    peak = n_sm * 128 * (clk.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
    val = h.flops_alg / ms / 1e9
    print(json.dumps({
        "metric": "su2_singlet_heff_apply_fp64_tflops", "value": val, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "sectors": len(wl.sectors_A), "largest_sector": max(d for _, d in wl.sectors_A),
                   "M_multiplets": wl.M_A, "K_pairs": len(wl.terms), "tasks": h.n_tasks, "psi_blocks": len(psi_a),
                   "zero_scalars": int((table == 0).sum()), "flops_alg_per_apply": h.flops_alg,
                   "op_bytes_resident": int(dp.op_arena.numel() * 8), "chunks": h.n_chunks, "source_hash": dmrgk.source_hash(),
                   "l2": "operator arena (>> 126 MB L2) is streamed once per step"},
        "apply_burst": {"ms": burst, "tflops": h.flops_alg / burst / 1e9},
        "gpu_launches": int(launches),
        "roofline": {"bound": "tensor", "kernel": "heff_gemm_dmma_kernel (spin-adapted work lists)", "achieved": val, "peak": peak,
                     "unit": UNIT, "frac": val / peak, "traffic": None, "peak_source": f"of derived: {n_sm} SMs x 128 FP64 flop/clk x max SM clock"},
        "clocks": clk}), flush=True)


def run_expect(args):
    """--op expect: one step = the per-pair expectation values e_k = <psi, c_k (L_k x R_k) psi> of EVERY operator pair
    of the workload (dmrgk_heff_expect: the reduced density matrices are such lists
    with the pairs {c+_i c_j}, {c+_i c+_j c_k c_l}): phase 1 as in the matvec, phase 2 per pair, fused dots.
    Default workload: config 3.  Its own metric."""
    import torch
    import workloads as wlmod
    from paper_2311_14106_b200 import dmrgk, problem
    torch.cuda.set_device(0)
    dmrgk.load()
    wl = make_workload(args.config if args.config != "4" else "3")
    dp = problem.from_workload(wl, per_pair_output=1)
    h = dp.heff
    psi = dp.psi_fill(wl.seed, wlmod.PSI_STREAM)
    K = len(wl.terms)
    for _ in range(max(args.warmup, 2)):
        out = dp.expect(psi, K)
    clocks = ClockSampler(0)
    clocks.start()
    dmrgk.launch_count(reset=True)
    ms = timed(dp.stream, lambda: dp.expect(psi, K), reps=args.steps) / args.steps
    launches = dmrgk.launch_count()
    clk = clocks.stop()
    n_sm = dp.ctx.query()[0]
    peak = n_sm * 128 * (clk.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
    val = h.flops_alg / ms / 1e9
    print(json.dumps({
        "metric": "per_pair_expectation_fp64_tflops", "value": val, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": max(args.warmup, 2), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "K_pairs": K, "pairs_per_second": K / ms * 1e3, "tasks": h.n_tasks,
                   "flops_alg_per_step": h.flops_alg, "chunks": h.n_chunks, "workspace_bytes": int(h.workspace_bytes),
                   "source_hash": dmrgk.source_hash()},
        "gpu_launches": int(launches),
        "roofline": {"bound": "tensor", "kernel": "heff_gemm_dmma_kernel (per-pair work lists)", "achieved": val, "peak": peak,
                     "unit": UNIT, "frac": val / peak, "traffic": None, "peak_source": f"of derived: {n_sm} SMs x 128 FP64 flop/clk x max SM clock"},
        "sum_check": float(out.sum().item()), "clocks": clk}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="4", choices=["1", "2", "3", "3b", "4", "4rs", "5", "5r"])
    ap.add_argument("--m-max", dest="m_max", type=int, default=16)
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--kernel", type=int, default=0, choices=[0, 2, 3, 4, 5],
                    help="GEMM kernel variant (dmrgk_heff_opts.kernel): 0 = product path; 2, 3, 4 = other (stages, CTAs/SM) "
                         "instantiations kept for measurement")
    ap.add_argument("--no-extras", dest="no_extras", action="store_true",
                    help="skip the extra rows (renormalisation, configs 3 and 2) of the default config-4 line")
    ap.add_argument("--shard", default="none", choices=["none", "k"],
                    help="N > 1 only: 'none' = independent replicas (the scope of BASELINE.json), 'k' = split the operator-pair "
                         "list over the ranks and all-reduce sigma (SURVEY §8(f) NEXT-2)")
    ap.add_argument("--op", default="davidson", choices=["davidson", "renorm", "enlarge", "ragged", "su2", "expect"],
                    help="davidson (default, the headline hot path) or renorm (NEXT-1 row, its own metric)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.op == "renorm":
        run_renorm(args)
    elif args.op == "enlarge":
        run_enlarge(args)
    elif args.op == "ragged":
        run_ragged(args)
    elif args.op == "su2":
        run_su2(args)
    elif args.op == "expect":
        run_expect(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
