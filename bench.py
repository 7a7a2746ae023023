#!/usr/bin/env python
"""bench.py — orbital evaluations/s (value + gradient + Laplacian, fp32) of the blip hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload tio2|small|tiny|large]
                    [--mode vgl|value] [--sweep] [--impl reference]

One "step" is one blipgpu_eval over one batch of synthetic positions: every row of SURVEY.md
§8a (cell map, weights, 64-row gather + FMA, grouping, output).  At N = 1 the workload is
BASELINE.json configs[2], the TiO2-sized cell the metric is quoted on (1,536 electrons x 32
walkers = 49,152 positions, 768 real orbitals, 64x64x40 grid, 503 MB table; PAPER.md:108,
120).  N > 1 (torchrun, one rank per GPU): the path shards over walkers with no data-path
collective — every rank holds a replica of the table and its own walkers ("weak" scaling);
timing is barrier + synchronize on both sides and the max over ranks.

Prints ONE JSON line on rank 0 (see DESIGN.md "Measurement" for every key).
`--impl reference` times the CPU fp64 oracle (oracle/) on the host cores instead.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402  (seeded input generators only; no arithmetic of the method)

METRIC = "orbital evals/s (val+grad+lap, fp32)"
UNIT = "evals/s"
PAPER_CONTEXT = ("paper (PAPER.md:120, Table II): GTX 480 fp32, value only, 30.67x over one i7-920 core; "
                 "derived ~5.8e8 real-channel value-only evals/s kernel-only (other hardware: context)")


def measured_peaks():
    """HBM GB/s denominator: MEASURED_PEAKS.json (driver-written), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            p = json.load(fh)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(p.get("sm_max_mhz", 1965.0))
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", 1965.0


def algorithmic_bytes(M, L, mode_vgl):
    """R_gather of SURVEY.md §8d: 64 gathered coefficients (256 B) + 20 B (VGL) or 4 B (V) of
    output per orbital evaluation."""
    return M * L * (256 + (20 if mode_vgl else 4))


def fma_count(M, L, mode_vgl):
    """FMAs the kernels issue per evaluation: 16 columns x (12 for the z contraction + 7 folds) for
    value + gradient + Laplacian, 16 x 5 for value only."""
    return M * L * (304 if mode_vgl else 80)


def max_over_ranks(dist, x, device):
    """Timing rule of the contract: a multi-rank number is the MAX over ranks.  `dist` is
    torch.distributed (None for a single process); works with nccl (GPU) and gloo (CPU tests)."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(positions_per_rank, norb, world, ms_per_step):
    """Weak scaling: every rank evaluates its own walkers on its replica of the table, so the job's
    evaluations per step are world x (positions per rank) x orbitals, over the slowest rank's time."""
    return positions_per_rank * norb * world / (ms_per_step * 1e-3)


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML in a thread)."""

    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap",
               0x8: "hw_slowdown", 0x10: "sync_boost", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz, self.err = [], set(), None, None
        self._stop = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as exc:           # pragma: no cover
            self.nv, self.err = None, repr(exc)
        self.thread = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                try:
                    mask = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    mask = int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self.REASONS.items():
                    if mask & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception as exc:       # pragma: no cover
                self.err = repr(exc)
                return
            time.sleep(0.002)

    def __enter__(self):
        if self.nv:
            self.thread.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self.nv:
            self.thread.join(timeout=2)

    def summary(self):
        out = {"sm_mhz": int(np.median(self.samples)) if self.samples else None,
               "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}
        if self.err:
            out["error"] = self.err
        return out


# ---------------------------------------------------------------------------------------------
# CPU legs (the only places bench.py executes oracle/): cpu_baseline and --impl reference
# ---------------------------------------------------------------------------------------------
def oracle_sample(cfg, coeffs, sample_positions, mode_vgl, repeats=1):
    """Times the oracle as it stands (gcc -O2, OpenMP over positions) on `sample_positions`
    positions x all orbitals of the workload.  Returns (evals/s, seconds, threads)."""
    import oracle
    A = workloads.lattice(cfg)
    pos = workloads.positions(cfg, M=sample_positions)
    mode = oracle.VGL if mode_vgl else oracle.VALUE
    oracle.eval_fast(A, cfg.grid, coeffs, pos[:64], mode=mode)          # load + warm the library
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        oracle.eval_fast(A, cfg.grid, coeffs, pos, mode=mode)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return pos.shape[0] * cfg.norb / best, best, oracle.num_threads()


def cpu_baseline(cfg, coeffs, mode_vgl):
    # bounded sample: ~10-30 s of CPU work.  Calibrate on 256 positions, then size the sample.
    rate, _, threads = oracle_sample(cfg, coeffs, min(256, cfg.M), mode_vgl)
    target_s = 4.0                                                     # wall seconds x threads ~ CPU work
    n = int(min(cfg.M, max(256, rate * target_s / cfg.norb)))
    rate, secs, threads = oracle_sample(cfg, coeffs, n, mode_vgl)
    return {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"first {n} positions x {cfg.norb} orbitals of {cfg.name}, {secs:.2f} s wall on "
                      f"{threads} threads, fp64, gcc -O2 (oracle/blip_oracle.c, untuned)",
            "paper_context": PAPER_CONTEXT}


def run_reference(args):
    """--impl reference: the oracle on the host cores; each step is a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    cfg = workloads.CONFIGS[args.workload]
    mode_vgl = args.mode == "vgl"
    coeffs = workloads.coefficients(cfg.grid, cfg.norb)
    A = workloads.lattice(cfg)
    rate, _, threads = oracle_sample(cfg, coeffs, min(256, cfg.M), mode_vgl)
    budget = 120.0 / max(1, args.steps + args.warmup)                  # whole run within minutes
    n = int(min(cfg.M, max(64, rate * min(budget, 5.0) / cfg.norb)))
    pos = workloads.positions(cfg, M=n)
    mode = oracle.VGL if mode_vgl else oracle.VALUE
    for _ in range(args.warmup):
        oracle.eval_fast(A, cfg.grid, coeffs, pos, mode=mode)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.eval_fast(A, cfg.grid, coeffs, pos, mode=mode)
    dt = time.perf_counter() - t0
    value = args.steps * n * cfg.norb / dt
    sample = f"first {n} positions x {cfg.norb} orbitals of {cfg.name} per step, fp64, {threads} threads"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(cfg, args, n_positions=n),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_config(cfg, args, n_positions=None):
    return {
        "workload": f"{cfg.name}: BASELINE.json configs[{list(workloads.CONFIGS).index(cfg.name)}]",
        "lattice_bohr": [list(r) for r in cfg.lattice], "grid": list(cfg.grid), "orbitals": cfg.norb,
        "positions_per_step": int(cfg.M if n_positions is None else n_positions),
        "electrons": cfg.electrons, "walkers": cfg.walkers, "clustered_20pct": bool(cfg.clustered),
        "mode": "value+grad+lap" if args.mode == "vgl" else "value",
        "table_bytes": cfg.table_bytes, "parallelism": f"walkers x{args.gpus} (table replicated, no collective)",
        "l2": ("no flush: table + outputs streamed per step exceed the 126 MB L2" if not needs_l2_flush(cfg, args)
               else "L2 flushed between timed steps (a 512 MB buffer is overwritten outside the per-step event pairs): "
                    "table + outputs would fit in L2"),
    }


L2_BYTES = 126 * 1024 * 1024


def needs_l2_flush(cfg, args):
    """Working set of one step: the table plus the outputs.  Below ~2x L2 a repeat of the step would
    find its data cached, so the timed loop flushes L2 between steps (timing rules of the task)."""
    out_bytes = cfg.M * cfg.norb * 4 * (5 if args.mode == "vgl" else 1)
    return cfg.table_bytes + out_bytes < 2 * L2_BYTES


# ---------------------------------------------------------------------------------------------
# GPU arm
# ---------------------------------------------------------------------------------------------
def run_gpu(args):
    import torch
    import paper_1204_1121_b200 as blip

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = workloads.CONFIGS[args.workload]
    mode_vgl = args.mode == "vgl"
    mode = blip.VGL if mode_vgl else blip.VALUE
    L, ld = cfg.norb, (cfg.norb + 3) // 4 * 4
    A = workloads.lattice(cfg)
    coeffs = workloads.coefficients(cfg.grid, cfg.norb)
    handle = blip.blipgpu_create(A, cfg.grid, L, coeffs)
    hpos = workloads.positions(cfg, rank=rank)                       # every rank: its own walkers
    M = hpos.shape[0]
    blip.blipgpu_reserve(handle, M)
    stream = torch.cuda.current_stream()
    dpos = torch.from_numpy(hpos).cuda()
    val = torch.empty((M, ld), dtype=torch.float32, device="cuda")
    grad = torch.empty((M, 3, ld), dtype=torch.float32, device="cuda") if mode_vgl else None
    lap = torch.empty((M, ld), dtype=torch.float32, device="cuda") if mode_vgl else None

    def step():
        blip.blipgpu_eval(handle, dpos, M, mode, val, grad, lap, ld, None, stream)

    # ---- device-resident timing: W warm-ups, then exactly K steps between two events --------
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    n0 = blip.blipgpu_launch_count(handle)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    flush = needs_l2_flush(cfg, args)
    with ClockSampler(local_rank) as clocks:
        if not flush:
            e0.record(stream)
            for _ in range(args.steps):
                step()
            e1.record(stream)
            barrier()
            ms_total = e0.elapsed_time(e1)
        else:
            scratch = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device="cuda")
            pairs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                     for _ in range(args.steps)]
            for a, b in pairs:
                scratch.add_(1)                                        # evicts the table and the outputs from L2
                a.record(stream)
                step()
                b.record(stream)
            barrier()
            ms_total = sum(a.elapsed_time(b) for a, b in pairs)
            del scratch
    launches = blip.blipgpu_launch_count(handle) - n0
    ms_total = max_over_ranks(dist, ms_total, "cuda")
    ms_step = ms_total / args.steps
    evals_step = M * L * world
    value = whole_job_value(M, L, world, ms_step)

    # ---- dominant kernel (gather + FMA) timed by the library's own events on the same stream
    blip.blipgpu_set_profiling(handle, 1)
    kms, gms = [], []
    for _ in range(min(args.steps, 20)):
        step()
        g_, k_ = blip.blipgpu_last_kernel_ms(handle)
        gms.append(g_)
        kms.append(k_)
    blip.blipgpu_set_profiling(handle, 0)
    k_ms, g_ms = float(np.mean(kms)), float(np.mean(gms))
    peak, peak_src, sm_max = measured_peaks()
    abytes = algorithmic_bytes(M, L, mode_vgl)
    achieved = abytes / (k_ms * 1e-3) / 1e9
    fp32_peak = 148 * 128 * 2 * sm_max * 1e6                          # FMA lanes x 2 flop x clock
    fp32_meas = blip.blipgpu_probe_fp32(handle, stream) * 1e12        # packed-FMA rate measured in this run
    # R_compulsory: distinct table rows the batch touches, once, plus the outputs
    cellbuf = torch.empty((M, 3), dtype=torch.int32, device="cuda")
    blip.blipgpu_eval(handle, dpos, M, mode, val, grad, lap, ld, cellbuf, stream)
    torch.cuda.synchronize()
    n = torch.tensor(list(cfg.grid), device="cuda", dtype=torch.int64)
    off = torch.arange(-1, 3, device="cuda", dtype=torch.int64)
    ci = cellbuf.to(torch.int64)
    k0 = (ci[:, 0:1] + off) % n[0]
    k1 = (ci[:, 1:2] + off) % n[1]
    k2 = (ci[:, 2:3] + off) % n[2]
    rows = ((k0[:, :, None, None] * n[1] + k1[:, None, :, None]) * n[2] + k2[:, None, None, :]).reshape(-1)
    distinct_rows = int(torch.unique(rows).numel())
    del rows, k0, k1, k2, ci, cellbuf
    comp_bytes = distinct_rows * L * 4 + M * L * (20 if mode_vgl else 4)
    roofline = {
        "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "traffic": None,
        "kernel": {1: "blip::eval_direct_kernel", 2: "blip::eval_staged_kernel", 3: "blip::eval_split_kernel"}.get(
            blip.blipgpu_last_path(handle), "?") + " (gather + FMA, steps a-2, a-3, a-5)",
        "kernel_ms": k_ms, "grouping_ms": g_ms, "kernel_share_of_step": k_ms / (k_ms + g_ms),
        "algorithmic_bytes": abytes, "bytes_per_eval": abytes / (M * L), "peak_source": peak_src,
        "fp32_fma_frac_of_nominal": 2 * fma_count(M, L, mode_vgl) / (k_ms * 1e-3) / fp32_peak,
        "fp32_peak_tflops_nominal": fp32_peak / 1e12,
        "fp32_peak_tflops_measured": fp32_meas / 1e12,
        "fp32_fma_frac_of_measured": 2 * fma_count(M, L, mode_vgl) / (k_ms * 1e-3) / fp32_meas,
        "distinct_rows": distinct_rows, "compulsory_bytes": comp_bytes,
        "compulsory_hbm_frac": comp_bytes / (k_ms * 1e-3) / 1e9 / peak,
        "note": "contract roofline of BASELINE.json north_star: every gathered coefficient (64 x 4 B) and every "
                "output byte per evaluation at the measured HBM copy rate.  The staged kernel reads each table "
                "row from HBM about 3 times instead of once per electron (see traffic), so achieved exceeds the "
                "HBM peak; what binds it is the shared-memory pipe and the FP32 issue ports (DESIGN.md §6)",
    }
    traffic_file = os.path.join(ROOT, "profiles", "traffic.json")     # written from an ncu --set full capture
    if os.path.exists(traffic_file):
        try:
            with open(traffic_file) as fh:
                tr = json.load(fh)
            key = f"{cfg.name}:{args.mode}"
            if key in tr:
                roofline["traffic"] = tr[key]["dram_bytes_per_launch"]
                roofline["traffic_source"] = tr[key].get("source")
        except Exception:
            pass

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D + eval + D2H per step --
    e2e = None
    if not args.no_e2e:
        ppos = torch.from_numpy(hpos).pin_memory()
        pval = torch.empty((M, ld), dtype=torch.float32).pin_memory()
        pgrad = torch.empty((M, 3, ld), dtype=torch.float32).pin_memory() if mode_vgl else None
        plap = torch.empty((M, ld), dtype=torch.float32).pin_memory() if mode_vgl else None
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        for _ in range(2):
            blip.blipgpu_eval_host(handle, ppos, M, mode, pval, pgrad, plap, ld, None, stream)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            blip.blipgpu_eval_host(handle, ppos, M, mode, pval, pgrad, plap, ld, None, stream)
        barrier()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dist, dt, "cuda")
        e2e = {"value": evals_step * e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": int(ppos.numel() * 8),
               "d2h_bytes_per_step": int(M * ld * 4 * (5 if mode_vgl else 1)), "steps": e2e_steps,
               "ms_per_step": 1e3 * dt / e2e_steps, "api": "blipgpu_eval_host (pinned host buffers)",
               "checksum": float(pval[0, :L].double().sum())}

    line = None
    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_config(cfg, args), "positions_per_s": M * world / (ms_step * 1e-3),
            "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline,
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(cfg, coeffs, mode_vgl)
        if args.sweep:
            line["sweep"] = run_sweep(torch, blip, handle, cfg, dpos, stream)
        if mode_vgl and not args.no_contract:
            line["contract"] = run_contract(torch, blip, handle, cfg, hpos, dpos, stream, args)
            line["f64"] = run_f64(torch, blip, handle, cfg, dpos, stream)
    blip.blipgpu_destroy(handle)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line), flush=True)
    return 0


def run_contract(torch, blip, handle, cfg, hpos, dpos, stream, args):
    """the same evaluations fused with the contraction of the orbital axis
    (blipgpu_eval_contract): no [M][L] outputs.  Device-resident timing, and end to end with the
    positions coming from pinned host memory and the [M][8] result read back every step (the
    vectors d stay on the device, as the inverse Slater matrices would)."""
    M, L = dpos.shape[0], cfg.norb
    ldd = (L + 3) // 4 * 4
    d = torch.zeros((M, ldd), dtype=torch.float32, device="cuda")
    d[:, :L] = torch.from_numpy(workloads.contraction_vectors(M, L)).cuda()
    out = torch.empty((M, 8), dtype=torch.float32, device="cuda")
    steps = max(1, min(args.steps, 50))
    for _ in range(3):
        blip.blipgpu_eval_contract(handle, dpos, M, blip.VGL, d, ldd, out, None, stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(steps):
        blip.blipgpu_eval_contract(handle, dpos, M, blip.VGL, d, ldd, out, None, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    ppos = torch.from_numpy(hpos).pin_memory()
    pout = torch.empty((M, 8), dtype=torch.float32).pin_memory()
    dstage = torch.empty_like(dpos)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        dstage.copy_(ppos, non_blocking=True)
        blip.blipgpu_eval_contract(handle, dstage, M, blip.VGL, d, ldd, out, None, stream)
        pout.copy_(out, non_blocking=True)
        torch.cuda.synchronize()
    dt = (time.perf_counter() - t0) / steps
    return {"api": "blipgpu_eval_contract", "ms_per_step": ms, "evals_per_s": M * L / (ms * 1e-3), "steps": steps,
            "e2e_ms_per_step": 1e3 * dt, "e2e_evals_per_s": M * L / dt, "h2d_bytes_per_step": int(ppos.numel() * 8),
            "d2h_bytes_per_step": int(M * 8 * 4), "checksum": float(pout[:, 0].double().sum()),
            "note": "d [M][L] fp32 resident on the device (151 MB read per step instead of 755 MB written)"}


def run_f64(torch, blip, handle, cfg, dpos, stream):
    """blipgpu_eval_f64 (fp64 weights, accumulation, outputs) on one walker's
    worth of positions — the paper's local-energy call."""
    M, L = min(int(dpos.shape[0]), max(1, cfg.electrons)), cfg.norb
    ld = (L + 3) // 4 * 4
    val = torch.empty((M, ld), dtype=torch.float64, device="cuda")
    grad = torch.empty((M, 3, ld), dtype=torch.float64, device="cuda")
    lap = torch.empty((M, ld), dtype=torch.float64, device="cuda")
    for _ in range(3):
        blip.blipgpu_eval_f64(handle, dpos, M, blip.VGL, val, grad, lap, ld, None, stream)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(20):
        blip.blipgpu_eval_f64(handle, dpos, M, blip.VGL, val, grad, lap, ld, None, stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 20
    return {"api": "blipgpu_eval_f64", "positions": M, "ms_per_call": ms, "evals_per_s": M * L / (ms * 1e-3), "dtype": "f64"}


def run_sweep(torch, blip, handle, cfg, dpos, stream):
    """BASELINE.json configs[3]: throughput vs batch size M on the resident table, both modes."""
    L, ld = cfg.norb, (cfg.norb + 3) // 4 * 4
    out = []
    for mode_name, mode in (("value", blip.VALUE), ("vgl", blip.VGL)):
        for M in workloads.CONFIGS["sweep"].sweep:
            val = torch.empty((M, ld), dtype=torch.float32, device="cuda")
            grad = torch.empty((M, 3, ld), dtype=torch.float32, device="cuda")
            lap = torch.empty((M, ld), dtype=torch.float32, device="cuda")
            reps = 200
            for _ in range(10):
                blip.blipgpu_eval(handle, dpos, M, mode, val, grad, lap, ld, None, stream)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(reps):
                blip.blipgpu_eval(handle, dpos, M, mode, val, grad, lap, ld, None, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            us = 1e3 * e0.elapsed_time(e1) / reps
            # the same calls captured once in a CUDA graph and replayed: device time per call
            # without the host's per-call cost (Python + ctypes + launch)
            gus = None
            if M <= 2048:                                    # these calls only launch kernels
                side = torch.cuda.Stream()
                side.wait_stream(stream)
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=side):
                    for _ in range(20):
                        blip.blipgpu_eval(handle, dpos, M, mode, val, grad, lap, ld, None, side)
                graph.replay()
                torch.cuda.synchronize()
                e0.record(stream)
                for _ in range(10):
                    graph.replay()
                e1.record(stream)
                torch.cuda.synchronize()
                gus = 1e3 * e0.elapsed_time(e1) / 200
            out.append({"M": M, "mode": mode_name, "us_per_call": us, "us_per_call_graph": gus,
                        "evals_per_s": M * L / (us * 1e-6),
                        "evals_per_s_graph": None if gus is None else M * L / (gus * 1e-6),
                        "gathered_GBps": algorithmic_bytes(M, L, mode == blip.VGL) / (us * 1e-6) / 1e9})
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="tio2", choices=["tiny", "small", "tio2", "large"])
    ap.add_argument("--mode", default="vgl", choices=["vgl", "value"])
    ap.add_argument("--sweep", action="store_true", help="also time BASELINE configs[3] (M sweep)")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-contract", action="store_true", help="skip the blipgpu_eval_contract timing")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
