#!/usr/bin/env python
"""bench.py — orbital evaluations/s (value + gradient + Laplacian, fp32) of the blip hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload tio2|small|tiny|large]
                    [--mode vgl|value] [--no-configs] [--impl reference]

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
import hashlib
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
def oracle_sample(cfg, coeffs, sample_positions, mode_vgl, repeats=1, keep=None):
    """Times the oracle as it stands (gcc -O2, OpenMP over positions) on `sample_positions`
    positions x all orbitals of the workload.  Returns (evals/s, seconds, threads); keep (a list)
    receives the oracle's outputs of the last repeat."""
    import oracle
    A = workloads.lattice(cfg)
    pos = workloads.positions(cfg, M=sample_positions)
    mode = oracle.VGL if mode_vgl else oracle.VALUE
    oracle.eval_fast(A, cfg.grid, coeffs, pos[:64], mode=mode)          # load + warm the library
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        out = oracle.eval_fast(A, cfg.grid, coeffs, pos, mode=mode)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    if keep is not None:
        keep[:] = list(out)
    return pos.shape[0] * cfg.norb / best, best, oracle.num_threads()


def cpu_baseline(cfg, coeffs, mode_vgl, gpu_outputs=None):
    """The oracle as it stands on the box's cores: on all of them (OpenMP) and on ONE (the paper compares
    with a single core, Table II), each on a bounded sample.  gpu_outputs
    = (val, grad, lap) torch tensors of the timed call: the all-core sample's results are then compared
    with the same positions of the GPU's — `parity`, the error as a fraction of north_star's tolerances,
    taken outside every timed region."""
    import oracle
    # bounded sample: ~10-30 s of CPU work.  Calibrate on 256 positions, then size the sample.
    rate, _, threads = oracle_sample(cfg, coeffs, min(256, cfg.M), mode_vgl)
    target_s = 4.0                                                     # wall seconds x threads ~ CPU work
    n = int(min(cfg.M, max(256, rate * target_s / cfg.norb)))
    kept = []
    rate, secs, threads = oracle_sample(cfg, coeffs, n, mode_vgl, keep=kept)
    out = {"value": rate, "unit": UNIT, "cores": threads, "kind": "oracle",
           "sample": f"first {n} positions x {cfg.norb} orbitals of {cfg.name}, {secs:.2f} s wall on "
                     f"{threads} threads, fp64, gcc -O2 (oracle/blip_oracle.c, untuned)",
           "paper_context": PAPER_CONTEXT}
    if gpu_outputs is not None and kept:
        A = workloads.lattice(cfg)
        h = float(oracle.spacing(A, cfg.grid).max())
        cmax = float(np.abs(coeffs).max())
        tol = (2e-5 * cmax, 2e-5 * cmax / h, 5e-5 * cmax / (h * h))
        par = {"positions": n, "orbitals": cfg.norb,
               "note": "max |gpu - oracle| over the sample, as a fraction of north_star's tolerance (2e-5 max|c|, 2e-5 max|c| / h, "
                       "5e-5 max|c| / h^2); the GPU outputs are those of the timed call's last step"}
        for name, g, o, t in zip(("val", "grad", "lap"), gpu_outputs, kept[:3], tol):
            if g is None or o is None:
                continue
            err, m0 = 0.0, 0
            while m0 < n:                                              # in slabs: the fp64 difference of the whole batch is GBs
                m1 = min(n, m0 + 4096)
                err = max(err, float(np.abs(g[m0:m1, ..., :cfg.norb].cpu().numpy().astype(np.float64) - o[m0:m1]).max()))
                m0 = m1
            par[name] = err / t
        out["parity"] = par
    del kept
    # one core
    prev = oracle.num_threads()
    oracle.set_num_threads(1)
    try:
        n1 = int(min(cfg.M, max(64, rate / max(threads, 1) * target_s / cfg.norb)))
        rate1, secs1, _ = oracle_sample(cfg, coeffs, n1, mode_vgl)
    finally:
        oracle.set_num_threads(prev)
    out["single_thread"] = {"value": rate1, "unit": UNIT, "cores": 1,
                            "sample": f"first {n1} positions x {cfg.norb} orbitals of {cfg.name}, {secs1:.2f} s wall on 1 thread"}
    return out


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
        "positions_per_step": int((getattr(args, "positions", 0) or cfg.M) if n_positions is None else n_positions),
        "electrons": cfg.electrons, "walkers": cfg.walkers, "clustered_20pct": bool(cfg.clustered),
        "mode": "value+grad+lap" if args.mode == "vgl" else "value",
        "table_bytes": cfg.table_bytes, "parallelism": f"walkers x{args.gpus} (table replicated, no collective)",
        "l2": ("no flush: table + outputs streamed per step exceed the 126 MB L2" if not needs_l2_flush(cfg, args)
               else "L2 flushed between timed steps (a 512 MB buffer is overwritten outside the per-step event pairs): "
                    "table + outputs would fit in L2"),
    }


L2_BYTES = 126 * 1024 * 1024


def needs_l2_flush(cfg, args):
    """Working set of one step: the table rows the batch can touch plus the outputs.  Below ~2x L2 a
    repeat of the step would find its data cached, so the timed loop flushes L2 between steps
    (timing rules of the task)."""
    M = getattr(args, "positions", 0) or cfg.M
    out_bytes = M * cfg.norb * 4 * (5 if args.mode == "vgl" else 1)
    return min(cfg.table_bytes, 64 * M * cfg.norb * 4) + out_bytes < 2 * L2_BYTES


# ---------------------------------------------------------------------------------------------
# GPU arm
# ---------------------------------------------------------------------------------------------
KERNEL_NAMES = {1: "blip::eval_direct_kernel", 2: "blip::eval_staged_kernel", 3: "blip::eval_split_kernel",
                5: "blip::eval_tc_kernel (tcgen05.mma, coefficient planes in tensor memory)"}
# `dtype` of the line = the arithmetic the timed kernel computes in (not a precision claim; `parity_frac` is that)
DTYPE_OF_PATH = {5: "f32 (tcgen05 kind::f16 MMAs on exact two-term fp16 splits of coefficients and weights, per-orbital "
                    "power-of-two scale, fp32 accumulate; fp64 cell map)",
                 1: "f32 (packed FP32 FMAs; fp64 cell map)", 2: "f32 (packed FP32 FMAs; fp64 cell map)",
                 3: "f32 (packed FP32 FMAs; fp64 cell map)"}
FMA_PER_EVAL_CONTRACT = {True: 320, False: 64}      # SURVEY.md §8d R_fp32: five weights per site x 64 sites


def distinct_rows(torch, cells, grid):
    """Number of distinct table rows the batch touches (R_compulsory of SURVEY.md §8d), counted on
    the device from the `cell` output of blipgpu_eval: the 4x4x4 block of sites of every position."""
    n = torch.tensor(list(grid), device="cuda", dtype=torch.int64)
    off = torch.arange(-1, 3, device="cuda", dtype=torch.int64)
    ci = cells.to(torch.int64)
    ci = ci[(ci >= 0).all(dim=1)]
    seen = torch.zeros(int(n[0] * n[1] * n[2]), dtype=torch.bool, device="cuda")
    for lo in range(0, ci.shape[0], 1 << 16):
        c = ci[lo:lo + (1 << 16)]
        k0 = (c[:, 0:1] + off) % n[0]
        k1 = (c[:, 1:2] + off) % n[1]
        k2 = (c[:, 2:3] + off) % n[2]
        rows = ((k0[:, :, None, None] * n[1] + k1[:, None, :, None]) * n[2] + k2[:, None, None, :]).reshape(-1)
        seen[rows] = True
    return int(seen.sum())


def roofline_block(torch, blip, handle, cfg, M, L, mode_vgl, k_ms, g_ms, n_rows, fp32_meas, nsm):
    """The `roofline` object of the JSON line for the dominant (gather + FMA) kernel.

    SURVEY.md §8d gives three figures per evaluation and says which one binds:
      R_gather      64 x 4 B gathered + 20 B (4 B) written, at the HBM copy rate — north_star's contract
                    roofline ("the slower of the gathered coefficient and output bytes at HBM bandwidth
                    and the FMAs at FP32 peak"), with its >= 60 % target;
      R_fp32        320 (64) FMAs at the FP32 peak;
      R_compulsory  distinct rows once + the outputs, at the HBM copy rate.
    A kernel that shares rows between electrons on chip runs faster than R_gather allows; then
    max(R_compulsory, R_fp32) is what binds it and `bound`/`achieved`/`peak`/`frac` describe that
    bound; the contract figure is kept under `contract_frac`."""
    peak_hbm, peak_src, sm_max = measured_peaks()
    evals = M * L
    gather_bytes = algorithmic_bytes(M, L, mode_vgl)
    comp_bytes = n_rows * L * 4 + evals * (20 if mode_vgl else 4)
    flops = 2.0 * FMA_PER_EVAL_CONTRACT[mode_vgl] * evals
    fp32_nominal = nsm * 128 * 2 * sm_max * 1e6                     # FP32 lanes x 2 flop x max SM clock (B200_PROFILING.md)
    t = k_ms * 1e-3
    t_gather = gather_bytes / (peak_hbm * 1e9)
    t_comp = comp_bytes / (peak_hbm * 1e9)
    t_fp32 = flops / fp32_meas
    beats_gather = t < t_gather
    t_hbm = t_comp if beats_gather else t_gather
    if t_fp32 >= t_hbm:
        bound, unit, achieved, peak = "alu", "TFLOP/s", flops / t / 1e12, fp32_meas / 1e12
        peak_source = ("packed-FP32 FMA rate measured in this run (blipgpu_probe_fp32); nominal "
                       f"{nsm} SMs x 128 lanes x 2 x {sm_max:.0f} MHz = {fp32_nominal / 1e12:.2f} TFLOP/s (DESIGN.md §6)")
        per_unit = f"{FMA_PER_EVAL_CONTRACT[mode_vgl]} FMA per evaluation (SURVEY.md §8d R_fp32)"
    else:
        hb = comp_bytes if beats_gather else gather_bytes
        bound, unit, achieved, peak = "hbm", "GB/s", hb / t / 1e9, peak_hbm
        peak_source = peak_src
        per_unit = ("distinct table rows once + outputs (SURVEY.md §8d R_compulsory)" if beats_gather
                    else "256 B gathered + 20 B (4 B) written per evaluation (SURVEY.md §8d R_gather)")
    out = {
        "bound": bound, "achieved": achieved, "peak": peak, "unit": unit, "frac": achieved / peak, "traffic": None,
        "kernel": KERNEL_NAMES.get(blip.blipgpu_last_path(handle), "?") + " (gather + FMA, steps a-2, a-3, a-5)",
        "kernel_ms": k_ms, "grouping_ms": g_ms, "kernel_share_of_step": k_ms / (k_ms + g_ms) if k_ms + g_ms > 0 else None,
        "algorithmic_per_unit": per_unit, "peak_source": peak_source,
        "binding": ("max(R_compulsory, R_fp32): the kernel beats R_gather by sharing rows on chip" if beats_gather
                    else "max(R_gather, R_fp32)"),
        "bound_ms": {"R_gather": 1e3 * t_gather, "R_fp32": 1e3 * t_fp32, "R_compulsory": 1e3 * t_comp},
        "contract_frac": gather_bytes / t / 1e9 / peak_hbm, "contract_target": 0.6,
        "contract_note": "north_star's roofline: R_gather bytes at the measured HBM copy rate; >= 0.6 asked, "
                         "> 1 means rows are served from shared memory / L2 instead of HBM",
        "gather_bytes": gather_bytes, "compulsory_bytes": comp_bytes, "distinct_rows": n_rows,
        "compulsory_hbm_frac": comp_bytes / t / 1e9 / peak_hbm,
        "fp32_frac_issued": 2 * fma_count(M, L, mode_vgl) / t / fp32_meas,
        "fp32_peak_tflops_measured": fp32_meas / 1e12, "fp32_peak_tflops_nominal": fp32_nominal / 1e12,
        "hbm_peak_GBps": peak_hbm,
    }
    if blip.blipgpu_last_path(handle) == 5:
        out["executed_on"] = ("tensor cores: the algorithm's FMAs are issued as 16 tcgen05.mma (M 128, N 16, K 16, fp16 x fp16 "
                              "-> fp32, two-term splits of both operands) per electron and 128 orbitals, not on the FP32 pipe; "
                              "SURVEY.md §8d's binding bound max(R_compulsory, R_fp32) is kept as the yardstick (frac > 1 would "
                              "mean faster than the FP32 pipe could be at its peak)")
    out["kernel_ms_note"] = ("kernel_ms / grouping_ms come from events the library records between the grouping launch and the "
                             "gather + FMA launch (blipgpu_set_profiling); an event there defeats the programmatic dependent launch "
                             "that overlaps the two in the timed steps, so kernel_ms + grouping_ms can exceed ms_per_step")
    out.update(recorded_traffic(f"{cfg.name}:{'vgl' if mode_vgl else 'value'}", comp_bytes))
    # what physically limits the kernel that ran (the §8d figure above is a yardstick once the FMAs run on
    # the tensor cores): compulsory HBM bytes and, from the separate ncu capture, DRAM bytes moved and pipe use
    phys = {"hbm_compulsory_frac": out["compulsory_hbm_frac"]}
    if out.get("traffic"):
        phys["dram_frac"] = out["traffic"] / t / 1e9 / peak_hbm
    pipes = out.pop("ncu_pipes", None)
    if pipes:
        phys.update(pipes)
        phys["pipes_source"] = "separate ncu capture (profiles/traffic.json), not this run"
    out["physical"] = phys
    return out


def kernel_source_digest(files):
    """sha256 over the named source files (repo-relative, in the given order): ties a number taken in a
    separate ncu capture to the kernel sources it was taken from."""
    h = hashlib.sha256()
    for f in files:
        with open(os.path.join(ROOT, f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read() + b"\0")
    return h.hexdigest()


def recorded_traffic(key, comp_bytes):
    """DRAM bytes per launch of the dominant kernel.  NOT measured in this run: it comes from a separate
    `ncu --set full` capture, recorded by hand in profiles/traffic.json together with the sha256 of the
    kernel's source files at the capture (`kernel_sources`, `kernel_sources_sha256`).  It is put on the
    line only while those files are unchanged; after any edit to them the line carries `traffic: null`
    and `traffic_stale` instead, until the capture is redone (`python bench.py --traffic-digests` prints
    the current digests to paste into the file)."""
    out = {"traffic": None}
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            entry = json.load(fh).get(key)
    except Exception:
        entry = None
    if not entry:
        return out
    try:
        now = kernel_source_digest(entry["kernel_sources"])
    except Exception:
        now = None
    if now is not None and now == entry.get("kernel_sources_sha256"):
        out["traffic"] = entry["dram_bytes_per_launch"]
        out["traffic_over_compulsory"] = entry["dram_bytes_per_launch"] / comp_bytes
        out["traffic_source"] = "separate ncu capture, not this run: " + str(entry.get("source"))
        if entry.get("pipes"):
            out["ncu_pipes"] = entry["pipes"]                  # e.g. tensor_pipe_busy, lsu_pipe_busy (fractions of elapsed cycles)
    else:
        out["traffic_stale"] = ("profiles/traffic.json has " + str(entry.get("dram_bytes_per_launch")) + " B per launch for this "
                                "kernel, captured from other sources than the ones loaded now (" + ", ".join(entry.get("kernel_sources", []))
                                + " changed since): not reported")
    return out


class Workload:
    """One config resident on the device: table handle, positions, output buffers."""

    def __init__(self, torch, blip, cfg, mode_vgl, rank=0, M=None):
        self.torch, self.blip, self.cfg, self.mode_vgl = torch, blip, cfg, mode_vgl
        self.mode = blip.VGL if mode_vgl else blip.VALUE
        self.L, self.ld = cfg.norb, (cfg.norb + 3) // 4 * 4
        self.coeffs = workloads.coefficients(cfg.grid, cfg.norb)
        self.handle = blip.blipgpu_create(workloads.lattice(cfg), cfg.grid, self.L, self.coeffs)
        self.hpos = workloads.positions(cfg, rank=rank, M=M)
        self.M = self.hpos.shape[0]
        blip.blipgpu_reserve(self.handle, self.M)
        self.stream = torch.cuda.current_stream()
        self.dpos = torch.from_numpy(self.hpos).cuda()
        self.val = torch.empty((self.M, self.ld), dtype=torch.float32, device="cuda")
        self.grad = torch.empty((self.M, 3, self.ld), dtype=torch.float32, device="cuda")
        self.lap = torch.empty((self.M, self.ld), dtype=torch.float32, device="cuda")

    def step(self, M=None, mode=None, pos=None, stream=None):
        self.blip.blipgpu_eval(self.handle, self.dpos if pos is None else pos, self.M if M is None else M,
                               self.mode if mode is None else mode, self.val, self.grad, self.lap, self.ld, None,
                               self.stream if stream is None else stream)

    def close(self):
        self.blip.blipgpu_destroy(self.handle)
        self.handle = None


def time_steps(torch, w, steps, warmup, flush, barrier=None):
    """W warm-ups, then exactly `steps` steps.  Without flush: one event pair around all steps.  With
    flush (working set would fit in L2): a 512 MB buffer is overwritten before every step and every
    step has its own event pair.  Returns (total milliseconds, kernels launched in the timed region)."""
    sync = barrier or torch.cuda.synchronize
    for _ in range(warmup):
        w.step()
    sync()
    n0 = w.blip.blipgpu_launch_count(w.handle)
    if not flush:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(w.stream)
        for _ in range(steps):
            w.step()
        e1.record(w.stream)
        sync()
        return e0.elapsed_time(e1), w.blip.blipgpu_launch_count(w.handle) - n0
    scratch = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    pairs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in pairs:
        scratch.add_(1)                                        # evicts the table and the outputs from L2
        a.record(w.stream)
        w.step()
        b.record(w.stream)
    sync()
    return sum(a.elapsed_time(b) for a, b in pairs), w.blip.blipgpu_launch_count(w.handle) - n0


def kernel_times(w, reps, flush_buf=None):
    """Device time of the grouping kernels and of the gather + FMA kernel of a step, from the
    library's own events on the launching stream (blipgpu_set_profiling), mean over `reps` steps."""
    blip = w.blip
    blip.blipgpu_set_profiling(w.handle, 1)
    kms, gms = [], []
    for _ in range(reps):
        if flush_buf is not None:
            flush_buf.add_(1)
        w.step()
        g_, k_ = blip.blipgpu_last_kernel_ms(w.handle)
        gms.append(g_)
        kms.append(k_)
    blip.blipgpu_set_profiling(w.handle, 0)
    return float(np.mean(kms)), float(np.mean(gms))


def measure_config(torch, blip, name, steps, fp32_meas, nsm, mode_vgl=True):
    """One of the other BASELINE.json configs for the `configs` block: ms per step, evaluations/s,
    the kernel that ran, and the same roofline object as the headline."""
    cfg = workloads.CONFIGS[name]

    class A:                                                   # needs_l2_flush reads .mode
        mode = "vgl" if mode_vgl else "value"
    flush = needs_l2_flush(cfg, A)
    w = Workload(torch, blip, cfg, mode_vgl)
    try:
        ms = time_steps(torch, w, steps, 3, flush)[0] / steps
        fb = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device="cuda") if flush else None
        k_ms, g_ms = kernel_times(w, min(steps, 10), fb)
        del fb
        cells = torch.empty((w.M, 3), dtype=torch.int32, device="cuda")
        blip.blipgpu_eval(w.handle, w.dpos, w.M, w.mode, w.val, w.grad, w.lap, w.ld, cells, w.stream)
        torch.cuda.synchronize()
        rows = distinct_rows(torch, cells, cfg.grid)
        roof = roofline_block(torch, blip, w.handle, cfg, w.M, w.L, mode_vgl, k_ms, g_ms, rows, fp32_meas, nsm)
        keep = ("bound", "achieved", "peak", "unit", "frac", "kernel", "kernel_ms", "grouping_ms", "binding", "bound_ms",
                "contract_frac", "compulsory_hbm_frac", "distinct_rows", "traffic", "traffic_source", "traffic_stale", "physical")
        return {"workload": f"{cfg.name}: BASELINE.json configs[{list(workloads.CONFIGS).index(cfg.name)}]",
                "positions": w.M, "orbitals": w.L, "grid": list(cfg.grid), "table_bytes": cfg.table_bytes,
                "mode": "value+grad+lap" if mode_vgl else "value", "steps": steps, "ms_per_step": ms,
                "evals_per_s": w.M * w.L / (ms * 1e-3), "positions_per_s": w.M / (ms * 1e-3),
                "last_path": blip.blipgpu_last_path(w.handle),
                "l2": "flushed between steps" if flush else "no flush (working set exceeds L2)",
                "roofline": {k: roof[k] for k in keep if k in roof}}
    finally:
        w.close()
        del w
        torch.cuda.empty_cache()


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
    nsm = torch.cuda.get_device_properties(local_rank).multi_processor_count
    w = Workload(torch, blip, cfg, mode_vgl, rank=rank, M=args.positions or None)   # every rank: a replica and its own walkers
    M, L, ld, handle, stream = w.M, w.L, w.ld, w.handle, w.stream

    # ---- device-resident timing: W warm-ups, then exactly K steps between CUDA events ---------
    flush = needs_l2_flush(cfg, args)
    for _ in range(max(args.warmup, 3)):
        w.step()
    barrier()
    with ClockSampler(local_rank) as clocks:
        ms_total, launches = time_steps(torch, w, args.steps, 0, flush, barrier)
    timed_path = blip.blipgpu_last_path(handle)                       # the gather + FMA kernel the timed steps ran
    ms_total = max_over_ranks(dist, ms_total, "cuda")
    ms_step = ms_total / args.steps
    evals_step = M * L * world
    value = whole_job_value(M, L, world, ms_step)

    # ---- dominant kernel (gather + FMA) timed by the library's own events on the same stream
    # (after half a second of idle: the chip is power-managed within tens of milliseconds — a kernel
    # timed right behind the K steps runs at the sagging clock of their end, not of their average)
    fb = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device="cuda") if flush else None
    time.sleep(0.5)
    k_ms, g_ms = kernel_times(w, min(args.steps, 20), fb)
    del fb
    fp32_meas = blip.blipgpu_probe_fp32(handle, stream) * 1e12        # packed-FMA rate measured in this run
    cellbuf = torch.empty((M, 3), dtype=torch.int32, device="cuda")
    blip.blipgpu_eval(handle, w.dpos, M, w.mode, w.val, w.grad, w.lap, ld, cellbuf, stream)
    torch.cuda.synchronize()
    n_rows = distinct_rows(torch, cellbuf, cfg.grid)
    m_walker = min(M, max(1, cfg.electrons))                           # batch of the f64 / Hessian calls: one walker
    n_rows_walker = distinct_rows(torch, cellbuf[:m_walker].contiguous(), cfg.grid)
    del cellbuf
    roofline = roofline_block(torch, blip, handle, cfg, M, L, mode_vgl, k_ms, g_ms, n_rows, fp32_meas, nsm)

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D + eval + D2H per step --
    e2e = None
    if not args.no_e2e:
        ppos = torch.from_numpy(w.hpos).pin_memory()
        pval = torch.empty((M, ld), dtype=torch.float32).pin_memory()
        pgrad = torch.empty((M, 3, ld), dtype=torch.float32).pin_memory() if mode_vgl else None
        plap = torch.empty((M, ld), dtype=torch.float32).pin_memory() if mode_vgl else None
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        for _ in range(2):
            blip.blipgpu_eval_host(handle, ppos, M, w.mode, pval, pgrad, plap, ld, None, stream)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            blip.blipgpu_eval_host(handle, ppos, M, w.mode, pval, pgrad, plap, ld, None, stream)
        barrier()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dist, dt, "cuda")
        e2e = {"value": evals_step * e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": int(ppos.numel() * 8),
               "d2h_bytes_per_step": int(M * ld * 4 * (5 if mode_vgl else 1)), "steps": e2e_steps,
               "ms_per_step": 1e3 * dt / e2e_steps, "api": "blipgpu_eval_host (pinned host buffers)",
               "checksum": float(pval[0, :L].double().sum())}
        del ppos, pval, pgrad, plap

    line = None
    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": DTYPE_OF_PATH.get(timed_path, "f32"), "data": "synthetic",
            "config": workload_config(cfg, args), "positions_per_s": M * world / (ms_step * 1e-3),
            "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline,
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(cfg, w.coeffs, mode_vgl, (w.val, w.grad, w.lap) if w.M == cfg.M else None)
            if "parity" in line["cpu_baseline"]:
                line["parity_frac"] = line["cpu_baseline"]["parity"]
        if mode_vgl and not args.no_contract:
            line["contract"] = run_contract(torch, blip, handle, cfg, w.hpos, w.dpos, stream, args)
            line["f64"] = run_f64(torch, blip, handle, cfg, w.dpos, stream)
            line["hessian"] = run_hessian(torch, blip, handle, cfg, w.dpos, stream)
            ev, evw = M * L, m_walker * L
            line["contract"]["roofline"] = compact_roofline(line["contract"]["ms_per_step"], M, L, n_rows, 32.0 * M,
                                                            4.0 * M * ld + 24.0 * M, 325, fp32_meas)
            line["f64"]["roofline"] = compact_roofline(line["f64"]["ms_per_call"], m_walker, L, n_rows_walker, 40.0 * evw, 24.0 * m_walker,
                                                       None, fp32_meas, "fp64 FMAs: no measured fp64 peak for this pool, HBM bounds only")
            for name, width in (("f32", 4.0), ("f64", 8.0)):
                if name in line["hessian"]:
                    line["hessian"][name]["roofline"] = compact_roofline(
                        line["hessian"][name]["ms_per_call"], m_walker, L, n_rows_walker, 10.0 * width * evw, 24.0 * m_walker,
                        640 if name == "f32" else None, fp32_meas, "10 quantities per site: 640 FMA per evaluation")
            fp32_staged = None
            if "eval_tc_kernel" in roofline["kernel"]:                    # the FP32-pipe staged kernel on the same batch, same run
                blip.blipgpu_set_tuning(handle, 2, 0)
                time.sleep(0.5)
                k2, g2 = kernel_times(w, 20)
                blip.blipgpu_set_tuning(handle, 0, 0)
                fp32_staged = {"kernel": KERNEL_NAMES[2], "kernel_ms": k2, "tensor_core_kernel_ms": roofline["kernel_ms"],
                               "speedup": k2 / roofline["kernel_ms"]}
            line["tensor_core_recast"] = {
                "shipped": fp32_staged,
                "note": "`shipped` = the tcgen05 kernel that replaced the FP32-pipe staged kernel for this workload, both timed "
                        "here (SURVEY.md §8f NEXT-2).  The mma.sync tf32 form of the recast was measured and rejected in round 2 "
                        "(profiles/r2_v1.md); its probe is the harness program tests/harness/mma_sync_probe.cu, no longer in the library"}
            if L % 2 == 0:
                line["complex"] = run_complex(torch, blip, w, args)
                line["complex"]["roofline"] = compact_roofline(line["complex"]["ms_per_step"], M, L, n_rows, 20.0 * M * L, 24.0 * M + 12.0 * L,
                                                               320, fp32_meas, "phase epilogue (fp64 k.r, sincospi, product rule) not counted")
        if world == 1 and not args.no_configs:
            # the other BASELINE.json configs (north_star item 4): sweep on this table, then small, tiny, large
            block = {}
            if cfg.name == "tio2":
                block["sweep"] = run_sweep(torch, blip, w)
                block["sweep_c_caller"] = run_c_harness()
            w.close()
            w = None
            torch.cuda.empty_cache()
            for name in ("small", "tiny", "large"):
                if name != cfg.name:
                    block[name] = measure_config(torch, blip, name, 20 if name != "large" else 10, fp32_meas, nsm)
            line["configs"] = block
    if w is not None and getattr(w, "handle", None) is not None:
        w.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line), flush=True)
    return 0


def run_c_harness():
    """Per-call latency of blipgpu_eval from a plain-C caller (tests/harness/blip_harness.c): no
    Python, ctypes or torch between the caller and the C ABI."""
    import subprocess
    try:
        sys.path.insert(0, os.path.join(ROOT, "tests", "harness"))
        import build as harness_build
        exe = harness_build.build()
        r = subprocess.run([exe, "latency", "300"], capture_output=True, text=True, timeout=600)
        if r.returncode != 0:
            return {"error": (r.stderr or r.stdout)[-300:]}
        return json.loads(r.stdout.strip().splitlines()[-1])
    except Exception as exc:                                          # the benchmark line must still be printed
        return {"error": repr(exc)}


def compact_roofline(ms, M, L, rows, out_bytes, in_bytes, fma_per_eval, fp32_meas, note=None):
    """The roofline object of the §8(f) entry points, same rules as roofline_block: R_gather
    (256 B per evaluation + the call's own input / output bytes) unless the call beats it by sharing rows
    on chip, then R_compulsory (distinct rows once + the same bytes); against R_fp32 where the arithmetic
    is fp32 (fma_per_eval None: fp64 arithmetic, no measured fp64 peak for this pool — HBM bounds only)."""
    peak_hbm, _, _ = measured_peaks()
    evals, t = M * L, ms * 1e-3
    t_gather = (256.0 * evals + out_bytes + in_bytes) / (peak_hbm * 1e9)
    t_comp = (4.0 * rows * L + out_bytes + in_bytes) / (peak_hbm * 1e9)
    beats = t < t_gather
    cands = {"R_compulsory" if beats else "R_gather": t_comp if beats else t_gather}
    bound_ms = {"R_gather": 1e3 * t_gather, "R_compulsory": 1e3 * t_comp}
    if fma_per_eval:
        cands["R_fp32"] = 2.0 * fma_per_eval * evals / fp32_meas
        bound_ms["R_fp32"] = 1e3 * cands["R_fp32"]
    name = max(cands, key=cands.get)
    out = {"bound": "alu" if name == "R_fp32" else "hbm", "binding": name, "frac": cands[name] / t, "bound_ms": bound_ms,
           "distinct_rows": int(rows), "hbm_peak_GBps": peak_hbm}
    if note:
        out["note"] = note
    return out


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


def run_hessian(torch, blip, handle, cfg, dpos, stream):
    """mode BLIPGPU_VGH (value, gradient, full Cartesian Hessian) on one walker's
    worth of positions — the paper's local-energy call — in fp32 and fp64."""
    M, L = min(int(dpos.shape[0]), max(1, cfg.electrons)), cfg.norb
    ld = (L + 3) // 4 * 4
    out = {"positions": M, "outputs_per_eval": 10}
    for name, tt, fn in (("f32", torch.float32, blip.blipgpu_eval), ("f64", torch.float64, blip.blipgpu_eval_f64)):
        val = torch.empty((M, ld), dtype=tt, device="cuda")
        grad = torch.empty((M, 3, ld), dtype=tt, device="cuda")
        hess = torch.empty((M, 6, ld), dtype=tt, device="cuda")
        for _ in range(3):
            fn(handle, dpos, M, blip.VGH, val, grad, hess, ld, None, stream)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(20):
            fn(handle, dpos, M, blip.VGH, val, grad, hess, ld, None, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 20
        out[name] = {"ms_per_call": ms, "evals_per_s": M * L / (ms * 1e-3)}
    return out


def run_complex(torch, blip, w, args):
    """the same step through blipgpu_eval_complex — L/2 complex orbitals with a
    Bloch phase per orbital (the paper's workload is complex); k-points from
    workloads.kpoints (one random twist per orbital: the worst case, no two orbitals share a phase)."""
    blip.blipgpu_set_kpoints(w.handle, workloads.kpoints(workloads.lattice(w.cfg), w.L // 2))
    steps = max(1, min(args.steps, 50))

    def step():
        blip.blipgpu_eval_complex(w.handle, w.dpos, w.M, blip.VGL, w.val, w.grad, w.lap, w.ld, None, w.stream)

    for _ in range(3):
        step()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(w.stream)
    for _ in range(steps):
        step()
    e1.record(w.stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    blip.blipgpu_set_kpoints(w.handle, None)
    return {"api": "blipgpu_eval_complex", "complex_orbitals": w.L // 2, "ms_per_step": ms, "steps": steps,
            "real_channel_evals_per_s": w.M * w.L / (ms * 1e-3), "complex_evals_per_s": w.M * (w.L // 2) / (ms * 1e-3)}


def run_sweep(torch, blip, w):
    """BASELINE.json configs[3]: throughput against the batch size M on the resident TiO2-sized
    table, both modes.  Device time per call from CUDA-graph replays (no host cost in the number):
      cold  every call of the graph evaluates a different slice of the 49,152-position set, enough
            slices that the table rows they touch exceed twice the L2 (the paper's particle-by-
            particle regime: new positions every call, rows come from HBM);
      warm  the same M positions every call (rows stay in L2) — an upper bound, labelled as such.
    Per call from the host (Python binding, eager) beside them; tests/harness measures it from C."""
    cfg, L, ld, stream = w.cfg, w.L, w.ld, w.stream
    out = []
    pool = w.dpos.shape[0]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for mode_name, mode in (("value", blip.VALUE), ("vgl", blip.VGL)):
        for M in workloads.CONFIGS["sweep"].sweep:
            slots = pool // M
            # touched rows per call ~ 64 M rows of 3 KB (less what positions share); want > 2 x L2 in total
            ncold = int(min(slots, max(16, -(-2 * L2_BYTES // (64 * M * L * 4)) + 1)))
            row = {"M": M, "mode": mode_name, "cold_calls_per_graph": ncold}
            for label, ncalls, slot_of in (("cold", ncold, lambda i: i % slots), ("warm", 20, lambda i: 0)):
                side = torch.cuda.Stream()
                side.wait_stream(stream)
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=side):
                    for i in range(ncalls):
                        w.step(M=M, mode=mode, pos=w.dpos[slot_of(i) * M:], stream=side)
                graph.replay()
                torch.cuda.synchronize()
                reps = max(2, 200 // ncalls)
                e0.record(stream)
                for _ in range(reps):
                    graph.replay()
                e1.record(stream)
                torch.cuda.synchronize()
                us = 1e3 * e0.elapsed_time(e1) / (reps * ncalls)
                row[f"us_per_call_{label}"] = us
                row[f"evals_per_s_{label}"] = M * L / (us * 1e-6)
                del graph
            for i in range(10):
                w.step(M=M, mode=mode, pos=w.dpos[(i % slots) * M:])
            torch.cuda.synchronize()
            e0.record(stream)
            for i in range(200):
                w.step(M=M, mode=mode, pos=w.dpos[(i % slots) * M:])
            e1.record(stream)
            torch.cuda.synchronize()
            row["us_per_call_python_eager"] = 1e3 * e0.elapsed_time(e1) / 200
            row["last_path"] = blip.blipgpu_last_path(w.handle)
            gb = algorithmic_bytes(M, L, mode == blip.VGL)
            row["gathered_GBps_cold"] = gb / (row["us_per_call_cold"] * 1e-6) / 1e9
            row["frac_of_R_gather_cold"] = row["gathered_GBps_cold"] / measured_peaks()[0]
            out.append(row)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="tio2", choices=["tiny", "small", "tio2", "large"])
    ap.add_argument("--mode", default="vgl", choices=["vgl", "value"])
    ap.add_argument("--no-configs", action="store_true",
                    help="skip the `configs` block (batch sweep, small, tiny, large)")
    ap.add_argument("--positions", type=int, default=0,
                    help="evaluate only the first M positions of the workload (a row of the batch sweep, configs[3])")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-contract", action="store_true", help="skip the blipgpu_eval_contract timing")
    ap.add_argument("--traffic-digests", action="store_true",
                    help="print the current sha256 of every profiles/traffic.json entry's kernel sources and exit (no GPU needed)")
    args = ap.parse_args()
    if args.traffic_digests:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            for key, entry in json.load(fh).items():
                now = kernel_source_digest(entry["kernel_sources"])
                print(key, now, "current" if now == entry.get("kernel_sources_sha256") else "STALE")
        return 0
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus != world:
        if "RANK" in os.environ or args.gpus < 1:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE is {world}")
        # run bare with --gpus N > 1: become the torchrun launch the contract describes
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
                                  f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
                                  "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]])
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
