#!/usr/bin/env python
"""bench.py -- chem-step throughput of libgpuann.so on synthetic LES-shaped states.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config c2] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

One "step" = one gpuann_chem_step over the whole batch of the workload (BASELINE.json configs[2] by default:
1,048,576 cells, Ns = 21, MLP 23-1600-800-400-21, BF16 tensor path).  Prints ONE JSON line (rank 0).

  value      cells/s, whole job, state resident in HBM (CUDA events around each step on the launching stream; the
             in-place state is restored from a pristine device copy between steps, outside the event pairs)
  e2e        the same metric through gpuann_chem_step_host with pinned HOST buffers: H2D + step + D2H inside
  roofline   dominant kernel class (per-class CUDA-event times from the library's timing hook, a second pass of
             the same K steps) against MEASURED_PEAKS.json
  cpu_baseline  the FP64 oracle (oracle/, untuned) timed on this box's host cores on a bounded sample

--impl reference times the oracle (this tier has no reference implementation).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "chem-step cells/sec at 1M cells, 21 species; % of B200 BF16 tensor roofline"
UNIT = "cells/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            d = json.loads(p.read_text())
            return {k: float(d[k]) for k in FALLBACK_PEAKS}, "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return dict(FALLBACK_PEAKS), "fallback (B200_PROFILING.md)"


def csrc_sha() -> str:
    """First 16 hex digits of the SHA-256 over the kernel sources (paper_2402_18858_b200/csrc/*.cu, *.cuh and
    include/gpuann.h, in name order, each as name + NUL + bytes): names the kernels an ncu capture was taken from.  The
    sources, not the built library, because -lineinfo puts the build directory into the .so."""
    import hashlib
    h = hashlib.sha256()
    csrc = ROOT / "paper_2402_18858_b200" / "csrc"
    files = sorted(list(csrc.glob("*.cu")) + list(csrc.glob("*.cuh")), key=lambda f: f.name) + [ROOT / "include" / "gpuann.h"]
    for f in files:
        h.update(f.name.encode() + b"\0" + f.read_bytes())
    return h.hexdigest()[:16]


def dram_capture_from_profiles(kernel_class: str, config_index: int, n_cells: int, sha: str = None):
    """The row of profiles/ncu_dram_bytes.csv (ncu --set full: dram__bytes_read.sum, dram__bytes_write.sum per launch) for
    this kernel class, configuration and cell count, as {"bytes", "source", "csrc_sha", "current"}; None if there is
    none.  "current" says whether the capture was taken from the kernel sources of this tree (csrc_sha())."""
    p = ROOT / "profiles" / "ncu_dram_bytes.csv"
    if not p.exists():
        return None
    sha = csrc_sha() if sha is None else sha
    try:
        rows = [l.strip().split(",") for l in p.read_text().splitlines() if l.strip() and not l.startswith("#")]
        hdr = rows[0]
        for r in rows[1:]:
            d = dict(zip(hdr, r))
            if d["kernel_class"] == kernel_class and int(d["config"]) == config_index and int(d["cells"]) == n_cells:
                return {"bytes": float(d["dram_bytes_read"]) + float(d["dram_bytes_write"]), "source": d.get("source"),
                        "csrc_sha": d.get("csrc_sha"), "current": d.get("csrc_sha") == sha}
    except Exception:
        return None
    return None


def dram_bytes_from_profiles(kernel_class: str, config_index: int, n_cells: int, sha: str = None):
    """roofline.traffic: the captured DRAM bytes per launch, or None when there is no capture of exactly this kernel class,
    configuration and cell count TAKEN FROM THE KERNEL SOURCES OF THIS TREE (a capture of older kernels is not reported as
    if it were current)."""
    cap = dram_capture_from_profiles(kernel_class, config_index, n_cells, sha)
    return cap["bytes"] if cap and cap["current"] else None


# ------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and clock-event reasons of one GPU while the timed region runs (pynvml)."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index: int, period_s: float = 0.01):
        self.period = period_s
        self.samples, self.reasons, self.power = [], set(), []
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "power_w_max": max(self.power) if self.power else None}


# ------------------------------------------------------------------ rank aggregation (tested with gloo, world 2)
def aggregate_over_ranks(ms_local: float, cells_local: int, dist=None, device=None):
    """Whole-job figures from per-rank ones: time = MAX over ranks, cells = SUM over ranks (weak scaling)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return ms_local, cells_local
    import torch
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    c = torch.tensor([cells_local], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), int(c.item())


# ------------------------------------------------------------------ oracle legs (cpu_baseline, --impl reference)
def oracle_sample_run(cfg, prob, sample_cells: int, repeats: int = 1):
    """Times oracle.chem_step on the first `sample_cells` cells of the problem.  Returns (cells/s, threads, seconds)."""
    import oracle
    st, th = prob.state, prob.thermo
    s = int(min(sample_cells, st.T.shape[0]))
    T, p, Y = st.T[:s].copy(), st.p[:s].copy(), np.ascontiguousarray(st.Y[:, :s])
    mean, std = oracle.input_moments(T, p, Y, cfg.lam)
    h = oracle.enthalpy_field(T, Y, th.nasa_lo, th.nasa_hi, th.T_mid, th.W).astype(np.float32)
    model = oracle.OracleModel(
        sizes=prob.net.sizes, weights=prob.net.weights, biases=prob.net.biases, in_mean=mean.astype(np.float32),
        in_std=std.astype(np.float32), out_mean=prob.out_mean, out_std=prob.out_std, lam=cfg.lam,
        nasa_lo=th.nasa_lo, W=th.W, nasa_hi=th.nasa_hi, T_mid=th.T_mid, T_min=cfg.T_min, T_max=cfg.T_max,
        newton_tol=cfg.newton_tol, newton_max_iter=cfg.newton_max_iter, T_active=cfg.T_active)
    orc = oracle.Oracle(model)
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        orc.chem_step(T, p, Y, h, cfg.dt)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return s / best, oracle.num_threads(), best, s


def calibrated_sample(cfg, prob, target_s: float):
    """Picks a sample size so that one oracle pass takes about target_s seconds on this box."""
    import oracle
    probe = 64 * oracle.num_threads()
    rate, _, _, _ = oracle_sample_run(cfg, prob, probe)
    s = int(rate * target_s)
    s = max(probe, min(s, prob.state.T.shape[0]))
    return (s // 64) * 64 or probe


def run_reference(args, rank: int, world: int):
    """--impl reference: the oracle as it stands, on the host cores, on a bounded sample per step (rank 0 only)."""
    if rank != 0:
        return
    from paper_2402_18858_b200 import inputs as I
    cfg = I.get_config(args.config)
    n_gen = min(cfg.n_cells, 65536)
    prob = I.make_problem(cfg, n=n_gen)
    sample = calibrated_sample(cfg, prob, target_s=max(1.0, 60.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample_run(cfg, prob, sample)
    t0 = time.perf_counter()
    threads = 1
    for _ in range(args.steps):
        _, threads, _, _ = oracle_sample_run(cfg, prob, sample)
    total = time.perf_counter() - t0
    value = sample * args.steps / total
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg, cfg.n_cells), "sample": f"first {sample} cells per step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": f"first {sample} cells of the workload per step, {args.steps} steps"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_name(cfg, n):
    return (f"configs[{cfg.index}]: {n} cells, Ns={cfg.n_species}, MLP {'-'.join(str(s) for s in cfg.sizes)} GELU, "
            f"{ {0: 'FP32', 1: 'BF16 tcgen05', 2: 'FP16 tcgen05'}[cfg.precision] }, dt={cfg.dt:g}s")


# ------------------------------------------------------------------ our arm
def run_ours(args, rank: int, local_rank: int, world: int):
    import torch
    import torch.distributed as dist
    from paper_2402_18858_b200 import binding as B
    from paper_2402_18858_b200 import inputs as I

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libgpuann has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg = I.get_config(args.config)
    n = int(args.cells) if args.cells else cfg.n_cells
    Ns = cfg.n_species
    prob = I.make_problem(cfg, n=n, seed=cfg.index + 1000 * rank)   # every rank owns its own cells (weak scaling)
    st, th = prob.state, prob.thermo

    prm = B.gpuann_default_params()
    prm.precision = cfg.precision
    prm.newton_max_iter, prm.newton_tol = cfg.newton_max_iter, cfg.newton_tol
    prm.T_min, prm.T_max, prm.T_active = cfg.T_min, cfg.T_max, cfg.T_active
    prm.device = local_rank
    if args.chunk:
        prm.chunk_cells = int(args.chunk)
    ctx = B.gpuann_create(prm)
    stream = torch.cuda.current_stream().cuda_stream

    T0 = torch.from_numpy(st.T).to(dev)
    p_d = torch.from_numpy(st.p).to(dev)
    Y0 = torch.from_numpy(st.Y).to(dev)
    h_d = torch.empty(n, dtype=torch.float32, device=dev)
    # derived inputs (G4, G5) from the library's own helpers -- no CPU implementation on this path
    B.gpuann_load_thermo(ctx, Ns, th.nasa_lo, th.nasa_hi, th.T_mid, th.W)
    B.gpuann_enthalpy(ctx, n, T0.data_ptr(), Y0.data_ptr(), h_d.data_ptr(), stream)
    mean, std = B.gpuann_input_moments(ctx, n, Ns, T0.data_ptr(), p_d.data_ptr(), Y0.data_ptr(), cfg.lam, stream)
    flop_per_cell = float(cfg.flop_per_cell)
    if args.ensemble:   # the paper's per-species architecture: Ns nets D-H1-H2-H3-1
        e_sizes, e_w, e_b = I.gen_ensemble(cfg, seed=cfg.index + 7000)
        B.gpuann_load_net_ensemble(ctx, Ns, e_sizes, e_w, e_b, mean.astype(np.float32), std.astype(np.float32),
                                   prob.out_mean, prob.out_std, cfg.lam)
        flop_per_cell = 2.0 * Ns * sum(e_sizes[i] * e_sizes[i + 1] for i in range(len(e_sizes) - 1))
        del e_w, e_b
    else:
        B.gpuann_load_net(ctx, Ns, prob.net.sizes, prob.net.weights, prob.net.biases, mean.astype(np.float32),
                          std.astype(np.float32), prob.out_mean, prob.out_std, cfg.lam)
    T_d, Y_d = T0.clone(), Y0.clone()

    def restore():
        T_d.copy_(T0)
        Y_d.copy_(Y0)

    ex = {}
    if args.ex:   # gpuann_chem_step_ex with every optional output (RR, HRR, cp, rho, psi): (Ns + 4) more output streams
        ex = {"rr": torch.empty((Ns, n), dtype=torch.float32, device=dev)}
        ex.update({k: torch.empty(n, dtype=torch.float32, device=dev) for k in ("hrr", "cp", "rho", "psi")})

    def step():
        if ex:
            B.gpuann_chem_step_ex(ctx, n, T_d.data_ptr(), p_d.data_ptr(), Y_d.data_ptr(), h_d.data_ptr(), cfg.dt, stream,
                                  **{k: v.data_ptr() for k, v in ex.items()})
        else:
            B.gpuann_chem_step(ctx, n, T_d.data_ptr(), p_d.data_ptr(), Y_d.data_ptr(), h_d.data_ptr(), cfg.dt, stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        restore()
        step()
    barrier()
    # ---- timed region: exactly K steps, CUDA events on the launching stream around each step
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    l0 = B.gpuann_launch_count(ctx)
    with ClockSampler(local_rank, period_s=0.002) as clk:   # the K-step window is ~60 ms: sample it densely enough to see the load
        barrier()
        for e0, e1 in ev:
            restore()
            e0.record()
            step()
            e1.record()
        barrier()
    launches = B.gpuann_launch_count(ctx) - l0
    clocks = clk.summary()
    ms_steps = [e0.elapsed_time(e1) for e0, e1 in ev]
    ms_local = float(sum(ms_steps))
    ms_total, cells_total = aggregate_over_ranks(ms_local, n * args.steps, dist if world > 1 else None, dev)
    value = cells_total / (ms_total * 1e-3)
    n_active, n_notconv, n_degen = B.gpuann_get_stats(ctx)

    # ---- sanity of the result of the last step (device-side reductions; plumbing only)
    sumY = Y_d.double().sum(dim=0)
    ok_finite = bool(torch.isfinite(T_d).all().item() and torch.isfinite(Y_d).all().item())
    active = (T0 >= cfg.T_active) if cfg.T_active > 0 else torch.ones_like(T0, dtype=torch.bool)
    sum_dev = float((sumY[active] - 1.0).abs().max().item())

    # ---- per-kernel-class times (second pass, the library's event hook) -> roofline of the dominant kernel
    B.gpuann_timing_enable(ctx, True)
    for _ in range(args.steps):
        restore()
        step()
    classes = B.gpuann_timing_read(ctx)
    B.gpuann_timing_enable(ctx, False)
    mac_issued, variant = B.gpuann_describe(ctx)
    peaks, peak_src = load_peaks()
    step_ms_sum = sum(v[0] for v in classes.values()) / args.steps
    dom = max(classes.items(), key=lambda kv: kv[1][0])
    dom_name, (dom_ms, dom_cnt) = dom
    sizes = cfg.sizes
    n_act_per_step = n_active / max(1, args.steps + 0) if cfg.T_active > 0 else n
    if cfg.T_active > 0:
        n_act_per_step = int(active.sum().item())
    if dom_name.startswith("layer"):
        l = int(dom_name[5])
        flop_step = 2.0 * sizes[l] * sizes[l + 1] * n_act_per_step
    elif dom_name == "bf16_fused":
        # the fused kernel holds layers 1 and 2 only (algorithmic: the per-pass recompute of layer 1 is not counted)
        flop_step = 2.0 * (sizes[0] * sizes[1] + sizes[1] * sizes[2]) * n_act_per_step * (Ns if args.ensemble else 1)
    else:
        flop_step = flop_per_cell * n_act_per_step
    dom_ms_per_step = dom_ms / args.steps
    achieved = flop_step / (dom_ms_per_step * 1e-3) / 1e12
    # DRAM bytes of the dominant kernel per launch: dram__bytes_read.sum + dram__bytes_write.sum of the committed
    # `ncu --set full` capture of exactly this kernel class, configuration and cell count (profiles/ncu_dram_bytes.csv,
    # written from the .ncu-rep with its command beside it, each row carrying the csrc_sha() of the sources it was
    # taken from); null when no capture matches or the capture is of other sources
    sha_now = csrc_sha()
    capture = dram_capture_from_profiles(dom_name, cfg.index, n, sha_now) if not args.chunk else None
    traffic = capture["bytes"] if capture and capture["current"] else None
    # what each kernel class must move by design (bytes per step): state in / out, h2 out / in, weights once
    h2_bytes = 2.0 * (sizes[2] if len(sizes) > 3 else 0) * n_act_per_step
    by_design = {"state_algorithmic": float(cfg.state_bytes_per_cell) * n_act_per_step,
                 "bf16_fused": (2 + Ns) * 4.0 * n_act_per_step + h2_bytes,
                 "bf16_tail": h2_bytes + ((2 + Ns) + (1 + Ns)) * 4.0 * n_act_per_step}
    roofline = {
        "bound": "tensor", "kernel": dom_name, "achieved": achieved, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
        "frac": achieved / peaks["bf16_tflops"], "traffic": traffic, "traffic_by_design": by_design,
        # where `traffic` comes from: the committed ncu capture and the kernel sources it was taken from; when those are
        # not this tree's sources, traffic is null and traffic_stale carries the old figure for context only
        "traffic_source": capture["source"] if capture else None,
        "traffic_csrc_sha": capture["csrc_sha"] if capture else None, "csrc_sha": sha_now,
        "traffic_stale": capture["bytes"] if capture and not capture["current"] else None,
        "peak_source": peak_src + ", burst",
        "launches_per_step": dom_cnt / args.steps, "ms_per_step_in_kernel": dom_ms_per_step,
        "share_of_step": dom_ms_per_step / step_ms_sum if step_ms_sum > 0 else None,
        "flop_per_step_algorithmic": flop_step,
        "kernel_classes_ms_per_step": {k: v[0] / args.steps for k, v in classes.items()},
    }
    whole_tflops = flop_per_cell * (n_act_per_step * world) / ((ms_total / args.steps) * 1e-3) / 1e12
    roofline["whole_step"] = {
        "achieved": whole_tflops,
        "frac_of_measured_burst": whole_tflops / peaks["bf16_tflops"],
        "frac_of_measured_sustained": whole_tflops / peaks["bf16_tflops_sustained"],
        "frac_of_nominal_2250": whole_tflops / 2250.0,
        "state_gbs": cfg.state_bytes_per_cell * n * world / ((ms_total / args.steps) * 1e-3) / 1e9,
    }
    if cfg.precision == 0:
        roofline["bound"] = "alu"

    # ---- e2e: HOST buffers through gpuann_chem_step_host (H2D + step + D2H inside the timed region)
    k_e2e = max(1, min(args.steps, 10))
    Th = torch.from_numpy(st.T).clone().pin_memory()
    ph = torch.from_numpy(st.p).clone().pin_memory()
    Yh = torch.from_numpy(st.Y).clone().pin_memory()
    hh = h_d.cpu().pin_memory()
    T_host0, Y_host0 = Th.clone(), Yh.clone()

    def step_host():
        B.gpuann_chem_step_host(ctx, n, Th.data_ptr(), ph.data_ptr(), Yh.data_ptr(), hh.data_ptr(), cfg.dt)

    step_host()
    Th.copy_(T_host0)
    Yh.copy_(Y_host0)
    barrier()
    t_e2e = 0.0
    for _ in range(k_e2e):
        t0 = time.perf_counter()
        step_host()                      # synchronous: returns when T, Y are back in host memory
        t_e2e += time.perf_counter() - t0
        Th.copy_(T_host0)
        Yh.copy_(Y_host0)
    barrier()
    t_e2e_ms, cells_e2e = aggregate_over_ranks(t_e2e * 1e3, n * k_e2e, dist if world > 1 else None, dev)
    e2e = {"value": cells_e2e / (t_e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": (3 + Ns) * 4 * n,
           "d2h_bytes_per_step": (1 + Ns) * 4 * n, "steps": k_e2e, "ms_per_step": t_e2e_ms / k_e2e,
           "api": "gpuann_chem_step_host (pinned host buffers)"}

    # ---- sustained leg (--sustain S, default 2 s): the same loop back to back for >= S seconds, clocks and power sampled
    # every 4 ms throughout.  `value` above is a burst of K steps (~0.06 s at the defaults, over before the power cap
    # reacts); a solver that calls the step every time step lives in the steady state reported here.
    sustained = None
    if args.sustain > 0:
        per_batch = 50
        evs = []
        with ClockSampler(local_rank, period_s=0.004) as clk_s:   # >= 100 samples under load in 2 s
            barrier()
            t_start = time.perf_counter()
            while time.perf_counter() - t_start < args.sustain:
                batch = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(per_batch)]
                for e0, e1 in batch:
                    restore()
                    e0.record()
                    step()
                    e1.record()
                torch.cuda.synchronize()
                evs.extend(batch)
            barrier()
        ms_s = np.array([e0.elapsed_time(e1) for e0, e1 in evs])
        tail_half = ms_s[len(ms_s) // 2:]
        ms_sust, _ = aggregate_over_ranks(float(np.median(tail_half)), 0, dist if world > 1 else None, dev)
        tf_s = flop_per_cell * (n_act_per_step * world) / (ms_sust * 1e-3) / 1e12
        sustained = {"seconds": args.sustain, "steps": int(len(ms_s)), "ms_per_step_median_second_half": ms_sust,
                     "ms_per_step_first_20_median": float(np.median(ms_s[:20])), "cells_per_s": n * world / (ms_sust * 1e-3),
                     "tflops": tf_s, "frac_of_measured_burst": tf_s / peaks["bf16_tflops"],
                     "frac_of_measured_sustained": tf_s / peaks["bf16_tflops_sustained"], "clocks": clk_s.summary()}
        roofline["whole_step"]["sustained"] = sustained

    B.gpuann_destroy(ctx)

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not args.ensemble:
        sample = calibrated_sample(cfg, prob, target_s=15.0)
        v, threads, secs, s = oracle_sample_run(cfg, prob, sample)
        import oracle
        oracle.set_num_threads(1)
        v1, _, secs1, s1 = oracle_sample_run(cfg, prob, max(64, sample // (4 * max(1, threads))))
        oracle.set_num_threads(threads)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                        "sample": f"first {s} cells of the workload, one pass, {secs:.1f} s",
                        "value_1_thread": v1, "sample_1_thread": f"first {s1} cells, one pass, {secs1:.1f} s"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": {0: "f32", 1: "bf16", 2: "f16"}[cfg.precision],
            "data": "synthetic",
            "config": {"workload": workload_name(cfg, n) + (f", per-species ensemble of {Ns} nets (PAPER.md:103)" if args.ensemble else ""), "cells_per_gpu": n, "variant": variant + ("+ex(rr,hrr,cp,rho,psi)" if args.ex else ""),
                       "l2": "state (184 B/cell x n) larger than L2 and restored from a pristine copy between steps",
                       "parallelism": f"cells sharded over {world} GPU(s), no collective on the data path"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "cpu_baseline": cpu_baseline,
            "checks": {"finite": ok_finite, "max_abs_sumY_minus_1": sum_dev, "newton_not_converged": int(n_notconv),
                       "degenerate": int(n_degen), "ms_min": min(ms_steps), "ms_median": float(np.median(ms_steps)),
                       "ms_max": max(ms_steps), "ms_steps": [round(x, 4) for x in ms_steps]},
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    if not ok_finite or sum_dev > 1e-6:
        raise SystemExit("bench: result sanity check failed (non-finite values or sum Y != 1)")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c2")
    ap.add_argument("--cells", type=int, default=0, help="override the cell count of the config (per GPU)")
    ap.add_argument("--chunk", type=int, default=0, help="override the library's cells-per-pass")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ensemble", action="store_true",
                    help="the per-species ensemble of the paper (Ns nets with one output each) instead of the single net")
    ap.add_argument("--ex", action="store_true", help="time gpuann_chem_step_ex with every optional output requested")
    ap.add_argument("--sustain", type=float, default=2.0,
                    help="after the K timed steps, run the step back to back for this many seconds and report the "
                         "power-capped steady state as roofline.whole_step.sustained (0 = skip)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if world != args.gpus:
        if world == 1 and args.gpus > 1:
            raise SystemExit("launch N > 1 with: python -m torch.distributed.run --nnodes=1 --nproc-per-node N "
                             "--master-addr 127.0.0.1 --master-port P bench.py --gpus N ...")
    run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
