#!/usr/bin/env python
"""bench.py -- one calibration interval per step on one B200 (replicas on N GPUs).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--coh full|scalar]
                    [--lm compressed|percluster|direct|fullgn] [--impl ours|reference] [--grid | --rows]

A step is one pass of the whole hot path over one synthetic interval:
sagecal_predict_coherencies for all K clusters, then sagecal_sage_calibrate (initial residual, n_em x K M-steps of
n_lm+1 cost/gradient/J^H J evaluations with the device-side LM control; in the default lm_mode the evaluations run on
per-baseline statistics that one streaming kernel per group of four clusters takes together with the write-back of
the previous group, in --lm direct every evaluation streams the cluster's samples).
Workload: BASELINE.json configs[4] (N=512, T=20, F=8, K=50 x 40 sources, 3 EM x 10 LM), the configuration
north_star's target is quoted on; it fits one GPU (67 GB of 2x2 coherencies).  Inputs are seeded and synthetic
(sagecal_inputs, recipe in DESIGN.md §4); the visibilities are built on the device by the CUDA path itself.

Prints ONE JSON line (rank 0).  `value` = seconds per interval with inputs resident in HBM; `e2e` = the same through
sagecal_calibrate_interval_host with pinned HOST buffers (copies inside the timed region); `roofline` = the dominant
streaming kernel of the mode (default: wbgroup_mma_kernel, 40 launches per step; --lm direct: the fused LM pass, 1650
launches) against the measured HBM copy rate, its launch durations taken live with CUDA events on the launching stream
inside the timed region; `cpu_baseline` = the oracle, as it
stands, on a bounded sample of the same workload on the host cores.

--impl reference times the oracle (the only other place bench.py executes oracle/) and prints the same line shape.
Multi-GPU: the path does not shard ("replicas only"): under torchrun every rank calibrates its own
interval, no data-path collective; time = max over ranks.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "calib_wall_time_per_interval"
UNIT = "s"
FALLBACK_HBM_GBS = 6650.0   # B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent
PASS_BYTES_PER_SAMPLE = {"full": 128, "scalar": 80}   # x (64 B) + C (64 B or 16 B): SURVEY.md §8(d), DESIGN.md §6
# compressed mode's streaming kernel (write-back of the previous cluster + statistics for the next):
# read R (64 B) + C_prev + C_next (64 B or 16 B each), write R (64 B)
WBSTAT_BYTES_PER_SAMPLE = {"full": 256, "scalar": 160}
LM_RECENTRE = 10                                       # SAGECAL_LM_RECENTRE of include/sagecal_b200.h
GRP = 4                                                # clusters per group of the streaming kernel (compress.cuh)


def group_sizes(K: int):
    return [min(GRP, K - k0) for k0 in range(0, K, GRP)]


def wbgroup_bytes_per_sample(K: int, n_em: int, coh: str):
    """Algorithmic bytes per sample of every wbgroup launch of one interval (DESIGN.md §5.5 "cluster groups"):
    R read (64 B), R written (64 B) if a previous group is pending, one coherency sample (64 B / 16 B) per cluster of
    the previous and of the next group.  n_em * groups + 1 launches: the first writes nothing back, the last takes
    no statistics."""
    cb = 64 if coh == "full" else 16
    seq = group_sizes(K) * n_em
    out, gp = [], 0
    for gn in seq + [0]:
        out.append(64 + (64 if gp else 0) + cb * (gp + gn))
        gp = gn
    return out


# ---------------------------------------------------------------------------------------------------------------
# helpers without a GPU in them (covered by tests/test_bench_host.py)
# ---------------------------------------------------------------------------------------------------------------
def workload_name(p, coh: str, lm: str = "") -> str:
    return (f"{p.name}: N={p.N} stations, B={p.B} baselines, T={p.T}, F={p.F}, K={p.K} clusters x "
            f"{p.S_tot // max(p.K, 1)} sources, {p.n_em} EM x {p.n_lm} LM, float64, coherencies {coh}"
            + (f", lm {lm}" if lm else ""))


def passes_per_interval(K: int, n_em: int, n_lm: int) -> int:
    """Fused LM evaluation passes in one interval: n_em * K * (n_lm + 1)  (SURVEY.md §8 size table)."""
    return n_em * K * (n_lm + 1)


def uses_groups(lm: str, coh: str, n_lm: int) -> bool:
    """Which streaming kernel sagecal_sage_calibrate runs (calibrate.cu): cluster groups in compressed mode whenever an
    M-step is one chunk; cluster by cluster for lm percluster, fullgn and longer M-steps."""
    return lm == "compressed" and n_lm <= LM_RECENTRE


def expected_launches(K: int, n_em: int, n_lm: int, trace: bool, lm: str = "direct", coh: str = "full") -> int:
    """Kernels one step launches: predict (prep + predict), initial residual, optional ||R||^2 (2), then
    direct:     per (em, k): add-back, write-back, (n_lm+1) x (pass, station reduction, LM control);
    compressed: per (em, k) and per chunk of LM_RECENTRE trial steps one write-back+statistics
                kernel and one cooperative M-step kernel (all evaluations and the LM control), one final write-back."""
    head = 2 + 1 + (2 if trace else 0)
    if lm == "direct":
        return head + n_em * K * (2 + 3 * (n_lm + 1))
    chunks = max(1, -(-n_lm // LM_RECENTRE))
    if uses_groups(lm, coh, n_lm):
        # cluster groups: per group one write-back+statistics kernel per EM iteration (in the first one it also takes
        # the cross grams of the group's coherencies), per cluster one M-step kernel, per cluster but the last of its
        # group one correction kernel; one final write-back
        gs = group_sizes(K)
        return head + n_em * (len(gs) + K + sum(g - 1 for g in gs)) + 1
    if lm == "fullgn":
        # per chunk: statistics kernel, evaluation (3 kernels) + control + commit, then per trial step
        # damping/rhs, step, evaluation (3), control, commit (cuSOLVER's own kernels are not counted)
        return head + n_em * K * (6 * chunks + 7 * n_lm) + 1
    return head + n_em * K * 2 * chunks + 1


def max_over_ranks(ms: float, world_size: int, device=None) -> float:
    """Step time of the job = the slowest rank's (all-reduce MAX over the default process group)."""
    if world_size <= 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def seconds_per_interval(ms_per_step: float, n_gpus: int) -> float:
    """Replicas: every rank finishes one interval per step, so the job finishes n_gpus intervals per step time."""
    return ms_per_step / 1000.0 / max(n_gpus, 1)


def load_peaks() -> tuple[float, str]:
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_traffic(coh: str, kernel: str = "lm_pass"):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the named kernel at the bench workload, from the
    committed ncu --set full summary (profiles/<kernel>_traffic.csv: coh,bytes_read,bytes_write), else None."""
    path = os.path.join(ROOT, "profiles", f"{kernel}_traffic.csv")
    try:
        rows = [l.strip().split(",") for l in open(path) if l.strip() and not l.startswith("#")]
        for r in rows:
            if r[0] == coh:
                return float(r[1]) + float(r[2])
    except Exception:
        pass
    return None


def load_counts(kernel: str, arm: str):
    """FP64 thread-instructions per unit of work of an ALU-bound kernel (predict: per visibility x source; mstep: per
    baseline x evaluation), from ncu's smsp__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on.sum at the bench
    workload divided by the launch's units: profiles/kernel_counts.csv (kernel,arm,unit,fp64_inst_per_unit), else None."""
    path = os.path.join(ROOT, "profiles", "kernel_counts.csv")
    try:
        for l in open(path):
            f = [x.strip() for x in l.split(",")]
            if len(f) >= 4 and not l.startswith("#") and f[0] == kernel and f[1] == arm:
                return float(f[3])
    except Exception:
        pass
    return None


def stream_bytes_per_interval(samples: int, K: int, n_em: int, coh: str, lm: str = "compressed", n_lm: int = 10,
                              fused: bool = False) -> int:
    """Algorithmic HBM bytes of the streaming kernels of one interval: the initial residual reads V and
    all K coherencies and writes R ((2 + K) x 64 B per sample; 16 B per scalar coherency), then the write-back /
    statistics launches (cluster groups: wbgroup_bytes_per_sample; cluster by cluster: 256 / 160 B per sample and
    launch but the first and last; direct: 128 / 80 B per pass plus add-back and write-back)."""
    cb = 64 if coh == "full" else 16
    # fused route (sagecal_predict_residual): the prediction leaves the initial residual, no pass over the coherencies
    init = 0 if fused else (128 + K * cb) * samples
    if K == 0 or n_em == 0:
        return init
    if uses_groups(lm, coh, n_lm):
        return init + sum(wbgroup_bytes_per_sample(K, n_em, coh)) * samples
    if lm == "direct":
        return init + n_em * K * ((n_lm + 1) * PASS_BYTES_PER_SAMPLE[coh] + 2 * (128 + cb)) * samples
    n_launch = n_em * K * max(1, -(-n_lm // LM_RECENTRE)) + 1
    return init + ((n_launch - 2) * WBSTAT_BYTES_PER_SAMPLE[coh] + (64 + cb) + (128 + cb)) * samples


def interval_floor(samples: int, vis_src: int, K: int, n_em: int, coh: str, hbm_gbs: float, dfma_per_s: float,
                   predict_inst_per_vis_src: float, lm: str = "compressed", n_lm: int = 10, fused: bool = False) -> dict:
    """Roofline floor of one interval: the streaming kernels' algorithmic bytes at the measured copy rate plus the
    prediction's arithmetic (station form: 4 FMAs per visibility x source at the measured DMMA rate; fused route: its
    FP64 instructions at the measured DFMA rate) -- or, if larger, the bytes the prediction itself moves
    (K coherencies written; fused route: V read and R written as well) -- the M-step and the small kernels count as
    overhead."""
    b = stream_bytes_per_interval(samples, K, n_em, coh, lm, n_lm, fused)
    hbm_s = b / (hbm_gbs * 1e9)
    alu_s = vis_src * predict_inst_per_vis_src / dfma_per_s if dfma_per_s and predict_inst_per_vis_src else 0.0
    pbytes = (K * (64 if coh == "full" else 16) + (128 if fused else 0)) * samples
    pred_s = max(alu_s, pbytes / (hbm_gbs * 1e9))
    return {"stream_bytes": int(b), "hbm_floor_s": hbm_s, "predict_alu_floor_s": alu_s, "predict_floor_s": pred_s,
            "floor_s": hbm_s + pred_s}


def cpu_model() -> str:
    try:
        for l in open("/proc/cpuinfo"):
            if l.startswith("model name"):
                return l.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu_index = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu_index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line)

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        return parse_clock_lines(self.lines)


def parse_clock_lines(lines) -> dict:
    sm, smax, power, reasons = [], [], [], set()
    names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
    for line in lines:
        f = [x.strip() for x in line.split(",")]
        if len(f) < 9:
            continue
        try:
            sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
        except ValueError:
            continue
        for n, v in zip(names, f[5:9]):
            if v.lower() == "active":
                reasons.add(n)
    if not sm:
        return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
    return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
            "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------------------
# the oracle on a bounded sample of the workload (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------------------------
# The bounded sample keeps ALL time slots (the oracle's per-baseline overheads then weigh as in a full run) and cuts
# clusters and iterations; smaller configs are clipped to their own sizes.  At configs[4] the scaled figure is within
# 10 % of the one full oracle run on record (FULL_RUN below).
SAMPLE = dict(T=10 ** 9, K=2, n_em=1, n_lm=3)
# tests/golden/make_golden_full.py cfg4, the whole configs[4] interval through the oracle on the 16 host cores of the
# GPU box (round 2; the times are in tests/golden/cfg4_oracle.txt): 432 s predict + 317 s SAGE-EM (+ simulate) = 754 s;
# the round-1 run took 752 s
FULL_RUN = {4: {"seconds": 754.0, "cores": 16, "what": "tests/golden/make_golden_full.py cfg4, the whole interval: "
                "432 s predict + 317 s SAGE-EM (host_seconds_* in tests/golden/cfg4_oracle.txt)"}}


def oracle_sample(p, sample=None, cache=None):
    """Runs the oracle, as it stands, on the first T_s time slots and first K_s clusters of problem `p` with
    n_em_s x n_lm_s iterations, and scales the measured time to one full interval: predict by samples*sources,
    calibration by time slots x (corrupt + pass) sweeps.  Returns (seconds_per_interval, description, parts).
    cache (a dict the caller keeps between steps; the reference arm with many steps): only the FIRST cluster's
    prediction is run and timed in every step (it scales exactly, per sample and source); the other sampled clusters'
    coherencies, which the calibration leg needs as input, are predicted once and kept."""
    from oracle import oracle
    from sagecal_inputs import noise_rows
    s = dict(SAMPLE if sample is None else sample)
    Ts, Ks = min(s["T"], p.T), min(s["K"], p.K)
    n_em_s, n_lm_s = min(s["n_em"], p.n_em), min(s["n_lm"], p.n_lm)
    rows = np.arange(Ts * p.B)                           # row r = t*B + b: the first T_s time slots
    Kp = Ks                                              # clusters whose prediction is timed in this call
    if cache is not None and Ks > 1:
        if "coh_rest" not in cache:
            cache["coh_rest"] = oracle.predict(p, rows=rows, clusters=range(1, Ks))
        Kp = 1
    t0 = time.perf_counter()
    coh = oracle.predict(p, rows=rows, clusters=range(Kp))
    t_pred = time.perf_counter() - t0
    if Kp < Ks:
        coh = np.concatenate([coh, cache["coh_rest"]], axis=0)
    vis = np.zeros((rows.size, p.F, 4), np.complex128)   # input preparation, not timed
    for k in range(Ks):
        oracle.corrupt_accumulate(p.N, Ts, p.F, coh[k], p.jones_true[k], +1.0, vis)
    vis += noise_rows(p, rows)
    t0 = time.perf_counter()
    oracle.sage(p.N, Ts, p.F, vis, coh, p.jones_init()[:Ks], n_em_s, n_lm_s, p.tau)
    t_cal = time.perf_counter() - t0
    S = p.S_tot // max(p.K, 1)
    sweeps = lambda K, n_em, n_lm: K + n_em * K * (2 + n_lm + 1)   # initial residual + add-back/write-back + passes
    f_pred = (p.T / Ts) * (p.K / Kp)
    f_cal = (p.T / Ts) * sweeps(p.K, p.n_em, p.n_lm) / sweeps(Ks, n_em_s, n_lm_s)
    total = t_pred * f_pred + t_cal * f_cal
    desc = (f"{'all' if Ts == p.T else 'first ' + str(Ts) + ' of'} {p.T} time slots x first {Ks} of {p.K} clusters ({S} sources each"
            f"{'' if Kp == Ks else '; prediction timed on the first ' + str(Kp)}), predict + "
            f"{n_em_s} EM x {n_lm_s} LM; measured {t_pred:.2f} s predict + {t_cal:.2f} s calibrate, scaled x{f_pred:.0f} "
            f"(samples x sources) and x{f_cal:.1f} (time slots x corrupt/pass sweeps) to one interval")
    return total, desc, dict(predict_s=t_pred, calibrate_s=t_cal, predict_scale=f_pred, calibrate_scale=f_cal)


def run_reference(args):
    """--impl reference: the oracle on the host cores, each step one bounded sample.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    from oracle import oracle
    from sagecal_inputs import make_config
    oracle.build()
    p = make_config(args.config)
    # every step is one bounded sample; with many steps only the first sampled cluster's prediction is repeated per
    # step (about 11 s of host time per step at configs[4]) so that the driver's --steps 20 --warmup 5 run still ends
    # within a few minutes
    cache = {} if args.steps + args.warmup > 6 else None
    for _ in range(args.warmup):
        oracle_sample(p, None, cache)
    vals, desc = [], ""
    t0 = time.perf_counter()
    for _ in range(args.steps):
        v, desc, _ = oracle_sample(p, None, cache)
        vals.append(v)
    wall_ms = (time.perf_counter() - t0) * 1000.0 / max(args.steps, 1)
    value = float(np.mean(vals))
    cores = oracle.num_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": wall_ms, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(p, "full"), "note": "each step is a bounded sample scaled to one interval"},
        "cpu_baseline": dict({"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                              "cpu": cpu_model()},
                             **({"full_run": FULL_RUN[args.config]} if args.config in FULL_RUN else {})),
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------------------------
# the CUDA path
# ---------------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1910_13908_b200 as sg
    from sagecal_inputs import make_config

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    sg.load_library()                                   # raises if libsagecal_b200.so was not built
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if world != args.gpus and rank == 0:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; using WORLD_SIZE", file=sys.stderr)

    # ---- inputs: replicas, every rank its own interval (seed offset by rank) ----
    p = make_config(args.config, seed=191013908 + args.config + 1000 * rank)
    fmt = sg.COH_FULL if args.coh == "full" else sg.COH_SCALAR
    lm_mode = {"compressed": sg.LM_COMPRESSED, "direct": sg.LM_DIRECT, "fullgn": sg.LM_FULLGN, "percluster": sg.LM_PERCLUSTER}[args.lm]
    # the dominant kernel of the step, the one `roofline` describes
    top = "lm_pass" if args.lm == "direct" else "wbstat"
    N, T, F, K = p.N, p.T, p.F, p.K
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    uvw, sl, sm_, sI, sa = t(p.uvw), t(p.src_l), t(p.src_m), t(p.src_I), t(p.src_alpha)
    coh_shape = (K, p.rows, F, 4) if fmt == sg.COH_FULL else (K, p.rows, F)
    coh = torch.empty(coh_shape, dtype=torch.complex128, device=dev)
    predict = lambda: sg.predict_coherencies(N, T, p.freqs, p.f0, uvw, p.cluster_offset, sl, sm_, sI, sa,
                                             coh_format=fmt, out=coh)
    predict()
    noise_host = torch.from_numpy(p.noise()).pin_memory()
    vis = sg.corrupt_subtract(N, T, F, coh, t(p.jones_true), noise_host.to(dev), sign=+1.0, coh_format=fmt)
    jones0 = t(p.jones_init())
    jones = jones0.clone()
    residual = torch.empty_like(vis)
    ws = torch.empty(sg.workspace_bytes(3 if args.lm == "fullgn" else 2, N, T, F, K), dtype=torch.uint8, device=dev)

    def step():
        # --fused: sagecal_predict_residual, the prediction of all K clusters also leaves R = V - sum_k J_k C_k J_k^H (rows
        # 8a-0 .. 8a-2 in one pass) and sagecal_sage_calibrate(vis = NULL) starts from it.  Measured SLOWER than the two
        # separate calls at configs[4] (51.3 ms against 31.5 + 11.7: the residual tile in shared memory leaves 8 warps
        # per SM where the prediction wants 24), so it is not the default.
        jones.copy_(jones0)
        if not args.fused:
            predict()
            return sg.sage_calibrate(N, T, F, vis, coh, jones, p.n_em, p.n_lm, p.tau, coh_format=fmt,
                                     residual=residual, trace=True, workspace=ws, lm_mode=lm_mode)
        sg.predict_residual(N, T, p.freqs, p.f0, uvw, p.cluster_offset, sl, sm_, sI, sa, jones, vis, coh_format=fmt,
                            out=coh, residual=residual)
        return sg.sage_calibrate(N, T, F, None, coh, jones, p.n_em, p.n_lm, p.tau, coh_format=fmt,
                                 residual=residual, trace=True, workspace=ws, lm_mode=lm_mode)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        out = step()
    barrier()

    # ---- timed region: device-resident, the LM pass kernel's launches timed live by the library's event pairs ----
    sg.profile_read()
    timed_kinds = sorted({top, "predict", "corrupt", "mstep"})
    sg.profile_enable(timed_kinds)
    launches0 = sg.launch_count()
    clocks = ClockSampler(local_rank)
    clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        out = step()
    e1.record()
    barrier()
    ms_per_step = max_over_ranks(e0.elapsed_time(e1) / max(args.steps, 1), world, dev)
    clk = clocks.stop()
    gpu_launches = sg.launch_count() - launches0
    prof = sg.profile_read()
    sg.profile_enable([])
    cost_sum = float(out["cost_per_cluster"].sum())
    trace_last = float(out["cost_trace"][-1])

    # ---- one extra untimed step with every kernel kind timed: where the step's device time goes ----
    sg.profile_enable(sg.kernel_kinds())
    step()
    torch.cuda.synchronize()
    breakdown = {k: round(v["ms"], 3) for k, v in sg.profile_read().items()}
    sg.profile_enable([])

    # ---- the mixed-precision predict variant (precision=1, parity 1e-5), reported next to the float64 one ----
    pm0, pm1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    predict_mixed = lambda: sg.predict_coherencies(N, T, p.freqs, p.f0, uvw, p.cluster_offset, sl, sm_, sI, sa,
                                                   coh_format=fmt, precision=1, out=coh)
    predict_mixed()
    pm0.record()
    predict_mixed()
    pm1.record()
    torch.cuda.synchronize()
    breakdown["predict_mixed_precision"] = round(pm0.elapsed_time(pm1), 3)

    npass = prof[top]["timed"]
    pass_ms = prof[top]["ms"] / max(npass, 1)
    if uses_groups(args.lm, args.coh, p.n_lm):
        per = wbgroup_bytes_per_sample(K, p.n_em, args.coh)
        pass_bytes = sum(per) * p.samples // len(per)
    elif args.lm != "direct":
        # per step: n_em*K launches; the first has no write-back (128/80 B per sample), the last no statistics
        # (192/144 B), the others both: algorithmic bytes per launch = the mean over the step's launches
        wb, cb = WBSTAT_BYTES_PER_SAMPLE[args.coh], (64 if args.coh == "full" else 16)
        n_launch = npass // max(args.steps, 1)
        pass_bytes = ((n_launch - 2) * wb + (64 + cb) + (128 + cb)) * p.samples // max(n_launch, 1)
    else:
        pass_bytes = PASS_BYTES_PER_SAMPLE[args.coh] * p.samples
    peak, peak_src = load_peaks()
    achieved = pass_bytes / (pass_ms * 1e-3) / 1e9 if pass_ms > 0 else 0.0
    grouped = uses_groups(args.lm, args.coh, p.n_lm)                         # both are timed as kind "wbstat"
    kname = "wbgroup" if grouped else top
    if grouped:
        kfull = "wbgroup_mma" if args.coh == "full" else "wbgroup_scalar"
    elif top == "lm_pass":
        kfull = "lm_pass_mma" if args.coh == "full" else "lm_pass_scalar"
    else:
        kfull = top
    roofline = {"bound": "hbm", "kernel": kfull + "_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": load_traffic(args.coh, kname),
                "traffic_source": f"stored ncu figure (profiles/{kname}_traffic.csv: dram bytes per launch at configs[4], "
                                  "mean over an interval's launches), not measured in this run",
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": pass_bytes, "launches_timed": npass, "avg_launch_ms": pass_ms,
                "share_of_step": prof[top]["ms"] / max(args.steps, 1) / ms_per_step}

    # ---- every north_star fraction, from this run's own timings (BASELINE.json:5) ----
    # ALU-bound kernels: FP64 thread-instructions (ncu count per unit of work, profiles/kernel_counts.csv) per second
    # of CUDA-event time inside the timed region, against the DFMA-chain peak measured NOW on this device.
    dfma = sg.profile_dfma_peak()
    dmma = sg.profile_dmma_peak()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    dfma_nominal = sms * 64 * (clk.get("sm_max_mhz") or 1965.0) * 1e6
    fused = args.fused
    arm = args.coh + ("_resid" if fused else "")
    rooflines = [dict(roofline)]

    def alu_entry(kernel, kind, units_per_launch, unit_name):
        ipu = load_counts(kernel, arm)
        n = prof[kind]["timed"]
        if not ipu or not n:
            return None
        ms = prof[kind]["ms"] / n
        ach = ipu * units_per_launch / (ms * 1e-3)
        return {"bound": "alu", "kernel": kernel, "achieved": ach / 1e12, "peak": dfma["fma_per_s"] / 1e12,
                "unit": "T FP64 thread-inst/s", "frac": ach / dfma["fma_per_s"], "traffic": None,
                "peak_source": "DFMA-chain kernel measured in this run (sagecal_profile_dfma_peak: 8 chains x 1024 "
                               "threads x %d SMs); nominal %d x 64 lanes x max clock = %.2fe12/s" % (sms, sms, dfma_nominal / 1e12),
                "fp64_inst_per_unit": ipu, "unit_of_work": unit_name, "units_per_launch": units_per_launch,
                "inst_source": "ncu smsp__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on.sum at configs[4] / units "
                               "(profiles/kernel_counts.csv)",
                "launches_timed": n, "avg_launch_ms": ms, "sm_mhz_under_load": clk.get("sm_mhz"),
                "share_of_step": prof[kind]["ms"] / max(args.steps, 1) / ms_per_step}

    if fused:
        e = alu_entry("predict_kernel", "predict", p.vis_src, "visibility x source")
        if e:
            e["note"] = ("RESID arm (sagecal_predict_residual): predicts all K clusters of its rows and leaves the initial "
                         "residual R = V - sum_k J_k C_k J_k^H, so no corrupt_kernel launch is in the step")
            rooflines.append(e)
    elif prof["predict"]["timed"]:
        # station form: a rank-S_k Hermitian update per (time slot, cluster, channel) on the FP64 tensor
        # cores: 4 real FMAs per visibility x source (one complex multiply-add), against the DMMA-chain peak measured
        # NOW on this device; the call also writes the K coherencies once (its HBM bound)
        n = prof["predict"]["timed"]
        ms = prof["predict"]["ms"] / n
        fma = 4.0 * p.vis_src
        cbytes = K * (64 if args.coh == "full" else 16) * p.samples
        rooflines.append({"bound": "tensor", "kernel": "predict_station_kernel", "achieved": fma / (ms * 1e-3) / 1e12,
                          "peak": dmma["fma_per_s"] / 1e12, "unit": "T FP64 FMA/s", "frac": fma / (ms * 1e-3) / dmma["fma_per_s"],
                          "traffic": None,
                          "peak_source": "DMMA-chain kernel measured in this run (sagecal_profile_dmma_peak: 8 chains x 16 "
                                         "warps x %d SMs, 256 FMAs per m8n8k4); DFMA chains in the same run: %.3e/s"
                                         % (sms, dfma["fma_per_s"]),
                          "fma_per_unit": 4.0, "unit_of_work": "visibility x source", "units_per_launch": p.vis_src,
                          "hbm_write_bytes": cbytes, "hbm_write_frac": cbytes / (ms * 1e-3) / 1e9 / peak,
                          "launches_timed": n, "avg_launch_ms": ms, "sm_mhz_under_load": clk.get("sm_mhz"),
                          "share_of_step": prof["predict"]["ms"] / max(args.steps, 1) / ms_per_step,
                          "note": "one sagecal_predict_coherencies call = uvw check + station phasors + contraction "
                                  "(+ the per-baseline kernel, which returns at once); the per-baseline form "
                                  "(sagecal_predict_set_form(1)) runs 8.77 FP64 instructions per visibility x source"})
    if args.lm != "direct":
        chunks = max(1, -(-p.n_lm // LM_RECENTRE))
        evals = (p.n_lm + chunks) / chunks                      # evaluations per launch: the chunk's trials + its centre
        arm = args.coh
        e = alu_entry("mstep_kernel", "mstep", p.B * evals, "baseline x evaluation")
        if e:
            e["note"] = ("latency-bound cooperative kernel: two grid barriers and a station reduction per evaluation "
                         "(DESIGN.md §5.5); the fraction is the baseline arithmetic alone against the FP64 issue peak")
            rooflines.append(e)
    cor = prof["corrupt"]
    if cor["timed"] != args.steps:                        # none (fused route) or one per add-back / write-back (direct)
        # fused route: the step has no residual pass of its own; BASELINE.json:5 item (c)'s kernel is timed on its own
        # here (sagecal_corrupt_subtract over all K clusters), after the timed region
        sg.profile_read()
        sg.profile_enable(["corrupt"])
        for _ in range(4):
            sg.corrupt_subtract(N, T, F, coh, jones, vis, sign=-1.0, coh_format=fmt, out=residual)
        torch.cuda.synchronize()
        cor = sg.profile_read()["corrupt"]
        sg.profile_enable([])
    if cor["timed"]:
        # residual pass: V read, K coherencies read, R written
        cb = 64 if args.coh == "full" else 16
        cbytes = (128 + K * cb) * p.samples
        cms = cor["ms"] / cor["timed"]
        rooflines.append({"bound": "hbm", "kernel": "corrupt_kernel", "achieved": cbytes / (cms * 1e-3) / 1e9, "peak": peak,
                          "unit": "GB/s", "frac": cbytes / (cms * 1e-3) / 1e9 / peak, "traffic": None, "peak_source": peak_src,
                          "algorithmic_bytes_per_launch": cbytes, "launches_timed": cor["timed"], "avg_launch_ms": cms,
                          "where": "inside the timed region" if prof["corrupt"]["timed"] == args.steps else
                                   "sagecal_corrupt_subtract over all K clusters after the timed region (the step's own "
                                   "initial residual is fused into the prediction)"})
    # the fused cost / gradient / J^H J pass as BASELINE.json:5 states it (the kernel of --lm direct): 20 launches of
    # sagecal_lm_cost_grad_jtj on the step's residual and the first cluster's coherencies, after the timed region
    if args.lm != "direct":
        sg.profile_read()
        sg.profile_enable(["lm_pass"])
        for _ in range(21):
            sg.lm_cost_grad_jtj(N, T, F, residual, coh[0], jones[0], coh_format=fmt)
        torch.cuda.synchronize()
        pr = sg.profile_read()["lm_pass"]
        sg.profile_enable([])
        if pr["timed"]:
            pms = pr["ms"] / pr["timed"]
            pbytes = PASS_BYTES_PER_SAMPLE[args.coh] * p.samples
            rooflines.append({"bound": "hbm", "kernel": ("lm_pass_mma" if args.coh == "full" else "lm_pass_scalar") + "_kernel",
                              "achieved": pbytes / (pms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                              "frac": pbytes / (pms * 1e-3) / 1e9 / peak, "traffic": load_traffic(args.coh, "lm_pass"),
                              "traffic_source": "stored ncu figure (profiles/lm_pass_traffic.csv)", "peak_source": peak_src,
                              "algorithmic_bytes_per_launch": pbytes, "launches_timed": pr["timed"], "avg_launch_ms": pms,
                              "where": "loop of sagecal_lm_cost_grad_jtj after the timed region (not part of the default step)"})
    pred_arm = args.coh + ("_resid" if fused else "")
    if fused:
        floor = interval_floor(p.samples, p.vis_src, K, p.n_em, args.coh, peak, dfma["fma_per_s"],
                               load_counts("predict_kernel", pred_arm) or 0.0, args.lm, p.n_lm, fused)
    else:                                                 # station form: 4 FMAs per visibility x source at the DMMA rate
        floor = interval_floor(p.samples, p.vis_src, K, p.n_em, args.coh, peak, dmma["fma_per_s"], 4.0, args.lm, p.n_lm, fused)
    floor["frac_of_floor"] = floor["floor_s"] / (ms_per_step * 1e-3)
    extras = {"rooflines": rooflines, "dfma_peak": dict(dfma, nominal_fma_per_s=dfma_nominal, sms=sms),
              "dmma_peak": dmma, "interval_floor": floor}

    # ---- end to end: HOST buffers in, HOST buffers out, through sagecal_calibrate_interval_host ----
    if args.no_e2e:
        e2e, e2e_cost_sum = None, None
        return _finish(args, p, world, rank, ms_per_step, clk, e2e, e2e_cost_sum, gpu_launches, roofline, breakdown,
                       pass_bytes, cost_sum, trace_last, extras)
    vis_host = torch.empty(vis.shape, dtype=vis.dtype).pin_memory()
    vis_host.copy_(vis)
    del coh, vis, residual, ws, out, noise_host
    torch.cuda.empty_cache()
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_uvw, h_l, h_m, h_I, h_a = pin(p.uvw), pin(p.src_l), pin(p.src_m), pin(p.src_I), pin(p.src_alpha)
    h_j0 = pin(p.jones_init())
    h_j = torch.empty_like(h_j0).pin_memory()
    h_res = torch.empty(vis_host.shape, dtype=vis_host.dtype).pin_memory()
    h_cpc = torch.zeros(K, dtype=torch.float64).pin_memory()
    h_js = [h_j] + [torch.empty_like(h_j0).pin_memory() for _ in range(2)]
    h_cpcs = [h_cpc] + [torch.zeros(K, dtype=torch.float64).pin_memory() for _ in range(2)]
    nbytes = lambda *ts: int(sum(x.numel() * x.element_size() for x in ts))
    h2d = nbytes(h_uvw, h_l, h_m, h_I, h_a, vis_host, h_j)
    d2h = nbytes(h_j, h_res, h_cpc)

    def e2e_step(asynchronous=False, k=0):
        hj, hc = h_js[k], h_cpcs[k]
        hj.copy_(h_j0)
        sg.calibrate_interval_host(N, T, p.freqs, p.f0, h_uvw, p.cluster_offset, h_l, h_m, h_I, h_a, vis_host, hj,
                                   p.n_em, p.n_lm, p.tau, coh_format=fmt, residual=h_res, cost_per_cluster=hc,
                                   lm_mode=lm_mode, asynchronous=asynchronous)

    # (1) one synchronous call per step: the latency of an interval from and to host buffers
    for _ in range(args.warmup):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()                                      # synchronises its streams before returning
    torch.cuda.synchronize()
    single_ms = max_over_ranks((time.perf_counter() - t0) * 1000.0 / max(args.steps, 1), world, dev)
    e2e_cost_sum = float(h_cpc.sum())
    # (2) a STREAM of intervals through the asynchronous entry (two in flight): the residual's device-to-host copy of
    # one interval overlaps the prediction of the next.  Every step still copies its inputs in and its results out
    # inside the timed region.  The Jones buffer is in/out, and a call only guarantees that the interval THREE back is
    # home when it is made: three sets of the small in/out arrays rotate.
    stream_ms, stream_note = None, None
    try:
        for i in range(max(args.warmup, 2)):
            e2e_step(True, i % 3)
        sg.host_sync()
        barrier()
        t0 = time.perf_counter()
        for i in range(args.steps):
            e2e_step(True, i % 3)
        sg.host_sync()
        stream_ms = max_over_ranks((time.perf_counter() - t0) * 1000.0 / max(args.steps, 1), world, dev)
        last = h_cpcs[(args.steps - 1) % 3]
        if abs(float(last.sum()) - e2e_cost_sum) > 1e-12 * abs(e2e_cost_sum):
            stream_note = "stream leg rejected: sum of costs %r differs from the synchronous call's %r" % (float(last.sum()), e2e_cost_sum)
            stream_ms = None                             # must be the very same answer
    except Exception as ex:
        stream_ms, stream_note = None, "stream leg failed: " + repr(ex)
    sg.host_trim()                                       # the library's cached arenas go back before the grid allocates
    e2e_ms = stream_ms if stream_ms is not None else single_ms
    e2e = {"value": seconds_per_interval(e2e_ms, world), "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms,
           "single_call_s": single_ms / 1000.0, "stream_s_per_interval": None if stream_ms is None else stream_ms / 1000.0,
           "stream_note": stream_note,
           "api": ("sagecal_calibrate_interval_host_async, a stream of intervals with two in flight, sagecal_host_sync at "
                   "the end (pinned host buffers in and out, copies of every step inside the timed region); "
                   "single_call_s = one synchronous sagecal_calibrate_interval_host per step"
                   if stream_ms is not None else "sagecal_calibrate_interval_host (pinned host buffers in and out)")}

    # ---- the paper's stations x clusters grid, every point but the headline's own, with its floor ----
    if world == 1 and not args.no_grid:
        del vis_host, h_res
        torch.cuda.empty_cache()
        try:
            extras["grid"] = measure_grid(sg, dev, args, peak, extras["dfma_peak" if args.fused else "dmma_peak"]["fma_per_s"],
                                          skip=[(p.N, p.K)] if args.config == 4 else [], steps=2, warmup=1)
        except Exception as ex:                          # the bench line must not depend on the grid
            extras["grid"] = {"error": repr(ex)}

    return _finish(args, p, world, rank, ms_per_step, clk, e2e, e2e_cost_sum, gpu_launches, roofline, breakdown,
                   pass_bytes, cost_sum, trace_last, extras)


def _finish(args, p, world, rank, ms_per_step, clk, e2e, e2e_cost_sum, gpu_launches, roofline, breakdown, pass_bytes,
            cost_sum, trace_last, extras=None):
    import torch.distributed as dist
    from sagecal_inputs import make_config
    K = p.K
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- the oracle on the host cores, bounded sample (rank 0, N=1 only) ----
    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import oracle
        oracle.build()
        v, desc, _ = oracle_sample(make_config(args.config))
        cpu_baseline = {"value": v, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": desc,
                        "cpu": cpu_model()}
        if args.config in FULL_RUN:
            cpu_baseline["full_run"] = FULL_RUN[args.config]

    predict_ms = breakdown.get("predict", 0.0) + breakdown.get("predict_prep", 0.0)
    line = {
        "metric": METRIC, "value": seconds_per_interval(ms_per_step, world), "unit": UNIT, "n_gpus": world,
        # replicas: every rank calibrates its own interval, so `value` (job seconds per interval) is the per-replica
        # time / n_gpus by construction; the per-replica wall time is what a kernel change moves
        "per_replica_s": ms_per_step / 1000.0, "intervals_per_s": max(world, 1) / (ms_per_step / 1000.0),
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": False,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(p, args.coh, args.lm), "parallelism": "replicas only (one interval per GPU)",
                   "l2": "inputs larger than L2 (per-pass working set %.2f GB vs 126 MB)" % (pass_bytes / 1e9),
                   "seed": p.seed},
        "clocks": clk, "e2e": e2e, "gpu_launches": int(gpu_launches),
        "gpu_launches_expected": args.steps * (expected_launches(K, p.n_em, p.n_lm, True, args.lm, args.coh)
                                               - (1 if args.fused else 0)),
        "roofline": roofline, "cpu_baseline": cpu_baseline,
        "breakdown_ms_one_step": breakdown,
        "predict_gvis_src_per_s": p.vis_src / (predict_ms * 1e-3) / 1e9 if predict_ms > 0 else None,
        "predict_mixed_gvis_src_per_s": (p.vis_src / (breakdown["predict_mixed_precision"] * 1e-3) / 1e9
                                         if breakdown.get("predict_mixed_precision") else None),
        "check": {"sum_cost_per_cluster": cost_sum, "cost_trace_last": trace_last, "e2e_sum_cost_per_cluster": e2e_cost_sum},
    }
    line.update(extras or {})
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


GRID_N, GRID_K = (64, 128, 256, 384, 512), (1, 50)


def measure_grid(sg, dev, args, hbm_gbs, dfma_per_s, skip=(), steps=None, warmup=None):
    """The paper's scaling experiment (runtime over stations x clusters, Figs. 1-3) with this
    build's own timings -- configs[4]'s recipe (T=20, F=8, 40 sources per cluster, 3 EM x 10 LM) at N in GRID_N x K in
    GRID_K.  Every point carries its roofline floor (interval_floor: the streaming kernels' algorithmic bytes at the
    measured copy rate + the prediction's FP64 instructions at the measured DFMA rate) and floor / measured."""
    import torch
    from sagecal_inputs import make_config
    fmt = sg.COH_FULL if args.coh == "full" else sg.COH_SCALAR
    lm_mode = {"compressed": sg.LM_COMPRESSED, "direct": sg.LM_DIRECT, "fullgn": sg.LM_FULLGN, "percluster": sg.LM_PERCLUSTER}[args.lm]
    steps = args.steps if steps is None else steps
    warmup = max(args.warmup, 1) if warmup is None else warmup
    fused = args.fused
    # prediction's floor: fused route FP64 instructions (ncu count) at the DFMA rate; else 4 FMAs at the DMMA rate
    ipu = (load_counts("predict_kernel", args.coh + "_resid") or 0.0) if fused else 4.0
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    out = []
    for N in GRID_N:
        for K in GRID_K:
            if (N, K) in skip:
                continue
            p = make_config(4, N=N, K=K)
            uvw, sl, sm_, sI, sa = t(p.uvw), t(p.src_l), t(p.src_m), t(p.src_I), t(p.src_alpha)
            shape = (K, p.rows, p.F, 4) if fmt == sg.COH_FULL else (K, p.rows, p.F)
            coh = torch.empty(shape, dtype=torch.complex128, device=dev)
            predict = lambda: sg.predict_coherencies(N, p.T, p.freqs, p.f0, uvw, p.cluster_offset, sl, sm_, sI, sa,
                                                     coh_format=fmt, out=coh)
            predict()
            vis = sg.corrupt_subtract(N, p.T, p.F, coh, t(p.jones_true), t(p.noise()), sign=+1.0, coh_format=fmt)
            jones0 = t(p.jones_init())
            jones = jones0.clone()
            residual = torch.empty_like(vis)
            ws = torch.empty(sg.workspace_bytes(3 if args.lm == "fullgn" else 2, N, p.T, p.F, K), dtype=torch.uint8, device=dev)

            def step():
                jones.copy_(jones0)
                if not fused:
                    predict()
                    return sg.sage_calibrate(N, p.T, p.F, vis, coh, jones, p.n_em, p.n_lm, p.tau, coh_format=fmt,
                                             residual=residual, trace=True, workspace=ws, lm_mode=lm_mode)
                sg.predict_residual(N, p.T, p.freqs, p.f0, uvw, p.cluster_offset, sl, sm_, sI, sa, jones, vis,
                                    coh_format=fmt, out=coh, residual=residual)
                return sg.sage_calibrate(N, p.T, p.F, None, coh, jones, p.n_em, p.n_lm, p.tau, coh_format=fmt,
                                         residual=residual, trace=True, workspace=ws, lm_mode=lm_mode)
            for _ in range(warmup):
                o = step()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(steps):
                o = step()
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / max(steps, 1)
            tr = o["cost_trace"].cpu().numpy()
            fl = interval_floor(p.samples, p.vis_src, K, p.n_em, args.coh, hbm_gbs, dfma_per_s, ipu, args.lm, p.n_lm, fused)
            out.append({"N": N, "B": p.B, "K": K, "samples": p.samples, "s_per_interval": ms / 1e3,
                        "hbm_floor_s": fl["hbm_floor_s"], "predict_floor_s": fl["predict_floor_s"],
                        "frac_of_floor": fl["floor_s"] / (ms / 1e3),
                        "cost_first": float(tr[0]), "cost_last": float(tr[-1]),
                        "monotone": bool(np.all(np.diff(tr) <= 1e-12 * tr[:-1]))})
            del coh, vis, residual, ws, o, jones, jones0
            torch.cuda.empty_cache()
    return out


def run_grid(args):
    """--grid: measure_grid at every point.  Prints one JSON object {"grid": [...]}; not the bench line."""
    import torch
    import paper_1910_13908_b200 as sg
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --grid: no CUDA device")
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    peak, peak_src = load_peaks()
    dfma = sg.profile_dfma_peak() if args.fused else sg.profile_dmma_peak()
    out = measure_grid(sg, dev, args, peak, dfma["fma_per_s"])
    print(json.dumps({"grid": out, "recipe": "configs[4] layout/T/F/S, 3 EM x 10 LM, float64, coherencies " + args.coh +
                      ", lm " + args.lm, "steps": args.steps, "warmup": max(args.warmup, 1),
                      "floor": "streaming kernels' algorithmic bytes at %.1f GB/s (%s) + predict's FP64 instructions at "
                               "%.3e FMA/s (DMMA chains; --fused: FP64 instructions at the DFMA-chain rate; measured in this run)" % (peak, peak_src, dfma["fma_per_s"])}), flush=True)
    return 0


def run_rows(args):
    """--rows: the measurement-set front end at the bench workload's size (second part):
    a seeded row list (5 % of the rows absent, 30 % given as (q, p), 5 % of the samples flagged, random order) is
    brought into canonical order, the flags are applied to all K clusters' coherencies, and the residual is handed
    back in row order.  Prints one JSON object {"rows": {...}}; not the bench line."""
    import torch
    import paper_1910_13908_b200 as sg
    from sagecal_inputs import make_config, make_rowlist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --rows: no CUDA device")
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    fmt = sg.COH_FULL if args.coh == "full" else sg.COH_SCALAR
    p = make_config(args.config)
    rl = make_rowlist(p, seed=p.seed + 1000, drop_frac=0.05, swap_frac=0.3, flag_frac=0.05)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    a1, a2, ts, uvw_in, fl_in, vis_in = t(rl.ant1), t(rl.ant2), t(rl.tslot), t(rl.uvw), t(rl.flags), t(rl.noise)
    n = int(a1.numel())
    shape = (p.K, p.rows, p.F, 4) if fmt == sg.COH_FULL else (p.K, p.rows, p.F)
    coh = torch.ones(shape, dtype=torch.complex128, device=dev)
    back = torch.empty((n, p.F, 4), dtype=torch.complex128, device=dev)
    can = sg.rows_to_canonical(p.N, p.T, p.F, a1, a2, ts, uvw_in, vis_in, fl_in)
    legs = {
        "rows_to_canonical": lambda: sg.rows_to_canonical(p.N, p.T, p.F, a1, a2, ts, uvw_in, vis_in, fl_in),
        "apply_flags": lambda: sg.apply_flags(p.N, p.T, p.F, can["flags"], coh, None, coh_format=fmt),
        "canonical_to_rows": lambda: sg.canonical_to_rows(p.N, p.T, p.F, can["row_map"], can["vis"], back),
    }
    nflag = int(can["flags"].count_nonzero().item())
    cbytes = 64 if fmt == sg.COH_FULL else 16
    # algorithmic bytes: gather = rows read once + canonical arrays written once (+ index arrays, flags);
    # flags = 1 B read per sample + the flagged samples' coherencies written; scatter = 64 B read + written per row sample
    alg = {"rows_to_canonical": n * p.F * 65 + p.samples * 65 + n * 44 + p.rows * 32,
           "apply_flags": p.samples + nflag * p.K * cbytes,
           "canonical_to_rows": n * p.F * 128 + n * 8}
    out = {}
    for name, fn in legs.items():
        for _ in range(max(args.warmup, 1)):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / max(args.steps, 1)
        out[name] = {"ms": ms, "algorithmic_bytes": alg[name], "GBps": alg[name] / ms / 1e6}
    print(json.dumps({"rows": out, "workload": workload_name(p, args.coh), "rows_in": n, "slots": p.rows,
                      "flagged_samples": nflag, "status": can["status"].cpu().tolist(), "steps": args.steps}), flush=True)
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--coh", choices=["full", "scalar"], default="full")
    ap.add_argument("--lm", choices=["compressed", "direct", "fullgn", "percluster"], default="compressed",
                    help="lm_mode of sagecal_sage_calibrate (DESIGN.md §5.5, §5.6); direct = every evaluation streams the "
                         "samples; fullgn = full Gauss-Newton matrix + cuSOLVER Cholesky (a different iteration, NEXT-2)")
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs only)")
    ap.add_argument("--fused", action="store_true",
                    help="prediction fused with the initial residual (sagecal_predict_residual) instead of two calls")
    ap.add_argument("--no-grid", action="store_true", help="skip the stations x clusters grid appended to the bench line")
    ap.add_argument("--grid", action="store_true",
                    help="time the paper's stations x clusters scaling grid instead of the bench step (SURVEY.md §8(f) NEXT-4)")
    ap.add_argument("--rows", action="store_true",
                    help="time the measurement-set front end (rows -> canonical, flags, canonical -> rows) at --config's size")
    args = ap.parse_args(argv)
    if args.rows:
        return run_rows(args)
    if args.grid:
        return run_grid(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
