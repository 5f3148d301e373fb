"""bench.py -- sec/step and FP64 TFLOP/s of the Triad-ATRG hot path at D = 32 on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Workload: BASELINE.json configs[3] -- 4D Ising, beta = 0.1497, h = 0, Triad-ATRG D = 32, p = 32 (K = l = 64), 2 power
iterations, Philox seed 42, 60 coarse-graining steps.  A "step" is one coarse-graining step of the whole hot path
(Fig. 5 a-f).  The run has three regimes: steps 1-5 unsaturated (legs grow 2 -> 32; never timed), steps 6-19 saturated
at criticality (full-rank tensors), steps 20-60 post-critical (the flow has left the critical surface, tensors are
numerically rank-deficient and the QR pre-reduction runs its rank-revealing path).  The cost of a step depends on
the regime, so the line says which steps every number describes:

  value               mean seconds per step over the K timed steps = steps 6+W .. 5+W+K of the run (`config.window`),
                      state resident in HBM; `step_ms` lists them by absolute step index
  value_critical      mean over steps 6-19, value_post_critical over steps 20-60, full_run.seconds over all 60:
                      from ONE separate run of the whole config (the same numbers whatever --steps is)
  e2e                 the `value` window through the C ABI with HOST buffers (state uploaded from pinned memory
                      before, and downloaded after, every step, inside the timed region)
  roofline, permute,  per-launch CUDA events of a separate pass over the SAME window (fresh handle advanced to the same
  stage_ms            step), split by regime
  scaling_vs_D        seconds per saturated step at D = 8 .. 48 (configs[4]: D = 48; plain ATRG D = 24; ILO D = 32)

Replicas only for N > 1: every rank coarse-grains its own network, no collective in the path.
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
import argparse
import gc
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

BETA, H, D, P, N_POW, SEED = 0.1497, 0.0, 32, 32, 2, 42
PRE_STEPS = 5                      # legs grow 2 -> 4 -> 16 -> 32: saturated from step 6 on
FIRST_POST_CRITICAL = 20           # sigma_2 / sigma_1 drops from 0.6 to 0.08 over steps 18-20: rank-deficient tensors from here on
FULL_RUN_STEPS = 60                # configs[3]: 2^15 per axis
METRIC = "sec_per_coarse_graining_step_D32"
UNIT = "s/step"
WORKLOAD = "configs[3]: 4D Ising beta=0.1497 h=0, 2^15 per axis (60 steps), Triad-ATRG D=32 p=32 (K=l=64), 2 power iterations, Philox seed 42"
# model FLOPs of one saturated step in the 2*M*N*K convention: counted live by the library
FP64_TO_BF16_NOMINAL = 45.0 / 2250.0   # guide's nominal B200 FP64-tensor : dense bf16 ratio (blackwell_cuda_programming.md)


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm=p["hbm_gbs"], bf16=p["bf16_tflops"], bf16_sus=p.get("bf16_tflops_sustained", p["bf16_tflops"]), src="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sus=1400.0, src="fallback")


class ClockSampler(threading.Thread):
    """SM clock and throttle reasons during the timed region (B200_PROFILING.md), read through NVML in-process (a query costs
    microseconds; spawning nvidia-smi several times inside a 0.4 s timed region perturbs the host-driven launches).  Falls back to
    nvidia-smi when the NVML binding is missing."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag = index, [], set(), False
        self.active = False       # the thread polls from before the warm-up on (first NVML queries are slow); samples count only while active
        self.max_mhz = None
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            # LOCAL_RANK indexes CUDA_VISIBLE_DEVICES, NVML indexes the physical devices
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and all(x.strip().isdigit() for x in vis.split(",")) else index
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def sample_nvml(self):
        n = self.nvml
        self.samples.append(float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM)))
        if self.max_mhz is None:          # constant: asked once (every NVML query takes a driver lock that a kernel launch may have to wait for)
            self.max_mhz = float(n.nvmlDeviceGetMaxClockInfo(self.handle, n.NVML_CLOCK_SM))
        r = n.nvmlDeviceGetCurrentClocksEventReasons(self.handle) if hasattr(n, "nvmlDeviceGetCurrentClocksEventReasons") \
            else n.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle)
        for name, bit in (("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20), ("sw_power_cap", 0x4)):
            if r & bit:
                self.reasons.add(name)

    def sample_smi(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q, "--format=csv,noheader,nounits"],
                             capture_output=True, text=True, timeout=5).stdout.strip().split(",")
        self.samples.append(float(out[0]))
        self.max_mhz = float(out[1])
        for n, v in zip(names, out[2:]):
            if v.strip().lower().startswith("active"):
                self.reasons.add(n)

    def run(self):
        while not self.stop_flag:
            try:
                n0, r0 = len(self.samples), set(self.reasons)
                if self.nvml:
                    self.sample_nvml()
                elif self.active:
                    self.sample_smi()
                if not self.active:               # outside the timed regions: discard
                    del self.samples[n0:]
                    self.reasons = r0
            except Exception:
                pass
            time.sleep(0.2)               # ~10 samples over a 20-step timed region; denser polling showed up as host stalls between launches

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s), "source": "nvml" if self.nvml else "nvidia-smi"}


# ---- the oracle on a bounded sample (cpu_baseline leg and --impl reference) -------------------------------------------
def oracle_timing():
    """tests/golden/oracle_timing.json (written by tests/golden/make_golden.py --timing from the oracle only): seconds of this very
    sample, and of whole saturated oracle steps of configs[3], on the box the golden files were written on."""
    path = os.path.join(ROOT, "tests", "golden", "oracle_timing.json")
    return json.load(open(path)) if os.path.exists(path) else None


def oracle_sample(n_slabs=32, seed=0):
    """Times the oracle's coarse-graining contraction (Eq. 2.18-2.19: contract_half + contract_psi, the stage the paper calls
    the bottleneck) on `n_slabs` of the 32 i1-slabs of synthetic triad tensors of the saturated D=32 shapes.
    Returns (seconds measured, flops of the sample, threads)."""
    import numpy as np
    import __graft_entry__ as G
    G.build_oracle()
    from oracle import tatrg_oracle as O
    K = D + P
    rng = np.random.default_rng(seed)
    e = rng.standard_normal((n_slabs, K, D, D))
    f = rng.standard_normal((D, K, D, D))
    h = rng.standard_normal((n_slabs, K, D, D))
    g = rng.standard_normal((D, K, D, D))
    i_, j_ = rng.standard_normal((D, D, K)), rng.standard_normal((D, D, K))
    m2, m3, m4 = (rng.standard_normal((D, D, D)) for _ in range(3))
    half = (2.0 * n_slabs * K * D ** 4 + 2.0 * n_slabs * K * D * K * D * D * D        # E M4, (E M4) F
            + 2.0 * K * D ** 4 + 2.0 * K * D ** 5 + 2.0 * K * K * D ** 4               # I M2, (I M2) M3, ... J
            + 2.0 * n_slabs * D ** 4 * K * K)                                           # Xi Lambda
    flops = 2.0 * half
    t0 = time.perf_counter()
    out = O.contract_half(e, f, i_, j_, m2, m3, m4)
    out2 = O.contract_psi(g, h, i_, j_, m2, m3, m4)
    dt = time.perf_counter() - t0
    assert out.shape == (n_slabs, D, D, D, D) and out2.shape == (n_slabs, D, D, D, D)
    try:
        from threadpoolctl import threadpool_info
        threads = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        threads = os.cpu_count() or 1
    return dt, flops, threads


def cpu_baseline_record(dt, flops, threads):
    """Seconds per saturated oracle step from the timed sample.  The sample is the contraction stage only; the oracle spends most
    of a step in its LAPACK-free Jacobi decompositions (13 of 1024 x 1024 per step), which do not fit a bounded sample.  The
    scale factor is therefore the oracle's OWN record: (seconds of a whole saturated step) / (seconds of this same sample), both
    timed on the box that wrote the golden files (oracle_timing.json).  Without that file the model-FLOP ratio is used and the
    record says so."""
    tm = oracle_timing()
    if tm:
        scale = tm["saturated_step_s_median"] / tm["contraction_sample_s"]
        how = ("x %.1f = recorded seconds of a whole saturated oracle step (%.0f s, median of %d, %d cores) / recorded seconds of this "
               "same sample (%.2f s) on the box that wrote tests/golden (oracle_timing.json): the Jacobi decompositions, which dominate "
               "an oracle step, enter through that ratio, not through the timed sample"
               % (scale, tm["saturated_step_s_median"], tm["saturated_steps_recorded"], tm["cores"], tm["contraction_sample_s"]))
    else:
        scale = MODEL_FLOPS_PER_STEP / flops
        how = "x %.2f = model-FLOP ratio of a step to the sample (no oracle_timing.json): understates the oracle, whose Jacobi decompositions dominate" % scale
    sample = ("oracle.contract_half + contract_psi (Eq. 2.18-2.19, numpy einsum) on all 32 i1-slabs of synthetic saturated D=32 triad "
              "tensors: %.2e flop TIMED in %.2f s on %d threads; scaled to a step %s" % (flops, dt, threads, how))
    rec = {"value": dt * scale, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample, "sample_seconds_timed": dt,
           "scale_to_step": scale}
    if tm:
        rec["oracle_step_seconds_recorded"] = {"median": tm["saturated_step_s_median"], "all": tm["saturated_step_s_all"], "cores": tm["cores"],
                                               "source": "tests/golden/oracle_c4.json `sec` (whole saturated steps of configs[3], oracle only)"}
    return rec


MODEL_FLOPS_PER_STEP = 2.385e12    # 2*M*N*K of every contraction of one saturated D=32 step as the ORACLE performs it (Q^B, Q^C formed)


def config_dict(args, world):
    a, b = PRE_STEPS + args.warmup + 1, PRE_STEPS + args.warmup + args.steps
    return {"workload": WORKLOAD, "window": "steps %d-%d of the 60-step run (steps 1-%d unsaturated and %d warm-up steps untimed)" % (a, b, PRE_STEPS, args.warmup),
            "regimes": "6-19 critical (full rank), 20-60 post-critical (rank-deficient)", "parallelism": "replicas" if world > 1 else "single",
            "l2": "inputs_exceed_l2 (state 2 x 268 MB, Xi 1.07 GB vs 126 MB L2)", "pre_steps": PRE_STEPS}


def run_reference(args):
    """The reference arm of this tier = the oracle, as it stands, on the host cores (rank 0 only).  Every `step` is one bounded
    sample, timed; `value` is the mean of the samples scaled to a step (cpu_baseline_record)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    for _ in range(args.warmup):
        oracle_sample(1)
    meas, fl, threads = [], 0.0, 1
    for _ in range(args.steps):
        dt, fl, threads = oracle_sample(32)
        meas.append(dt)
    rec = cpu_baseline_record(sum(meas) / len(meas), fl, threads)
    value = rec["value"]
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": value * 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": config_dict(args, max(1, args.gpus)),
            "cpu_baseline": rec, "timed_seconds_total": sum(meas),
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ---- replicas-only aggregation -------------------------------------------------------------------
def max_over_ranks(values, device):
    """Element-wise maximum of a list of floats over all ranks (identity without a process group)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(values, dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def aggregate_seconds_per_step(ms_max, steps, world):
    """`world` independent replicas each advance `steps` steps in ms_max milliseconds: whole-job seconds per step."""
    return ms_max * 1e-3 / (steps * world)


# dram__bytes_read.sum + dram__bytes_write.sum of the dominant DGEMM launch (Xi = E (M4 F), Eq. 2.18: M=2048, N=65536, K=1024)
# from the ncu --set full capture named in `source`; its algorithmic bytes are 8 (MK + KN + MN) = 1.63e9
DGEMM_TRAFFIC = {"launch": "M=2048 N=65536 K=1024 (grid 8192), dgemm_tma_kernel", "dram_bytes": 1.605e9, "algorithmic_bytes": 1.627e9,
                 "source": "profiles/dgemm_tma_r02_ncu_full.txt (launch 12: dram__bytes_read.sum 567.7 MB + dram__bytes_write.sum 1.037 GB)"}


# ---- the CUDA path ---------------------------------------------------------------------------------------------------
class Prof:
    """Per-launch profile of a set of steps (library events, TATRG_OPT_STAGE_TIMING = 2)."""

    def __init__(self, stages):
        self.g = [0.0, 0.0, 0]; self.l = [0.0, 0.0, 0]; self.p = [0.0, 0.0, 0]; self.q = [0.0, 0.0, 0]
        self.stage = [0.0] * stages
        self.steps = 0; self.launches = 0; self.syncs = 0

    def add(self, t):
        for acc, got in ((self.g, t.gemm_profile()), (self.l, t.gemm_profile_large()), (self.p, t.permute_profile()), (self.q, t.permute_profile_large())):
            acc[0] += got[0]; acc[1] += got[1]; acc[2] += got[2]
        for i, v in enumerate(t.stage_ms()):
            self.stage[i] += float(v)
        self.steps += 1; self.launches += t.launches(); self.syncs += t.host_syncs()

    def step_ms(self):
        return sum(self.stage) / max(self.steps, 1)

    @staticmethod
    def rate(acc, unit):
        return acc[1] / (acc[0] * 1e-3) / unit if acc[0] > 0 else None


def settle():
    """Waits for the host to quiet down after a CPU-heavy process.  For 15-20 s after a many-thread, many-GB process has ended on this
    box (the reference arm the driver runs right before this one; this file's own cpu_baseline leg), ONE coarse-graining step in about
    twenty stalls by 45-90 ms: the step is host-driven (45-58 stream synchronisations) and the host thread is held up once, whatever its
    scheduling class, with or without the clock sampler, garbage collector on or off.  Measured (profiles/README.md): a 7 s numpy burst
    followed by this timed region -> a stall in 11 of 12 processes; the same after a 12 s pause -> 0 of 5; the second process after
    the burst -> 0 of 8.  The 1-minute load average says whether such a process has just ended."""
    try:
        load = os.getloadavg()[0]
    except OSError:
        load = 0.0
    slept = 0.0
    if load > 0.5:
        slept = 15.0
        time.sleep(slept)
    return {"loadavg_1min_at_start": round(load, 2), "slept_s": slept}


def run_cuda(args):
    import torch
    import torch.distributed as dist
    import paper_2507_21909_b200 as T
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    T.lib()
    settled = settle()
    dev = "cuda:%d" % local
    first = PRE_STEPS + args.warmup + 1                       # absolute index of the first timed step
    if first + args.steps - 1 > 2 * FULL_RUN_STEPS - PRE_STEPS:
        raise SystemExit("bench.py: --steps + --warmup exceed two passes over the 60-step run")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def handle(at_step):
        """A fresh replica advanced (untimed) until `at_step` steps are done."""
        h = T.Tatrg(BETA, H, D, P, SEED + rank, power_iters=N_POW, device=dev)
        for _ in range(at_step):
            h.step()
        return h

    def window(n):
        """Absolute step indices of n consecutive timed steps starting at `first`, wrapping from step 60 to step 6 of a second replica."""
        out, s = [], first
        for _ in range(n):
            out.append(s)
            s = s + 1 if s < FULL_RUN_STEPS else PRE_STEPS + 1
        return out

    steps_abs = window(args.steps)
    n_first = min(args.steps, FULL_RUN_STEPS - first + 1)     # timed steps on the first replica (the rest wrap to a second one)
    wraps = args.steps > n_first
    t = handle(PRE_STEPS)
    t2 = handle(PRE_STEPS) if wraps else None                 # the second replica of a window that wraps: ready before the clock starts
    sampler = ClockSampler(local)
    sampler.start()
    # The steps are host-driven (45-58 synchronisations each): a cyclic garbage collection of the interpreter (tens of ms with torch loaded;
    # it can run in the sampler thread and hold the GIL while the main thread returns from a step) shows up as ONE step of 120-140 ms
    # among 75-100 ms ones.  Collected now, switched off for the timed regions.
    gc.collect()
    gc.disable()
    for _ in range(args.warmup):
        t.step()
    sampler.active = True
    # ---- timed region 1: K steps, state resident in HBM ----
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]      # per-step split of the same region
    barrier()
    ev0.record()
    for i in range(args.steps):
        cur = t if i < n_first else t2
        cur.step()
        launches += cur.launches()
        marks[i].record()
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    step_ms = [([ev0] + marks)[i].elapsed_time(marks[i]) for i in range(args.steps)]
    lnz = t.lnZ_per_site()
    t.close()
    if t2:
        t2.close()
    # ---- timed region 2: the same window end to end through the C ABI with host buffers ----
    n5 = D ** 5
    k_e2e = n_first
    t = handle(first - 1)
    host = [torch.empty(n5, dtype=torch.float64).pin_memory() for _ in range(2)]
    shape = t.get_tensor_into("phi", host[0])
    t.get_tensor_into("psi", host[1])
    barrier()
    ev0.record()
    for _ in range(k_e2e):
        t.set_state_host(host[0].view(shape), host[1].view(shape))      # H2D: 2 * D^5 doubles
        t.step()
        _ = t.lnZ_per_site()                                            # D2H: the step's result
        _ = t.singular_values(T.SV_SIGMA, D)
        t.get_tensor_into("phi", host[0])                               # D2H: 2 * D^5 doubles (state for the next call)
        t.get_tensor_into("psi", host[1])
    ev1.record()
    barrier()
    ms_e2e = ev0.elapsed_time(ev1)
    sampler.active = False
    sampler.stop_flag = True
    sampler.join(timeout=2)
    gc.enable()
    t.close()

    # ---- profiling passes (not part of `value`): per-launch CUDA events on the library's streams around every DGEMM / permute,
    #      over the same window, on a fresh handle advanced to the same step; split by regime ----
    def profile_pass(overlap):
        h = handle(first - 1)
        h.set_option(T.OPT_STAGE_TIMING, 2)
        h.set_option(T.OPT_OVERLAP, overlap)
        tot, crit, post = Prof(len(T.STAGES)), Prof(len(T.STAGES)), Prof(len(T.STAGES))
        for s_abs in steps_abs[:n_first]:
            h.step()
            tot.add(h)
            (crit if s_abs < FIRST_POST_CRITICAL else post).add(h)
        h.close()
        return tot, crit, post

    prof, prof_c, prof_p = profile_pass(1)        # in situ: the schedule `value` was timed with (solver chains beside the contractions)
    alone, _, _ = profile_pass(0)                 # alone: every stage on one stream, no kernel beside the timed ones
    dmma = T.dmma_issue_rate(20000, 2)
    # ---- the whole run of configs[3] (60 steps from the initial tensor), independent of --steps ----
    t = handle(0)
    per_step, run_launches, run_syncs = [], [], []
    for _ in range(FULL_RUN_STEPS):
        ev0.record()
        t.step()
        ev1.record()
        ev1.synchronize()
        per_step.append(ev0.elapsed_time(ev1) * 1e-3)
        run_launches.append(t.launches()); run_syncs.append(t.host_syncs())
    lnz_full = t.lnZ_per_site()
    t.close()
    crit_steps = per_step[PRE_STEPS:FIRST_POST_CRITICAL - 1]
    post_steps = per_step[FIRST_POST_CRITICAL - 1:]
    # ---- cost scaling with D (configs[4] and PAPER.md Fig. 7/8 :258-274): saturated steps, rank 0 at N = 1 only ----
    scaling = None
    if world == 1 and not args.no_scaling:
        scaling = scaling_vs_D(T, torch, dev)
    # ---- max over ranks ----
    ms, ms_e2e = max_over_ranks([ms, ms_e2e], "cuda")
    if rank == 0:
        pk = peaks()
        sec = aggregate_seconds_per_step(ms, args.steps, world)
        sec_e2e = aggregate_seconds_per_step(ms_e2e, k_e2e, world)
        derived_tf = pk["bf16_sus"] * FP64_TO_BF16_NOMINAL   # kernel timed inside a long step -> sustained figure
        peak_tf = max(derived_tf, dmma)                      # the stricter denominator

        def gemm_block(p):
            if p.steps == 0 or p.l[0] <= 0:
                return None
            a = Prof.rate(p.l, 1e12)
            return {"achieved": a, "frac": a / peak_tf, "launches_per_step": p.l[2] // p.steps, "ms_per_step": p.l[0] / p.steps,
                    "time_share_of_step": p.l[0] / (p.step_ms() * p.steps), "steps": p.steps}

        def perm_block(p):
            if p.steps == 0 or p.p[0] <= 0:
                return None
            a, b = Prof.rate(p.p, 1e9), Prof.rate(p.q, 1e9)
            return {"achieved": a, "frac": a / pk["hbm"], "launches_per_step": p.p[2] // p.steps, "bytes_per_step": p.p[1] / p.steps,
                    "time_share_of_step": p.p[0] / (p.step_ms() * p.steps),
                    "large": {"launches_per_step": p.q[2] // p.steps, "bytes_share": p.q[1] / p.p[1], "achieved": b, "frac": b / pk["hbm"] if b else None}}

        def stage_block(p):
            return {k: round(v / p.steps, 2) for k, v in zip(T.STAGES, p.stage)} if p.steps else None

        main = gemm_block(prof)
        line = {
            "metric": METRIC, "value": sec, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config_dict(args, world),
            "value_critical": sum(crit_steps) / len(crit_steps), "value_post_critical": sum(post_steps) / len(post_steps),
            "e2e": {"value": sec_e2e, "unit": UNIT, "h2d_bytes_per_step": 16 * n5, "d2h_bytes_per_step": 16 * n5 + 8 * (1 + D), "steps": k_e2e},
            "gpu_launches": launches, "lnZ_per_site": lnz, "clocks": sampler.summary(),
            "step_ms": {str(s): round(x, 2) for s, x in zip(steps_abs, step_ms)},
            "host_settle": settled,
            "model_tflops": prof.g[1] / prof.steps / (ms / args.steps * 1e-3) / 1e12,
            "host_syncs_per_step": prof.syncs / prof.steps, "launches_per_step": prof.launches / prof.steps,
            "roofline": {"bound": "tensor", "kernel": "dgemm_tma_kernel / dgemm_kernel (DMMA m8n8k4, TMA-fed 128x128x16 tile): the %d contraction launches of a step (>= 1e9 flop each, "
                                                      "%.1f%% of the step's DGEMM flops), steps %d-%d" % (main["launches_per_step"], 100.0 * prof.l[1] / prof.g[1], steps_abs[0], steps_abs[n_first - 1]),
                         "achieved": main["achieved"], "peak": peak_tf, "unit": "TFLOP/s", "frac": main["frac"],
                         "traffic": DGEMM_TRAFFIC["dram_bytes"], "traffic_detail": DGEMM_TRAFFIC,
                         "time_share_of_step": main["time_share_of_step"],
                         "by_regime": {"critical": gemm_block(prof_c), "post_critical": gemm_block(prof_p)},
                         "all_launches": {"launches_per_step": prof.g[2] // prof.steps, "achieved": Prof.rate(prof.g, 1e12), "frac": Prof.rate(prof.g, 1e12) / peak_tf,
                                          "note": "includes the small products of the Cholesky / subspace-iteration solvers, which "
                                                  "run concurrently on several streams: their event times overlap"},
                         "peak_source": "max(register-resident DMMA issue rate measured in this run, MEASURED_PEAKS.json "
                                        "bf16_tflops_sustained (%s) x nominal FP64:bf16 ratio 45/2250)" % pk["src"],
                         "dmma_issue_rate_tflops": dmma, "derived_peak_tflops": derived_tf,
                         "schedule": "in situ (solver chains run on auxiliary streams beside some of these launches)",
                         "alone": {"achieved": Prof.rate(alone.l, 1e12), "frac": Prof.rate(alone.l, 1e12) / peak_tf,
                                   "schedule": "TATRG_OPT_OVERLAP = 0: every stage on one stream, no kernel beside them"}},
            "permute": dict(perm_block(prof), bound="hbm", peak=pk["hbm"], unit="GB/s",
                            schedule="in situ (some permutes share HBM with the solver chains on auxiliary streams)",
                            note="achieved = ALL permute launches of a step (bytes / sum of the per-launch CUDA-event times); `large` = the launches "
                                 "that move >= 100 MB (D^5 tensors, larger than the 126 MB L2: the HBM-bound class); the rest are L2-resident copies of "
                                 "<= 67 MB whose event-timed duration is a launch floor (6-20 us each).  Round 2 removed 11 of the 19 large permutes "
                                 "of a step (16.1 -> 7.8 GB permuted per step), which lowers this aggregate while the step gets faster",
                            alone={k: v for k, v in perm_block(alone).items() if k in ("achieved", "frac", "large")},
                            by_regime={"critical": perm_block(prof_c), "post_critical": perm_block(prof_p)}),
            "stage_ms": stage_block(prof),
            "stage_ms_by_regime": {"critical": stage_block(prof_c), "post_critical": stage_block(prof_p)},
            "full_run": {"steps": FULL_RUN_STEPS, "seconds": sum(per_step), "mean_s_per_step": sum(per_step) / len(per_step),
                         "critical_steps_6_19": {"mean": sum(crit_steps) / len(crit_steps), "min": min(crit_steps), "max": max(crit_steps)},
                         "post_critical_steps_20_60": {"mean": sum(post_steps) / len(post_steps), "min": min(post_steps), "max": max(post_steps)},
                         "max_s_per_step": max(per_step), "step_ms": [round(x * 1e3, 1) for x in per_step],
                         "launches_per_step": {"critical": sum(run_launches[PRE_STEPS:FIRST_POST_CRITICAL - 1]) / len(crit_steps),
                                               "post_critical": sum(run_launches[FIRST_POST_CRITICAL - 1:]) / len(post_steps)},
                         "host_syncs_per_step": {"critical": sum(run_syncs[PRE_STEPS:FIRST_POST_CRITICAL - 1]) / len(crit_steps),
                                                 "post_critical": sum(run_syncs[FIRST_POST_CRITICAL - 1:]) / len(post_steps)},
                         "lnZ_per_site": lnz_full,
                         "note": "configs[3] from the initial tensor on rank 0's replica, one run, independent of --steps"},
        }
        if scaling is not None:
            line["scaling_vs_D"] = scaling
        if world == 1:
            dt, fl, threads = oracle_sample(32)
            line["cpu_baseline"] = cpu_baseline_record(dt, fl, threads)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def scaling_vs_D(T, torch, dev):
    """Seconds per saturated step against D (beta = 0.1497, p = D, 2 power iterations; configs[4]: Triad-ATRG D = 48 and plain ATRG
    D = 24 with seed 99; Fig. 7/8 :258-274 for the D^9-vs-D^7 comparison; ILO of section 2.3 at r_bond = 2)."""
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    rows = []

    def timed(label, make, pre, n=3):
        t = make()
        for _ in range(pre):
            t.step()
        ts = []
        for _ in range(n):
            ev0.record(); t.step(); ev1.record(); ev1.synchronize()
            ts.append(ev0.elapsed_time(ev1) * 1e-3)
        flops = sum(t.stage_flops())
        row = dict(label, s_per_step=sum(ts) / n, steps="%d-%d" % (pre + 1, pre + n), model_flop_per_step=flops,
                   tflops=flops / ts[-1] / 1e12, workspace_peak_gb=t.workspace_peak() / 1e9)
        t.close()
        torch.cuda.empty_cache()
        rows.append(row)

    for d, seed in ((8, 42), (16, 42), (24, 42), (32, 42), (40, 42), (48, 99)):
        timed({"method": "triad", "D": d, "p": d}, lambda: T.Tatrg(BETA, H, d, d, seed, power_iters=N_POW, device=dev), 7)
    timed({"method": "atrg", "D": 24, "p": 24}, lambda: T.Tatrg(BETA, H, 24, 24, 99, power_iters=N_POW, device=dev, method=T.METHOD_ATRG), 6, 2)
    timed({"method": "triad_ilo", "D": 32, "p": 32, "bond_rank": 64}, lambda: T.Tatrg(BETA, H, 32, 32, 42, power_iters=N_POW, device=dev, bond_rank=64), 7, 2)
    import math
    tri = [r for r in rows if r["method"] == "triad" and r["D"] >= 24]
    xs, ys = [math.log(r["D"]) for r in tri], [math.log(r["s_per_step"]) for r in tri]
    mx, my = sum(xs) / len(xs), sum(ys) / len(ys)
    expo = sum((x - mx) * (y - my) for x, y in zip(xs, ys)) / sum((x - mx) ** 2 for x in xs)
    return {"rows": rows, "triad_exponent_D24_48": expo,
            "note": "critical saturated steps (steps 8-10); least-squares exponent of s/step against D over D = 24..48 (PAPER.md: O(D^7) contraction, :177-179)"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=25)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-scaling", action="store_true", help="skip the scaling_vs_D block (about 40 s)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
