"""bench.py -- sec/step and FP64 TFLOP/s of the Triad-ATRG hot path at D = 32 on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Workload: BASELINE.json configs[3] -- 4D Ising, beta = 0.1497, h = 0, Triad-ATRG D = 32, p = 32 (K = l = 64), 2 power
iterations, Philox seed 42.  A "step" is one coarse-graining step of the whole hot path (Fig. 5 a-f) in the
saturated regime (all legs = D, reached after 5 steps; those 5 unsaturated steps are run before the warm-up).
`value` = seconds per step with the state resident in HBM; `e2e` = the same through the C ABI with HOST buffers
(state uploaded from pinned memory before, and downloaded after, every step, inside the timed region).
Replicas only for N > 1: every rank coarse-grains its own network, no collective in the path.

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
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

BETA, H, D, P, N_POW, SEED = 0.1497, 0.0, 32, 32, 2, 42
PRE_STEPS = 5                      # legs grow 2 -> 4 -> 16 -> 32: saturated from step 6 on
FULL_RUN_STEPS = 60                # configs[3]: 2^15 per axis
METRIC = "sec_per_coarse_graining_step_D32"
UNIT = "s/step"
WORKLOAD = "configs[3]: 4D Ising beta=0.1497 h=0, Triad-ATRG D=32 p=32 (K=l=64), 2 power iterations, Philox seed 42, saturated steps"
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
            time.sleep(0.05 if self.nvml else 0.2)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s), "source": "nvml" if self.nvml else "nvidia-smi"}


# ---- the oracle on a bounded sample (cpu_baseline leg and --impl reference) -------------------------------------------
MODEL_FLOPS_PER_STEP = 2.385e12    # 2*M*N*K of every contraction of one saturated D=32 step as the ORACLE performs it (Q^B, Q^C formed
                                   # explicitly; the library counted this before it made them implicit, it now counts 2.115e12)


def oracle_sample(n_slabs=32, seed=0):
    """Times the oracle's coarse-graining contraction (Eq. 2.18-2.19: contract_half + contract_psi, the FLOP-dominant
    stage, ~48 % of a step's model FLOPs) on `n_slabs` of the 32 i1-slabs of synthetic triad tensors of the saturated
    D=32 shapes, and extrapolates to a whole step by the model-FLOP ratio.  The oracle's Jacobi decompositions are NOT
    in the sample (one saturated oracle step took 12 min on 8 cores when tests/golden/oracle_c4.json was written).
    Returns (seconds per step extrapolated, seconds measured, flops of the sample, threads)."""
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
    return dt * MODEL_FLOPS_PER_STEP / flops, dt, flops, threads


SAMPLE_TEXT = ("oracle.contract_half + contract_psi (Eq. 2.18-2.19, numpy einsum) on all 32 i1-slabs of synthetic saturated D=32 triad "
               "tensors: %.2e flop in %.2f s, extrapolated to a step by the model-FLOP ratio (%.3e flop/step); the oracle's "
               "Jacobi decompositions are not in the sample")


def run_reference(args):
    """The reference arm of this tier = the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    for _ in range(args.warmup):
        oracle_sample(1)
    vals, meas, threads = [], [], 1
    for _ in range(args.steps):
        v, dt, fl, threads = oracle_sample(32)
        vals.append(v)
        meas.append(dt)
    value = sum(vals) / len(vals)
    sample = SAMPLE_TEXT % (fl, sum(meas) / len(meas), MODEL_FLOPS_PER_STEP)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": value * 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": WORKLOAD, "l2": "inputs_exceed_l2"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
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


# dram__bytes_read.sum + dram__bytes_write.sum of the dominant DGEMM launch (Xi = E (M4 F), Eq. 2.18: M=2048, N=65536, K=1024, 8.6 ms)
# from the ncu --set full capture in profiles/dgemm_r01_ncu_full.txt; its algorithmic bytes are 8 (MK + KN + MN) = 1.63e9
DGEMM_TRAFFIC = {"launch": "M=2048 N=65536 K=1024 (grid 8192)", "dram_bytes": 1.602e9, "algorithmic_bytes": 1.627e9,
                 "source": "profiles/dgemm_r01_ncu_full.txt"}


# ---- the CUDA path ---------------------------------------------------------------------------------------------------
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

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    t = T.Tatrg(BETA, H, D, P, SEED + rank, power_iters=N_POW, device="cuda:%d" % local)
    for _ in range(PRE_STEPS):
        t.step()
    sampler = ClockSampler(local)
    sampler.start()
    for _ in range(args.warmup):
        t.step()
    sampler.active = True
    # ---- timed region 1: K steps, state resident in HBM ----
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]      # per-step split of the same region (diagnostic)
    barrier()
    ev0.record()
    for i in range(args.steps):
        t.step()
        launches += t.launches()
        marks[i].record()
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    step_ms = [([ev0] + marks)[i].elapsed_time(marks[i]) for i in range(args.steps)]
    lnz = t.lnZ_per_site()
    # ---- timed region 2: end to end through the C ABI with host buffers ----
    n5 = D ** 5
    host = [torch.empty(n5, dtype=torch.float64).pin_memory() for _ in range(2)]
    shape = t.get_tensor_into("phi", host[0])
    t.get_tensor_into("psi", host[1])
    k_e2e = max(1, min(args.steps, 3))
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
    # ---- profiling pass (not part of `value`): per-launch CUDA events on the library's stream around every DGEMM / permute ----
    t.set_option(T.OPT_STAGE_TIMING, 2)
    n_prof = max(1, min(args.steps, 3))

    def profile_pass():
        g_ms = g_fl = p_ms = p_by = l_ms = l_fl = q_ms = q_by = 0.0
        g_n = p_n = l_n = q_n = 0
        stage = None
        step_ms_prof = 0.0
        for _ in range(n_prof):
            t.step()
            a, b, c = t.gemm_profile()
            g_ms, g_fl, g_n = g_ms + a, g_fl + b, g_n + c
            a, b, c = t.gemm_profile_large()
            l_ms, l_fl, l_n = l_ms + a, l_fl + b, l_n + c
            a, b, c = t.permute_profile()
            p_ms, p_by, p_n = p_ms + a, p_by + b, p_n + c
            a, b, c = t.permute_profile_large()
            q_ms, q_by, q_n = q_ms + a, q_by + b, q_n + c
            sm = t.stage_ms()
            stage = sm if stage is None else stage + sm
            step_ms_prof += float(sm.sum())
        return g_ms, g_fl, g_n, l_ms, l_fl, l_n, p_ms, p_by, p_n, stage, step_ms_prof, q_ms, q_by, q_n

    # in situ: the schedule `value` was timed with (solver chains on auxiliary streams beside the contractions)
    g_ms, g_fl, g_n, l_ms, l_fl, l_n, p_ms, p_by, p_n, stage, step_ms_prof, q_ms, q_by, q_n = profile_pass()
    # alone: the same kernels with every stage on one stream (TATRG_NO_OVERLAP=1), i.e. without other kernels beside them
    os.environ["TATRG_NO_OVERLAP"] = "1"
    _, _, _, la_ms, la_fl, _, pa_ms, pa_by, _, _, _, qa_ms, qa_by, _ = profile_pass()
    del os.environ["TATRG_NO_OVERLAP"]
    t.set_option(T.OPT_STAGE_TIMING, 0)
    dmma = T.dmma_issue_rate(20000, 2)
    # ---- the whole run of configs[3] (60 steps from the initial tensor), not part of `value`: total run time (north_star) ----
    # After the flow has left criticality (step ~20 at this beta) the local tensor is numerically rank-deficient and the
    # rank-revealing full decompositions replace Cholesky QR / subspace iteration: those steps are slower.
    t.close()
    t = T.Tatrg(BETA, H, D, P, SEED + rank, power_iters=N_POW, device="cuda:%d" % local)
    per_step = []
    for _ in range(FULL_RUN_STEPS):
        ev0.record()
        t.step()
        ev1.record()
        ev1.synchronize()
        per_step.append(ev0.elapsed_time(ev1) * 1e-3)
    lnz_full = t.lnZ_per_site()
    sat = sorted(per_step[PRE_STEPS:])
    # ---- max over ranks ----
    ms, ms_e2e = max_over_ranks([ms, ms_e2e], "cuda")
    if rank == 0:
        pk = peaks()
        sec = aggregate_seconds_per_step(ms, args.steps, world)
        sec_e2e = aggregate_seconds_per_step(ms_e2e, k_e2e, world)
        derived_tf = pk["bf16_sus"] * FP64_TO_BF16_NOMINAL   # kernel timed inside a long step -> sustained figure
        peak_tf = max(derived_tf, dmma)                      # the stricter denominator
        ach_tf = l_fl / (l_ms * 1e-3) / 1e12         # the contractions proper: DGEMM launches of >= 1e9 flop
        all_tf = g_fl / (g_ms * 1e-3) / 1e12         # every DGEMM launch, the small products of the solvers included
        line = {
            "metric": METRIC, "value": sec, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": WORKLOAD, "parallelism": "replicas" if world > 1 else "single",
                                            "l2": "inputs_exceed_l2 (state 2 x 268 MB, Xi 1.07 GB vs 126 MB L2)", "pre_steps": PRE_STEPS},
            "e2e": {"value": sec_e2e, "unit": UNIT, "h2d_bytes_per_step": 16 * n5, "d2h_bytes_per_step": 16 * n5 + 8 * (1 + D), "steps": k_e2e},
            "gpu_launches": launches, "lnZ_per_site": lnz, "clocks": sampler.summary(), "step_ms": [round(x, 2) for x in step_ms],
            "model_tflops": g_fl / n_prof / (ms / args.steps * 1e-3) / 1e12,
            "roofline": {"bound": "tensor", "kernel": "dgemm_kernel (DMMA m8n8k4): the %d contraction launches of a step (>= 1e9 flop each, "
                                                      "%.1f%% of the step's DGEMM flops)" % (l_n // n_prof, 100.0 * l_fl / g_fl),
                         "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach_tf / peak_tf,
                         "traffic": DGEMM_TRAFFIC["dram_bytes"], "traffic_detail": DGEMM_TRAFFIC,
                         "all_launches": {"launches_per_step": g_n // n_prof, "achieved": all_tf, "frac": all_tf / peak_tf,
                                          "note": "includes the small products of the Cholesky / subspace-iteration solvers, which "
                                                  "run concurrently on several streams: their event times overlap"},
                         "peak_source": "max(register-resident DMMA issue rate measured in this run, MEASURED_PEAKS.json "
                                        "bf16_tflops_sustained (%s) x nominal FP64:bf16 ratio 45/2250)" % pk["src"],
                         "dmma_issue_rate_tflops": dmma, "derived_peak_tflops": derived_tf, "time_share_of_step": l_ms / step_ms_prof,
                         "schedule": "in situ (solver chains run on auxiliary streams beside some of these launches)",
                         "alone": {"achieved": la_fl / (la_ms * 1e-3) / 1e12, "frac": la_fl / (la_ms * 1e-3) / 1e12 / peak_tf,
                                   "schedule": "TATRG_NO_OVERLAP=1: every stage on one stream, no kernel beside them"}},
            "permute": {"bound": "hbm", "achieved": p_by / (p_ms * 1e-3) / 1e9, "peak": pk["hbm"], "unit": "GB/s",
                        "frac": p_by / (p_ms * 1e-3) / 1e9 / pk["hbm"], "launches_per_step": p_n // n_prof,
                        "time_share_of_step": p_ms / step_ms_prof,
                        "schedule": "in situ (some permutes share HBM with the solver chains on auxiliary streams)",
                        "alone": {"achieved": pa_by / (pa_ms * 1e-3) / 1e9, "frac": pa_by / (pa_ms * 1e-3) / 1e9 / pk["hbm"],
                                  "schedule": "TATRG_NO_OVERLAP=1: every stage on one stream, no kernel beside them"},
                        "large": {"what": "the %d permutes of a step that move >= 100 MB (tensors larger than L2: the D^5 operands); the other "
                                          "launches are L2-resident permutes of ~10 us, where the events around a launch cost as much as the "
                                          "launch" % (q_n // n_prof),
                                  "bytes_share": q_by / p_by, "achieved": q_by / (q_ms * 1e-3) / 1e9, "frac": q_by / (q_ms * 1e-3) / 1e9 / pk["hbm"],
                                  "alone": {"achieved": qa_by / (qa_ms * 1e-3) / 1e9, "frac": qa_by / (qa_ms * 1e-3) / 1e9 / pk["hbm"]}}},
            "stage_ms": {k: round(float(v) / n_prof, 2) for k, v in zip(T.STAGES, stage) if not k.startswith("_")},
            "full_run": {"steps": FULL_RUN_STEPS, "seconds": sum(per_step), "mean_s_per_step": sum(per_step) / len(per_step),
                         "median_s_per_step_saturated": sat[len(sat) // 2], "min_s_per_step_saturated": sat[0], "max_s_per_step": max(per_step),
                         "lnZ_per_site": lnz_full,
                         "note": "configs[3] from the initial tensor on rank 0's replica; steps after the flow leaves criticality run "
                                 "rank-revealing full decompositions (numerically rank-deficient tensors) and are slower than `value`"},
        }
        if world == 1:
            v, dt, fl, threads = oracle_sample(32)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                                    "sample": SAMPLE_TEXT % (fl, dt, MODEL_FLOPS_PER_STEP)}
        print(json.dumps(line))
    t.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
