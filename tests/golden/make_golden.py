"""Writes tests/golden/oracle_<name>.json from the CPU oracle ONLY (never from the CUDA path).

    python tests/golden/make_golden.py c1 c2 c3 [c4:12]      (name[:steps])
    GOLDEN_CKPT=/some/dir python tests/golden/make_golden.py c4:26    (long runs: state saved after each step)
    GOLDEN_OUT=/some/dir ...                                         (write there instead of tests/golden/: a run restarted from
                                                                      step 0 must not shorten the committed file while it grows)
    python tests/golden/make_golden.py --timing                      (oracle_timing.json: what bench.py scales its CPU sample by)

Each file holds, per step: ln Z/V, the bond-swap spectrum sigma/sigma_1 and the T-decomposition spectrum s/s_1
for one BASELINE.json config (see tests/inputs.py::configs); these take minutes to hours on a CPU, so the GPU
parity tests read them instead of re-running the oracle.  Expected values are reproducible: rerun this script.
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import tatrg_oracle as O  # noqa: E402

RUNS = {
    # name: list of (tag, beta, h, D, p, n_pow, seed, steps)
    "c1": [("b0.14", 0.14, 0.0, 4, 4, 1, 1234, 16)],
    "c2": [("b%g_s%d" % (b, s), b, 0.0, 8, 8, 2, s, 40)
           for b, s in zip((0.140, 0.145, 0.1497, 0.155, 0.160), (1, 2, 3, 4, 5))],
    "c3": [("h+1e-3", 0.1497, 1e-3, 16, 16, 2, 7, 48), ("h-1e-3", 0.1497, -1e-3, 16, 16, 2, 7, 48)],
    "c4": [("b0.1497", 0.1497, 0.0, 32, 32, 2, 42, 60)],
    # configs[4]: only the first steps are affordable (c5:3, c5a:3 -- step 4 of either takes hours: n = 2304 Jacobi problems resp. the one-einsum
    # O(D^9) definition at D = 24); the saturated steps are checked slab by slab / fibre by fibre on the GPU box
    "c5": [("d48", 0.1497, 0.0, 48, 48, 2, 99, 60)],
    "c5a": [("atrg_d24", 0.1497, 0.0, 24, 24, 2, 99, 60, {"method": "atrg"})],
}

def timing():
    """oracle_timing.json: seconds of the oracle's coarse-graining contraction (Eq. 2.18-2.19, contract_half + contract_psi on
    saturated D = 32 shapes: the bounded sample bench.py times as cpu_baseline) on THIS box, next to the seconds the oracle took
    for whole saturated steps of configs[3] on the same box (oracle_c4.json `sec`).  Their ratio turns bench.py's timed sample
    into seconds per step; both numbers are oracle timings, none comes from the CUDA path."""
    D, K = 32, 64
    rng = np.random.default_rng(0)
    e, h = rng.standard_normal((D, K, D, D)), rng.standard_normal((D, K, D, D))
    f, g = rng.standard_normal((D, K, D, D)), rng.standard_normal((D, K, D, D))
    i_, j_ = rng.standard_normal((D, D, K)), rng.standard_normal((D, D, K))
    m2, m3, m4 = (rng.standard_normal((D, D, D)) for _ in range(3))
    best = None
    for _ in range(3):
        t0 = time.time()
        O.contract_half(e, f, i_, j_, m2, m3, m4)
        O.contract_psi(g, h, i_, j_, m2, m3, m4)
        dt = time.time() - t0
        best = dt if best is None else min(best, dt)
    here = os.path.dirname(__file__)
    sec = json.load(open(os.path.join(here, "oracle_c4.json")))["runs"][0]["sec"]
    sat = sorted(sec[5:])                      # steps 6.. are saturated
    out = {"generator": "tests/golden/make_golden.py --timing (oracle only)", "cores": os.cpu_count(),
           "contraction_sample_s": round(best, 3), "saturated_step_s_median": sat[len(sat) // 2], "saturated_steps_recorded": len(sat),
           "saturated_step_s_all": sat}
    json.dump(out, open(os.path.join(here, "oracle_timing.json"), "w"), indent=1)
    print(out)


if __name__ == "__main__":
    if "--timing" in sys.argv:
        timing()
        sys.exit(0)
    outdir = os.environ.get("GOLDEN_OUT") or os.path.dirname(__file__)
    for arg in sys.argv[1:]:
        name, _, lim = arg.partition(":")
        out = {"generator": "tests/golden/make_golden.py (oracle only)", "runs": []}
        for tag, beta, h, D, p, n_pow, seed, steps, *kw in RUNS[name]:
            steps = min(steps, int(lim)) if lim else steps
            o = O.TatrgOracle(beta, h, D, p, seed, n_pow=n_pow, **(kw[0] if kw else {}))
            rec = dict(tag=tag, beta=beta, h=h, D=D, oversample=p, n_pow=n_pow, seed=seed, lnZ=[], sigma=[], s=[], sec=[], **(kw[0] if kw else {}))
            # optional resume of a multi-hour run: the oracle's whole state is (Phi, Psi, [ln c_m], m) plus what was recorded
            ckpt = os.environ.get("GOLDEN_CKPT") and os.path.join(os.environ["GOLDEN_CKPT"], "ckpt_%s_%s.npz" % (name, tag))
            if ckpt and os.path.exists(ckpt):
                z = np.load(ckpt, allow_pickle=False)
                o.phi, o.psi, o.lnc, o.m = z["phi"], z["psi"], list(z["lnc"]), int(z["m"])
                rec = json.loads(str(z["rec"]))
            for m in range(o.m, steps):
                t0 = time.time()
                o.step()
                rec["lnZ"].append(o.lnZ_per_site())
                rec["sigma"].append([float(x) for x in o.last["sigma"][:D]])
                rec["s"].append([float(x) for x in o.last["s"][:D]])
                rec["sec"].append(round(time.time() - t0, 3))
                print(name, tag, m + 1, rec["lnZ"][-1], rec["sec"][-1], flush=True)
                json.dump(out | {"runs": out["runs"] + [rec]}, open(os.path.join(outdir, "oracle_%s.json" % name), "w"), indent=0)
                if ckpt:
                    np.savez(ckpt + ".tmp.npz", phi=o.phi, psi=o.psi, lnc=np.array(o.lnc), m=o.m, rec=json.dumps(rec))
                    os.replace(ckpt + ".tmp.npz", ckpt)
            out["runs"].append(rec)
        json.dump(out, open(os.path.join(outdir, "oracle_%s.json" % name), "w"), indent=0)
