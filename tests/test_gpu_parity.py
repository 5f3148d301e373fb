"""GPU parity tests proper: the CUDA Triad-ATRG path, through the C ABI, against the CPU oracle on the same seeded
inputs.  Only gauge-invariant quantities are compared (SVD signs and bases are not unique):

    ln Z / V                          relative error <= 1e-10   (north_star)
    retained singular values          absolute error <= 1e-9 of the leading value   (north_star)
    projectors / reconstructions      stage by stage, teacher-forced from the oracle's state

Expected values come from tests/golden/*.json, written by tests/golden/make_golden.py from the oracle ONLY, or from
the oracle run inside the test for the small cases."""
import json
import math
import os

import numpy as np
import pytest

import paper_2507_21909_b200 as T

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))
TOL_LNZ, TOL_SV = 1e-10, 1e-9


def golden(name):
    path = os.path.join(HERE, "golden", "oracle_%s.json" % name)
    if not os.path.exists(path):
        pytest.skip("golden file %s not generated" % name)
    return json.load(open(path))["runs"]


def run_against(rec, max_steps=None, subspace=1):
    t = T.Tatrg(rec["beta"], rec["h"], rec["D"], rec["oversample"], rec["seed"], power_iters=rec["n_pow"])
    t.set_option(T.OPT_SUBSPACE, subspace)
    n = len(rec["lnZ"]) if max_steps is None else min(max_steps, len(rec["lnZ"]))
    worst = [0.0, 0.0, 0.0]
    for m in range(n):
        t.step()
        lz = t.lnZ_per_site()
        worst[0] = max(worst[0], abs(lz - rec["lnZ"][m]) / abs(rec["lnZ"][m]))
        for i, (which, key) in enumerate(((T.SV_SIGMA, "sigma"), (T.SV_S, "s"))):
            got = t.singular_values(which, rec["D"])
            ref = np.zeros(rec["D"])
            ref[:len(rec[key][m])] = rec[key][m]
            g = np.zeros(rec["D"])
            g[:len(got)] = got
            worst[1 + i] = max(worst[1 + i], float(np.abs(g - ref).max()))
    assert t.steps_done() == n and t.launches() > 0
    t.close()
    return worst


def test_config1_full_run():
    """BASELINE.json configs[0]: 16^4, beta=0.14, D=4, p=4, 1 power iteration, seed 1234."""
    (rec,) = golden("c1")
    w = run_against(rec)
    assert w[0] <= TOL_LNZ and w[1] <= TOL_SV and w[2] <= TOL_SV, w


@pytest.mark.parametrize("idx", range(5))
def test_config2_beta_sweep(idx):
    """configs[1]: 2^10 per axis (40 steps), D=8, p=8, 2 power iterations, five (beta, seed) pairs around T_c."""
    rec = golden("c2")[idx]
    w = run_against(rec)
    assert w[0] <= TOL_LNZ and w[1] <= TOL_SV and w[2] <= TOL_SV, w


@pytest.mark.parametrize("idx", range(2))
@pytest.mark.parametrize("subspace", [1, 0])
def test_config3_field(idx, subspace):
    """configs[2]: 2^12 per axis (48 steps), D=16, p=16, h = +-1e-3, seed 7.  subspace = 1: leading eigenvectors by subspace
    iteration + Cholesky QR (the default path); 0: full eigen-decompositions everywhere (TATRG_OPT_SUBSPACE)."""
    rec = golden("c3")[idx]
    w = run_against(rec, subspace=subspace)
    assert w[0] <= TOL_LNZ and w[1] <= TOL_SV and w[2] <= TOL_SV, w


@pytest.mark.parametrize("subspace", [1, 0])
def test_config4_first_steps_at_full_size(subspace):
    """configs[3] (headline, D=32, p=32): as many steps as the oracle could afford (the weight of step m in ln Z/V is
    2^-m); the remaining steps are covered by test_d32_stage_properties."""
    (rec,) = golden("c4")
    w = run_against(rec, subspace=subspace)
    assert w[0] <= TOL_LNZ and w[1] <= TOL_SV and w[2] <= TOL_SV, w


@pytest.mark.parametrize("idx", range(2))
def test_config3_field_with_plain_orthogonal_iteration(idx):
    """configs[2] once more with TATRG_OPT_CHEBYSHEV = 0: plain powers of the Gram matrix per orthonormalisation instead of the
    Chebyshev-filtered cycles the default path takes (which test_config3_field covers); same oracle, same tolerance."""
    rec = golden("c3")[idx]
    t = T.Tatrg(rec["beta"], rec["h"], rec["D"], rec["oversample"], rec["seed"], power_iters=rec["n_pow"])
    t.set_option(T.OPT_CHEBYSHEV, 0)
    for m in range(len(rec["lnZ"])):
        t.step()
        assert abs(t.lnZ_per_site() - rec["lnZ"][m]) <= TOL_LNZ * abs(rec["lnZ"][m]), m
        got = t.singular_values(T.SV_SIGMA, rec["D"])
        ref = np.zeros(rec["D"]); ref[:len(rec["sigma"][m])] = rec["sigma"][m]
        g = np.zeros(rec["D"]); g[:len(got)] = got
        assert np.abs(g - ref).max() <= TOL_SV, m
    t.close()


def test_chebyshev_and_plain_iterations_agree_at_d32():
    """TATRG_OPT_CHEBYSHEV 1 / 0 at D = 32 through 24 steps (critical and post-critical regime, block widening included): the filtered
    iteration converges to the same isometries (ln Z/V to 1e-12, spectra to 1e-10) in fewer launches."""
    runs = []
    for cheb in (1, 0):
        t = T.Tatrg(0.1497, 0.0, 32, 32, 42)
        t.set_option(T.OPT_CHEBYSHEV, cheb)
        out, launches = [], 0
        for _ in range(24):
            t.step()
            launches += t.launches()
            out.append((t.lnZ_per_site(), t.singular_values(T.SV_SIGMA, 32), t.singular_values(T.SV_S, 32)))
        runs.append((out, launches))
        t.close()
    for a, b in zip(runs[0][0], runs[1][0]):
        assert abs(a[0] - b[0]) <= 1e-12 * abs(b[0])
        assert np.abs(a[1] - b[1]).max() <= 1e-10 and np.abs(a[2] - b[2]).max() <= 1e-10
    assert runs[0][1] < runs[1][1]


def test_subspace_and_full_decompositions_agree_at_d32():
    """The two ways of getting the triad isometries / squeezers / QR factors (TATRG_OPT_SUBSPACE 1 / 0) give the same
    physics over 10 steps at D = 32, well inside the parity tolerance, and the iteration is the faster one."""
    runs = []
    for sub in (1, 0):
        t = T.Tatrg(0.1497, 0.0, 32, 32, 42)
        t.set_option(T.OPT_SUBSPACE, sub)
        out = []
        for _ in range(10):
            t.step()
            out.append((t.lnZ_per_site(), t.singular_values(T.SV_SIGMA, 32), t.singular_values(T.SV_S, 32), t.launches()))
        runs.append(out)
        t.close()
    for a, b in zip(*runs):
        assert abs(a[0] - b[0]) <= 1e-12 * abs(b[0])
        assert np.abs(a[1] - b[1]).max() <= 1e-10 and np.abs(a[2] - b[2]).max() <= 1e-10
    assert runs[0][-1][3] < runs[1][-1][3]


# ---- pins that need no oracle run: exact values the mathematics fixes ------------------------------------------------------
@pytest.mark.parametrize("beta,h", [(0.14, 0.0), (0.1497, 1e-3), (0.3, -0.2)])
def test_one_step_is_exact_closed_form(beta, h):
    """Lattice 2x1x1x1 (periodic): Z = e^{6 beta} [2 e^{2 beta} cosh(2 beta h) + 2 e^{-2 beta}]; nothing is truncated at D>=4."""
    t = T.Tatrg(beta, h, 4, 4, 1)
    t.step()
    z = math.exp(6 * beta) * (2 * math.exp(2 * beta) * math.cosh(2 * beta * h) + 2 * math.exp(-2 * beta))
    assert abs(t.lnZ_per_site() - math.log(z) / 2) <= 1e-13


def test_low_temperature_limit():
    """beta = 2, 16 steps: ln Z/V - 4 beta = ln 2 / 2^16 (two ordered ground states); the spectrum collapses to rank 2 then 1."""
    t = T.Tatrg(2.0, 0.0, 4, 4, 3, power_iters=1)
    for _ in range(16):
        t.step()
    assert abs(t.lnZ_per_site() - 8.0 - math.log(2) / 2 ** 16) <= 1e-11


def test_high_temperature_limit():
    t = T.Tatrg(1e-3, 0.0, 4, 4, 3, power_iters=1)
    for _ in range(12):
        t.step()
    b = 1e-3
    assert abs(t.lnZ_per_site() - math.log(2) - 4 * math.log(math.cosh(b))) <= 1e-10


# ---- oracle run inside the test: small and edge configurations ----------------------------------------------------------------
@pytest.mark.parametrize("beta,h,D,p,n_pow,seed,steps", [
    (0.1497, 0.0, 2, 0, 0, 5, 8),        # minimal D, no oversampling, no power iteration
    (0.1497, 0.0, 3, 2, 1, 6, 8),        # odd D: ragged everywhere
    (0.16, 5e-2, 5, 3, 2, 7, 10),        # ordered phase with field
    (0.12, 0.0, 6, 6, 3, 8, 8),
    (0.1497, 0.0, 4, 4, 1, 2 ** 40 + 17, 6),   # 64-bit seed
])
def test_small_runs_against_live_oracle(beta, h, D, p, n_pow, seed, steps):
    from oracle import tatrg_oracle as O
    t = T.Tatrg(beta, h, D, p, seed, power_iters=n_pow)
    o = O.TatrgOracle(beta, h, D, p, seed, n_pow=n_pow)
    for m in range(steps):
        t.step()
        o.step()
        lo = o.lnZ_per_site()
        assert abs(t.lnZ_per_site() - lo) <= TOL_LNZ * abs(lo), m
        for which, key in ((T.SV_SIGMA, "sigma"), (T.SV_S, "s")):
            got, ref = t.singular_values(which, D), o.last[key][:D]
            k = min(len(got), len(ref))
            assert np.abs(got[:k] - ref[:k]).max() <= TOL_SV, (m, key)
            assert np.all(np.abs(ref[k:]) <= TOL_SV) and np.all(np.abs(got[k:]) <= TOL_SV)


def test_k_triad_option_and_full_rank_equals_atrg():
    """K = chi2*chi3 (no triad truncation) and a smaller K both follow the oracle (PAPER.md :179 'r = D recovers ATRG')."""
    from oracle import tatrg_oracle as O
    for K in (16, 5):
        t = T.Tatrg(0.1497, 0.0, 4, 12, 9, power_iters=1, K=K)
        o = O.TatrgOracle(0.1497, 0.0, 4, 12, 9, n_pow=1, K=K)
        for m in range(6):
            t.step()
            o.step()
            assert abs(t.lnZ_per_site() - o.lnZ_per_site()) <= TOL_LNZ * abs(o.lnZ_per_site()), (K, m)


# ---- stage-wise, teacher-forced: the GPU step is fed the oracle's state; gauge-invariant stage outputs are compared ---------------
def _proj(x, nlast=1):
    m = x.reshape(-1, int(np.prod(x.shape[-nlast:])))
    return m @ m.T


@pytest.mark.parametrize("implicit", [1, 0])
@pytest.mark.parametrize("D,p,n_pow,presteps", [(4, 4, 1, 3), (6, 6, 2, 4)])
def test_stagewise_teacher_forced(D, p, n_pow, presteps, implicit):
    """implicit = 1 (default): the path takes the triad Gram matrices and F, G from U^bond, sigma, V^bond (:394); X and Y are formed for
    this inspection only.  implicit = 0: X, Y formed and used as Eq. 2.9-2.12 print them.  Both against the same oracle step."""
    from oracle import tatrg_oracle as O
    beta, h, seed = 0.1497, 0.0, 21
    o = O.TatrgOracle(beta, h, D, p, seed, n_pow=n_pow)
    t = T.Tatrg(beta, h, D, p, seed, power_iters=n_pow)
    t.set_option(T.OPT_KEEP_TENSORS, 1)
    t.set_option(T.OPT_IMPLICIT_XY, implicit)
    for _ in range(presteps):
        o.step()
        t.step()
    t.set_state(o.phi, o.psi)          # teacher forcing: identical inputs to the compared step
    o.step()
    t.step()
    L = o.last
    a, dt, core, x, y, sig = (t.get_tensor(n) for n in ("A", "Dt", "core", "X", "Y", "sigma"))
    tol = 1e-10
    # (a) canonical gauge makes A, Dt, core themselves comparable
    assert np.abs(a - L["a"]).max() <= tol and np.abs(dt - L["dt"]).max() <= tol and np.abs(core - L["core"]).max() <= tol
    am = a.reshape(-1, a.shape[-1])
    assert np.abs(am.T @ am - np.eye(a.shape[-1])).max() <= 1e-12          # isometry (:137)
    # (b) X sigma Y^T is gauge invariant; X, Y isometric
    assert np.abs(sig - L["sig"]).max() <= tol * L["sig"][0]
    rec_g = np.einsum("aig,g,bjg->aibj", x.reshape(x.shape[0], -1, x.shape[-1]), sig, y.reshape(y.shape[0], -1, y.shape[-1]))
    rec_o = np.einsum("aig,g,bjg->aibj", L["x"].reshape(x.shape[0], -1, x.shape[-1]), L["sig"], L["y"].reshape(y.shape[0], -1, y.shape[-1]))
    assert np.abs(rec_g - rec_o).max() <= tol * L["sig"][0]
    xm = x.reshape(-1, x.shape[-1])
    assert np.abs(xm.T @ xm - np.eye(x.shape[-1])).max() <= 1e-11
    # (c) triad isometries: projectors U U^T
    for name, uo in zip(("UA", "UX", "UY", "UD"), L["u"]):
        ug = t.get_tensor(name)                                            # [k, leg2, leg3]
        pg = ug.reshape(ug.shape[0], -1).T @ ug.reshape(ug.shape[0], -1)
        po = uo.reshape(-1, uo.shape[-1]) @ uo.reshape(-1, uo.shape[-1]).T
        assert ug.shape[0] == uo.shape[-1], name
        assert np.abs(pg - po).max() <= 1e-9, name
    # (c') triad tensors (Eq. 2.10-2.13): invariant under the basis of the kept subspace (internal line summed) and under the signs of
    #      the swapped bond gamma (summed as well for F, G; E, H carry only physical legs and the canonically gauged alpha / beta)
    eo, fo, go, ho = L["efgh"]
    for name, ref in (("F", fo), ("G", go), ("E", eo), ("H", ho)):
        got = t.get_tensor(name)
        assert got.shape == ref.shape, name
        spec = "axlg,bxmg->albm" if name in ("F", "G") else "axlg,bxmh->algbmh"
        gg, rr = np.einsum(spec, got, got), np.einsum(spec, ref, ref)
        assert np.abs(gg - rr).max() <= 1e-9 * np.abs(rr).max(), name
    # (d) squeezers: canonical gauge makes M, N comparable up to nothing
    for mu in (2, 3, 4):
        mg, ng = t.get_tensor("M%d" % mu), t.get_tensor("N%d" % mu)        # [k, u, l]
        mo, no = L["m"][mu], L["n"][mu]                                    # [u, l, k]
        assert mg.shape[0] == mo.shape[-1], mu
        pg = np.einsum("kul,kvw->ulvw", mg, ng)
        po = np.einsum("ulk,vwk->ulvw", mo, no)
        assert np.abs(pg - po).max() <= 1e-8 * max(1.0, np.abs(po).max()), mu
        assert np.abs(np.einsum("kul,jul->kj", mg, ng) - np.eye(mg.shape[0])).max() <= 1e-9    # N^T M = 1
    # (e,f) new state: T' = Phi' Psi'^T is gauge invariant
    phi, psi = t.get_tensor("phi"), t.get_tensor("psi")
    assert phi.shape == o.phi.shape
    tg = phi.reshape(-1, phi.shape[-1]) @ psi.reshape(-1, psi.shape[-1]).T
    to = o.phi.reshape(-1, o.phi.shape[-1]) @ o.psi.reshape(-1, o.psi.shape[-1]).T
    assert np.abs(tg - to).max() <= 1e-9 * np.abs(to).max()


# ---- full size (D = 32, the launch configuration bench.py times): properties and sampled outputs ----------------------------------
def test_d32_stage_properties_and_sampled_contraction():
    from oracle import tatrg_oracle as O
    D, p = 32, 32
    t = T.Tatrg(0.1497, 0.0, D, p, 42)
    t.set_option(T.OPT_KEEP_TENSORS, 1)
    for _ in range(6):
        t.step()
    assert t.workspace_peak() <= T.workspace_bytes(D, p)
    a, x, sig = t.get_tensor("A"), t.get_tensor("X"), t.get_tensor("sigma")
    assert a.shape == (32, 32, 32, 32, 32) and x.shape[:4] == (32, 32, 32, 32)
    for m in (a.reshape(-1, a.shape[-1]), x.reshape(-1, x.shape[-1])):
        assert np.abs(m.T @ m - np.eye(m.shape[1])).max() <= 1e-10       # isometries (:137)
    assert np.all(np.diff(sig) <= 0) and sig[-1] > 0
    ua = t.get_tensor("UA")
    um = ua.reshape(ua.shape[0], -1)
    assert np.abs(um @ um.T - np.eye(um.shape[0])).max() <= 1e-10
    for mu in (2, 3, 4):
        mg, ng = t.get_tensor("M%d" % mu), t.get_tensor("N%d" % mu)
        assert np.abs(np.einsum("kul,jul->kj", mg, ng) - np.eye(mg.shape[0])).max() <= 1e-8
    # sampled outputs of the O(r^2 D^7) contraction (Eq. 2.18 :175), recomputed one slab at a time with the oracle's
    # contract_half from the GPU's own E, F, I, J, M (teacher-forced stage parity at full size)
    e, f = t.get_tensor("E"), t.get_tensor("F")
    ux = t.get_tensor("UX")
    m2, m3, m4 = (t.get_tensor("M%d" % mu) for mu in (2, 3, 4))
    phi = t.get_tensor("phi")                                              # [k2,k3,k4,i1,g]
    tr = lambda m: np.ascontiguousarray(m.transpose(1, 2, 0))             # [k,u,l] -> oracle's [u,l,k]
    tu = lambda u: np.ascontiguousarray(u.transpose(1, 2, 0))             # [k,j,k'] -> oracle's [j,k',k]
    rng = np.random.default_rng(0)
    for _ in range(2):
        i1 = int(rng.integers(0, e.shape[0]))
        slab = O.contract_half(e[i1:i1 + 1], f, tu(ua), tu(ux), tr(m2), tr(m3), tr(m4))[0]     # [k2,k3,k4,g]
        got = phi[:, :, :, i1, :]
        assert np.abs(got - slab).max() <= 1e-11 * max(1.0, np.abs(slab).max())


def test_config5_d48_against_the_oracle():
    """BASELINE.json configs[4], Triad half (D=48, p=48, K=96, seed 99): the largest size; n = 2304 eigen-problems.
    (i) the first steps against the oracle's golden run (tests/golden/oracle_c5.json: the unsaturated steps, which the oracle
    affords); (ii) at step 6 (saturated: a whole oracle step would take hours) the O(r^2 D^7) contraction of Eq. 2.18-2.19 :175
    recomputed slab by slab with the oracle's contract_half / contract_psi from the GPU's own triad tensors and squeezers
    (teacher-forced stage parity at full size), isometries, N^T M = 1; (iii) ln Z/V above the D=32 value after the same number of
    steps (the free energy decreases monotonically with D, Fig. 9 :286-288)."""
    from oracle import tatrg_oracle as O
    path = os.path.join(HERE, "golden", "oracle_c5.json")
    rec = json.load(open(path))["runs"][0] if os.path.exists(path) else None
    t48 = T.Tatrg(0.1497, 0.0, 48, 48, 99)
    t32 = T.Tatrg(0.1497, 0.0, 32, 32, 99)
    for m in range(6):
        if m == 5:
            t48.set_option(T.OPT_KEEP_TENSORS, 1)
        t48.step()
        t32.step()
        if rec is not None and m < len(rec["lnZ"]):
            assert abs(t48.lnZ_per_site() - rec["lnZ"][m]) <= TOL_LNZ * abs(rec["lnZ"][m]), m
            for which, key in ((T.SV_SIGMA, "sigma"), (T.SV_S, "s")):
                got, ref = np.zeros(48), np.zeros(48)
                g = t48.singular_values(which, 48)
                got[:len(g)] = g
                ref[:len(rec[key][m])] = rec[key][m]
                assert np.abs(got - ref).max() <= TOL_SV, (m, key)
    assert t48.workspace_peak() <= T.workspace_bytes(48, 48)
    a = t48.get_tensor("A")
    assert a.shape == (48, 48, 48, 48, 48)
    am = a.reshape(-1, 48)
    assert np.abs(am.T @ am - np.eye(48)).max() <= 1e-10
    del a, am
    sig = t48.singular_values(T.SV_SIGMA, 48)
    assert len(sig) == 48 and np.all(np.diff(sig) <= 0) and sig[-1] > 0
    z48, z32 = t48.lnZ_per_site(), t32.lnZ_per_site()
    assert np.isfinite(z48) and z48 > z32 and z48 - z32 < 5e-3
    t32.close()
    tr = lambda m: np.ascontiguousarray(m.transpose(1, 2, 0))             # [k,u,l] -> oracle's [u,l,k]; [k,j,k'] -> [j,k',k]
    for mu in (2, 3, 4):
        mg, ng = t48.get_tensor("M%d" % mu), t48.get_tensor("N%d" % mu)
        assert np.abs(np.einsum("kul,jul->kj", mg, ng) - np.eye(mg.shape[0])).max() <= 1e-8
    e, f, g, h = (t48.get_tensor(n) for n in "EFGH")
    ua, ux, uy, ud = (tr(t48.get_tensor(n)) for n in ("UA", "UX", "UY", "UD"))
    ms = [tr(t48.get_tensor("M%d" % mu)) for mu in (2, 3, 4)]
    ns = [tr(t48.get_tensor("N%d" % mu)) for mu in (2, 3, 4)]
    assert e.shape == (48, 96, 48, 48) and ua.shape == (48, 48, 96)
    rng = np.random.default_rng(1)
    phi = t48.get_tensor("phi")                                            # [k2,k3,k4,i1,g]
    i1 = int(rng.integers(0, 48))
    slab = O.contract_half(e[i1:i1 + 1], f, ua, ux, *ms)[0]                # [k2,k3,k4,g]
    assert np.abs(phi[:, :, :, i1, :] - slab).max() <= 1e-11 * max(1.0, np.abs(slab).max())
    del phi
    psi = t48.get_tensor("psi")
    j1 = int(rng.integers(0, 48))
    slab = O.contract_psi(g, h[j1:j1 + 1], uy, ud, *ns)[0]
    assert np.abs(psi[:, :, :, j1, :] - slab).max() <= 1e-11 * max(1.0, np.abs(slab).max())
    t48.close()


def test_config5_plain_atrg_d24_sliced_contraction_against_the_oracle():
    """BASELINE.json configs[4], plain-ATRG half (D=24, p=24, seed 99; Eq. 2.7-2.8 :106-109).  The library never stores
    the D^7 intermediate (fn 6 :205 "memory blocking"): it slices the O(D^9) contraction over the outer leg.  At a saturated step
    (a whole oracle step is out of reach) 24 fibres of Phi' and 24 of Psi' are recomputed with the oracle's contract_atrg -- ONE
    einsum, the definition -- from the GPU's own A, X sigma, Y, D and squeezers; plus the first steps against the golden run when
    tests/golden/oracle_c5a.json exists."""
    from oracle import tatrg_oracle as O
    path = os.path.join(HERE, "golden", "oracle_c5a.json")
    rec = json.load(open(path))["runs"][0] if os.path.exists(path) else None
    D = 24
    t = T.Tatrg(0.1497, 0.0, D, D, 99, method=T.METHOD_ATRG)
    for m in range(6):
        if m == 5:
            t.set_option(T.OPT_KEEP_TENSORS, 1)
        t.step()
        if rec is not None and m < len(rec["lnZ"]):
            assert abs(t.lnZ_per_site() - rec["lnZ"][m]) <= TOL_LNZ * abs(rec["lnZ"][m]), m
            got, ref = np.zeros(D), np.zeros(D)
            g = t.singular_values(T.SV_SIGMA, D)
            got[:len(g)] = g
            ref[:len(rec["sigma"][m])] = rec["sigma"][m]
            assert np.abs(got - ref).max() <= TOL_SV, m
    a, x, y, dt, sig = (t.get_tensor(n) for n in ("A", "X", "Y", "Dt", "sigma"))
    assert a.shape == (D,) * 5 and x.shape[:4] == (D,) * 4
    tr = lambda m: np.ascontiguousarray(m.transpose(1, 2, 0))             # [k,u,l] -> oracle's [u,l,k]
    ms = [tr(t.get_tensor("M%d" % mu)) for mu in (2, 3, 4)]
    ns = [tr(t.get_tensor("N%d" % mu)) for mu in (2, 3, 4)]
    xs = x * sig
    phi = t.get_tensor("phi")                                              # [k2,k3,k4,i1,g]
    rng = np.random.default_rng(2)
    # sampled outputs, one fibre (all k4 at fixed i1, k2, k3, g) at a time: with every free leg but one cut to a single value
    # the oracle's one-einsum definition costs O(D^5) per fibre (a whole slab of it would take hours: its einsum path degenerates)
    scale = np.abs(phi).max()
    for _ in range(24):
        i1, k2, k3, gg = (int(v) for v in rng.integers(0, D, size=4))
        fib = O.contract_atrg(a[i1:i1 + 1], xs[..., gg:gg + 1], ms[0][:, :, k2:k2 + 1], ms[1][:, :, k3:k3 + 1], ms[2])[0, 0, 0, :, 0]   # Eq. 2.7
        assert np.abs(phi[k2, k3, :, i1, gg] - fib).max() <= 1e-11 * scale
    # Eq. 2.8: the lower half is Y[be,u2,u3,u4,g] (upper site) . D[j1,l2,l3,l4,be] (lower site) with the squeezers N
    yp = np.ascontiguousarray(y.transpose(4, 1, 2, 3, 0))                 # [g,u2,u3,u4,be]
    dp = np.ascontiguousarray(dt.transpose(4, 1, 2, 3, 0))                # [be,l2,l3,l4,j1]
    psi = t.get_tensor("psi")                                              # [k2,k3,k4,j1,g]
    scale = np.abs(psi).max()
    for _ in range(24):
        j1, k2, k3, gg = (int(v) for v in rng.integers(0, D, size=4))
        fib = O.contract_atrg(yp[gg:gg + 1], dp[..., j1:j1 + 1], ns[0][:, :, k2:k2 + 1], ns[1][:, :, k3:k3 + 1], ns[2])[0, 0, 0, :, 0]
        assert np.abs(psi[k2, k3, :, j1, gg] - fib).max() <= 1e-11 * scale
    t.close()


def test_x_ratio_matches_oracle_and_closed_form():
    """Eq. 3.3 :298-303.  Initial tensor: X = e^{2 beta} / cosh 2 beta; then step by step against the oracle."""
    from oracle import tatrg_oracle as O
    beta = 0.1497
    t = T.Tatrg(beta, 0.0, 6, 6, 5, power_iters=2)
    o = O.TatrgOracle(beta, 0.0, 6, 6, 5, n_pow=2)
    assert abs(t.x_ratio() - math.exp(2 * beta) / math.cosh(2 * beta)) <= 1e-13
    for m in range(8):
        t.step()
        o.step()
        assert abs(t.x_ratio() - o.x_ratio()) <= 1e-9 * o.x_ratio(), m
    lo = T.Tatrg(1.0, 0.0, 4, 4, 3, power_iters=1)
    for _ in range(8):
        lo.step()
    assert abs(lo.x_ratio() - 2.0) <= 1e-6


@pytest.mark.parametrize("D,p,n_pow,steps", [(3, 3, 1, 8), (4, 4, 2, 10), (5, 3, 1, 6)])
def test_plain_atrg_method_matches_untriaded_oracle(D, p, n_pow, steps):
    """SURVEY A9 / PAPER.md Eq. 2.7-2.8 :104-113: the plain-ATRG path (no triad isometries, squeezers from Gamma^ATRG,
    sliced O(D^9) contraction) against the oracle's plain-ATRG method (one einsum per equation)."""
    from oracle import tatrg_oracle as O
    beta, seed = 0.1497, 31
    t = T.Tatrg(beta, 0.0, D, p, seed, power_iters=n_pow, method=T.METHOD_ATRG)
    o = O.TatrgOracle(beta, 0.0, D, p, seed, n_pow=n_pow, method="atrg")
    for m in range(steps):
        t.step()
        o.step()
        lo = o.lnZ_per_site()
        assert abs(t.lnZ_per_site() - lo) <= TOL_LNZ * abs(lo), m
        got, ref = t.singular_values(T.SV_SIGMA, D), o.last["sigma"][:D]
        k = min(len(got), len(ref))
        assert np.abs(got[:k] - ref[:k]).max() <= TOL_SV, m
    # and it differs from the truncated triad run (K = D + p < D^2 at D = 4), i.e. the option does something
    if D == 4:
        tt = T.Tatrg(beta, 0.0, D, 1, seed, power_iters=n_pow, K=5)
        ta = T.Tatrg(beta, 0.0, D, 1, seed, power_iters=n_pow, method=T.METHOD_ATRG)
        for _ in range(steps):
            tt.step()
            ta.step()
        assert abs(tt.lnZ_per_site() - ta.lnZ_per_site()) > 1e-8


@pytest.mark.parametrize("D,bond_rank,p,n_pow,steps", [(3, 6, 3, 2, 8), (4, 8, 4, 1, 8), (4, 12, 4, 2, 6), (6, 9, 6, 2, 6)])
def test_ilo_triad_atrg_matches_oracle(D, bond_rank, p, n_pow, steps):
    """SURVEY A10 / PAPER.md section 2.3 :183-209, App. A: ILO Triad-ATRG -- the bond swap keeps r_bond D values (Eq. A.1 :337), the
    next decomposition keeps the whole overspanned bond (fn 5 :203), the squeezed legs stay at D -- against the oracle run with
    the same bond_rank; and the state has the shape fn 5 states."""
    from oracle import tatrg_oracle as O
    beta, seed = 0.1497, 17
    t = T.Tatrg(beta, 0.0, D, p, seed, power_iters=n_pow, bond_rank=bond_rank)
    t.set_option(T.OPT_KEEP_TENSORS, 1)
    o = O.TatrgOracle(beta, 0.0, D, p, seed, n_pow=n_pow, bond_rank=bond_rank)
    for m in range(steps):
        t.step()
        o.step()
        lo = o.lnZ_per_site()
        assert abs(t.lnZ_per_site() - lo) <= TOL_LNZ * abs(lo), m
        for which, key in ((T.SV_SIGMA, "sigma"), (T.SV_S, "s")):
            got, ref = t.singular_values(which, bond_rank), o.last[key][:bond_rank]
            k = min(len(got), len(ref))
            assert np.abs(got[:k] - ref[:k]).max() <= TOL_SV, (m, key)
    assert t.get_tensor("phi").shape == o.phi.shape == (D, D, D, D, bond_rank)
    assert t.get_tensor("X").shape == (bond_rank, D, D, D, bond_rank)


@pytest.mark.parametrize("implicit", [1, 0])
@pytest.mark.parametrize("D,bond_rank,p,n_pow,steps", [(3, 6, 3, 2, 8), (4, 8, 4, 1, 8), (4, 12, 4, 2, 6), (6, 9, 6, 2, 6), (5, 5, 5, 2, 8)])
def test_ilo_without_x_y_matches_oracle(D, bond_rank, p, n_pow, steps, implicit):
    """SURVEY NEXT-2 as the paper states it (PAPER.md :394 "the tensors X and Y are not explicitly constructed. Instead, we work directly
    with U^bond, sigma, and V^*bond to create isometries of the triad representation", :201): TATRG_OPT_IMPLICIT_XY = 1 against the
    oracle's implicit route, = 0 against its explicit one (the two oracle routes are pinned to each other in test_oracle_pins.py).
    Without TATRG_OPT_KEEP_TENSORS no X, Y exist on the device in the implicit setting.  (5, 5) is r_bond = 1."""
    from oracle import tatrg_oracle as O
    beta, seed = 0.1497, 23
    t = T.Tatrg(beta, 0.0, D, p, seed, power_iters=n_pow, bond_rank=bond_rank)
    t.set_option(T.OPT_IMPLICIT_XY, implicit)
    o = O.TatrgOracle(beta, 0.0, D, p, seed, n_pow=n_pow, bond_rank=bond_rank, implicit_xy=bool(implicit))
    for m in range(steps):
        t.step()
        o.step()
        lo = o.lnZ_per_site()
        assert abs(t.lnZ_per_site() - lo) <= TOL_LNZ * abs(lo), m
        for which, key in ((T.SV_SIGMA, "sigma"), (T.SV_S, "s")):
            got, ref = t.singular_values(which, bond_rank), o.last[key][:bond_rank]
            k = min(len(got), len(ref))
            assert np.abs(got[:k] - ref[:k]).max() <= TOL_SV, (m, key)
    assert t.get_tensor("phi").shape == o.phi.shape == (D, D, D, D, bond_rank)
    with pytest.raises(Exception):
        t.get_tensor("X")                      # nothing kept: X was never formed (implicit) or not retained (explicit)


def test_ilo_without_x_y_at_d16_equals_the_explicit_route():
    """r_bond = 2 at D = 16, a size the oracle does not reach in seconds: the run without X, Y agrees with the run that forms them
    (rounding order only), both stay inside the workspace bound, and no X is left on the device."""
    D, p, rb = 16, 16, 32
    lnz, sig = {}, {}
    for implicit in (1, 0):
        t = T.Tatrg(0.1497, 0.0, D, p, 7, bond_rank=rb)
        t.set_option(T.OPT_IMPLICIT_XY, implicit)
        for _ in range(9):
            t.step()
        assert t.workspace_peak() <= T.lib().tatrg_workspace_bytes_ilo(D, p, rb)
        lnz[implicit], sig[implicit] = t.lnZ_per_site(), t.singular_values(T.SV_SIGMA, rb)
        with pytest.raises(Exception):
            t.get_tensor("X")
        t.close()
    assert abs(lnz[1] - lnz[0]) <= 1e-11 * abs(lnz[0])
    assert np.abs(sig[1] - sig[0]).max() <= 1e-10


def test_ilo_at_d16_runs_and_differs_from_plain():
    """r_bond = 2 at D = 16 (bond rank 32, sketch 48 wide): properties at a size the oracle cannot reach in seconds -- workspace
    bound, isometries, ordered spectrum of 32 values -- and a free energy that differs from (and, near T_c, lies above) r_bond = 1."""
    D, p = 16, 16
    ti = T.Tatrg(0.1497, 0.0, D, p, 7, bond_rank=32)
    ti.set_option(T.OPT_KEEP_TENSORS, 1)
    tp = T.Tatrg(0.1497, 0.0, D, p, 7)
    for _ in range(12):
        ti.step()
        tp.step()
    assert ti.workspace_peak() <= T.lib().tatrg_workspace_bytes_ilo(D, p, 32)
    x = ti.get_tensor("X")
    assert x.shape == (32, D, D, D, 32)
    xm = x.reshape(-1, 32)
    assert np.abs(xm.T @ xm - np.eye(32)).max() <= 1e-10
    sig = ti.singular_values(T.SV_SIGMA, 32)
    assert len(sig) == 32 and np.all(np.diff(sig) <= 0) and sig[-1] > 0
    zi, zp = ti.lnZ_per_site(), tp.lnZ_per_site()
    assert np.isfinite(zi) and 1e-7 < zi - zp < 5e-3


def test_converged_sketch_mode_is_independent_of_the_random_tensor():
    """SURVEY NEXT-4 / PAPER.md :258 (q = 20), fn 4 :189 (q = O(D)): with 19 power iterations the RSVD subspace has converged, the
    result follows the oracle and no longer depends on the random tensor (two Philox seeds agree far below the parity tolerance),
    whereas with the configs' 2 power iterations the seed moves ln Z/V at the 1e-6 level."""
    from oracle import tatrg_oracle as O
    beta, D, p = 0.1497, 8, 8
    runs = {}
    for seed in (1, 2):
        t = T.Tatrg(beta, 0.0, D, p, seed, power_iters=19)
        for _ in range(6):
            t.step()
        runs[seed] = t.lnZ_per_site()
    o = O.TatrgOracle(beta, 0.0, D, p, 1, n_pow=19)
    for _ in range(6):
        o.step()
    assert abs(runs[1] - o.lnZ_per_site()) <= TOL_LNZ * abs(o.lnZ_per_site())
    assert abs(runs[1] - runs[2]) <= 1e-10
    loose = []
    for seed in (1, 2):
        t = T.Tatrg(beta, 0.0, D, p, seed, power_iters=2)
        for _ in range(6):
            t.step()
        loose.append(t.lnZ_per_site())
    assert abs(loose[0] - loose[1]) > 1e-9


@pytest.mark.parametrize("D,beta,h,steps", [(24, 0.12, 0.0, 8), (16, 0.2, 0.0, 14), (16, 0.1497, 0.05, 14)])
def test_subspace_path_falls_back_on_rank_deficient_blocks(D, beta, h, steps):
    """Away from criticality and in the unsaturated first steps the Gram matrices have fewer significant directions than the
    iteration block (D = 24, beta = 0.12, step 4: rank 64 of a 96-wide block).  The Cholesky guard flags the dependent columns
    and the full decomposition takes over: the run completes and agrees with TATRG_OPT_SUBSPACE = 0 throughout."""
    runs = []
    for sub in (1, 0):
        t = T.Tatrg(beta, h, D, D, 11)
        t.set_option(T.OPT_SUBSPACE, sub)
        out = []
        for _ in range(steps):
            t.step()
            out.append(t.lnZ_per_site())
        runs.append(out)
        t.close()
    for a, b in zip(*runs):
        assert np.isfinite(a) and abs(a - b) <= 1e-11 * abs(b)


@pytest.mark.gpu
@pytest.mark.parametrize("D,steps", [(16, 10), (32, 8)])
def test_overlapped_schedule_equals_the_serial_one(D, steps):
    """Saturated steps run the squeezer chains on an auxiliary stream beside the Gram matrices and the Xi products of
    Eq. 2.18-2.19 (schedule).  TATRG_OPT_OVERLAP = 0 issues the same work on one stream, TATRG_OPT_GRAPHS = 0
    launches the iteration steps one by one instead of replaying a captured graph: the results are the same numbers (no arithmetic
    differs, only what runs beside what; the bound leaves room for nothing but that)."""
    runs = []
    for overlap, graphs in ((1, 1), (0, 1), (1, 0)):
        t = T.Tatrg(0.1497, 0.0, D, D, 5)
        t.set_option(T.OPT_OVERLAP, overlap)
        t.set_option(T.OPT_GRAPHS, graphs)
        out = []
        for _ in range(steps):
            t.step()
            out.append((t.lnZ_per_site(), t.singular_values(T.SV_SIGMA, D), t.singular_values(T.SV_S, D)))
        runs.append(out)
        t.close()
    for other in runs[1:]:
        for a, b in zip(runs[0], other):
            assert abs(a[0] - b[0]) <= 1e-13 * abs(b[0])
            assert np.abs(a[1] - b[1]).max() <= 1e-12 and np.abs(a[2] - b[2]).max() <= 1e-12


@pytest.mark.gpu
def test_post_critical_steps_at_d32_agree_with_full_decompositions():
    """configs[3] beyond criticality: around step 20 the flow leaves the critical surface, the local tensor becomes numerically
    rank-deficient (s_32 / s_1 ~ 1e-8) and the default path hands the QR pre-reduction, and often the triad isometries, to the
    rank-revealing full decompositions while the squeezers still run on the auxiliary stream (full_run).
    Through 28 steps the default path and TATRG_OPT_SUBSPACE = 0 (full decompositions everywhere, one stream) give the same physics."""
    runs = []
    for sub in (1, 0):
        t = T.Tatrg(0.1497, 0.0, 32, 32, 42)
        t.set_option(T.OPT_SUBSPACE, sub)
        out = []
        for _ in range(28):
            t.step()
            out.append((t.lnZ_per_site(), t.singular_values(T.SV_S, 32)))
        runs.append(out)
        t.close()
    assert min(len(a[1]) for a in runs[0][19:]) >= 1 and runs[0][-1][1][-1] < 1e-4       # the regime is reached: s_32 / s_1 has collapsed
    for a, b in zip(*runs):
        assert np.isfinite(a[0]) and abs(a[0] - b[0]) <= 1e-11 * abs(b[0])
        n = min(len(a[1]), len(b[1]))
        assert np.abs(a[1][:n] - b[1][:n]).max() <= 1e-8
