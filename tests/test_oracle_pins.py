"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path involved).

Each test names the passage (PAPER.md:<line>) or the closed form it checks.  A plausible mistake in the oracle
(dropped term, wrong sign or index, transposed operand) must fail at least one of these.
"""
import itertools
import math
import os

import numpy as np
import pytest

from oracle import philox
from oracle import tatrg_oracle as O
from tests import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------------------------------------ Philox
def _kat():
    rows = []
    for line in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")):
        line = line.split("#")[0].split()
        if len(line) == 10:
            rows.append([int(x, 16) for x in line])
    return rows


def test_philox_known_answers():
    """Random123 known-answer vectors for philox4x32-10 (tests/golden/philox4x32_10_kat.txt)."""
    rows = _kat()
    assert len(rows) == 3
    for r in rows:
        out = philox.philox4x32_10(r[0], r[1], r[2], r[3], r[4], r[5])
        assert [int(x) for x in out] == r[6:]


def test_gaussian_box_muller_by_hand():
    """Counter 0, key 0 -> x = 6627e8d5 e169c58d bc57ac4c 9b00dbd8; the uniforms and z recomputed with integers."""
    x0, x1, x2, x3 = 0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8
    u1 = ((x0 >> 6) * 2 ** 27 + (x1 >> 5) + 0.5) / 2 ** 53
    u2 = ((x2 >> 6) * 2 ** 27 + (x3 >> 5) + 0.5) / 2 ** 53
    z = math.sqrt(-2 * math.log(u1)) * math.cos(2 * math.pi * u2)
    got = philox.gaussians(0, 0, 0, 0, 1)[0]
    assert abs(got - z) < 4e-16
    assert 0 < u1 < 1 and 0 < u2 < 1


def test_gaussian_counter_layout_beyond_32_bits():
    """R11: counter = (e & 0xffffffff, e >> 32, call, stream), key = (seed lo, seed hi).  Random123's third known-answer
    vector has ctr = (243f6a88, 85a308d3, 13198a2e, 03707344), key = (a4093822, 299f31d0) -> d16cfe09 94fdcceb 5001e420
    24126ea1, i.e. element e = 0x85a308d3243f6a88 >= 2^32 of call 0x13198a2e, stream 0x03707344, seed 0x299f31d0a4093822.
    The Gaussian is recomputed by hand from the PUBLISHED integers (not from the oracle's generator)."""
    x0, x1, x2, x3 = 0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1
    u1 = ((x0 >> 6) * 2 ** 27 + (x1 >> 5) + 0.5) / 2 ** 53
    u2 = ((x2 >> 6) * 2 ** 27 + (x3 >> 5) + 0.5) / 2 ** 53
    z = math.sqrt(-2 * math.log(u1)) * math.cos(2 * math.pi * u2)
    e = (0x85A308D3 << 32) | 0x243F6A88
    got = philox.gaussians((0x299F31D0 << 32) | 0xA4093822, 0x13198A2E, 0x03707344, e, 1)[0]
    assert abs(got - z) < 4e-16 * max(1.0, abs(z))
    # consecutive elements across the 2^32 boundary: e = 2^32 - 1 -> ctr (ffffffff, 0), e = 2^32 -> ctr (0, 1)
    zz = philox.gaussians(42, 3, 0, 2 ** 32 - 1, 2)
    for j, (c0, c1) in enumerate([(0xFFFFFFFF, 0), (0, 1)]):
        y0, y1, y2, y3 = (int(v) for v in philox.philox4x32_10(c0, c1, 3, 0, 42, 0))
        v1 = ((y0 >> 6) * 2 ** 27 + (y1 >> 5) + 0.5) / 2 ** 53
        v2 = ((y2 >> 6) * 2 ** 27 + (y3 >> 5) + 0.5) / 2 ** 53
        assert abs(zz[j] - math.sqrt(-2 * math.log(v1)) * math.cos(2 * math.pi * v2)) < 4e-16 * max(1.0, abs(zz[j]))


def test_gaussian_moments():
    z = philox.gaussians(1234, 7, 0, 0, 2_000_000)
    assert abs(z.mean()) < 4 / math.sqrt(z.size)
    assert abs(z.var() - 1) < 6 * math.sqrt(2 / z.size)
    assert abs((z ** 4).mean() - 3) < 0.03
    # different call / stream / seed give different, uncorrelated streams
    z2 = philox.gaussians(1234, 8, 0, 0, 100000)
    assert abs(np.corrcoef(z[:100000], z2)[0, 1]) < 0.02


# ------------------------------------------------------------------------------------------------ Jacobi
def test_jacobi_eigh_closed_form_toeplitz():
    """tridiag(-1,2,-1) of order n has eigenvalues 2 - 2 cos(k pi/(n+1)) and sine eigenvectors."""
    n = 37
    t = 2 * np.eye(n) - np.eye(n, k=1) - np.eye(n, k=-1)
    lam, v = O.jacobi_eigh(t)
    exact = np.sort(2 - 2 * np.cos(np.arange(1, n + 1) * np.pi / (n + 1)))[::-1]
    assert np.abs(lam - exact).max() < 1e-13
    assert np.abs(v.T @ v - np.eye(n)).max() < 1e-13
    vec = np.sin(np.arange(1, n + 1) * n * np.pi / (n + 1))          # eigenvector of the largest eigenvalue
    vec /= np.linalg.norm(vec)
    assert abs(abs(vec @ v[:, 0]) - 1) < 1e-12


def test_jacobi_eigh_2x2_and_indefinite():
    lam, v = O.jacobi_eigh(np.array([[2.0, 1.0], [1.0, 2.0]]))
    assert np.allclose(lam, [3, 1], atol=1e-15)
    assert np.allclose(np.abs(v), 1 / math.sqrt(2), atol=1e-15)
    s = inputs.random_tensor((9, 9), 3)
    s = s + s.T
    lam, v = O.jacobi_eigh(s)
    assert np.abs((v * lam) @ v.T - s).max() < 1e-13
    assert np.all(np.diff(lam) <= 0)


def test_jacobi_eigh_rank_deficient_gram():
    g = inputs.random_psd(48, 5, 11)
    lam, v = O.jacobi_eigh(g)
    assert np.abs(lam[:5] - 0.6 ** np.arange(5)).max() < 1e-13
    assert np.abs(lam[5:]).max() < 1e-14
    assert np.abs((v * lam) @ v.T - g).max() < 1e-13


def test_jacobi_svd_known_spectrum_and_shapes():
    for (m, n) in [(40, 7), (7, 40), (16, 16), (5, 1), (1, 5)]:
        a = inputs.lowrank_plus_noise(m, n, min(m, n), 0.0, 5)
        u, s, v = O.jacobi_svd(a)
        r = min(m, n)
        assert np.abs(s - 0.7 ** np.arange(r)).max() < 1e-13
        assert np.abs((u * s) @ v.T - a).max() < 1e-13
        assert np.abs(u.T @ u - np.eye(r)).max() < 1e-12
        assert np.abs(v.T @ v - np.eye(r)).max() < 1e-12


def test_jacobi_svd_rank_deficient_and_graded():
    a = inputs.lowrank_plus_noise(60, 20, 4, 0.0, 2)
    u, s, v = O.jacobi_svd(a)
    assert np.abs(s[:4] - 0.7 ** np.arange(4)).max() < 1e-13 and s[4:].max() < 1e-14
    q, r = O.orth(a)
    assert q.shape == (60, 4) and np.abs(q @ r - a).max() < 1e-13 and np.abs(q.T @ q - np.eye(4)).max() < 1e-13
    d = np.diag(10.0 ** -np.arange(12))                               # strongly graded: 1 .. 1e-11
    u, s, v = O.jacobi_svd(inputs.random_tensor((30, 12), 4) @ d)
    ref = inputs.random_tensor((30, 12), 4) @ d
    assert np.abs((u * s) @ v.T - ref).max() < 1e-14


# ------------------------------------------------------------------------------------------------ rank / gauge
def test_select_rank_never_splits_a_multiplet():
    v = np.array([1.0, 0.5, 0.3, 0.3 * (1 - 1e-9), 0.3 * (1 - 2e-9), 0.1, 0.0])
    assert O.select_rank(v, 6, 1e-12) == 6          # nothing real is cut: keep all non-zero
    assert O.select_rank(v, 5, 1e-12) == 5
    assert O.select_rank(v, 4, 1e-12) == 2          # 0.3-triplet would be split -> dropped as a whole
    assert O.select_rank(v, 3, 1e-12) == 2
    assert O.select_rank(v, 2, 1e-12) == 2
    assert O.multiplets(v, 6) == [(0, 1), (1, 2), (2, 5), (5, 6)]
    assert O.select_rank(np.array([1.0, 1e-13, 0.0]), 3, 1e-12) == 1


def test_canonical_rotation_is_gauge_invariant():
    rng = np.random.default_rng(0)
    w, _ = np.linalg.qr(rng.standard_normal((50, 6)))
    groups = [(0, 1), (1, 4), (4, 5), (5, 6)]
    g0 = O.canonical_rotation(w, groups, 9, 3, 1)
    o = np.zeros((6, 6))
    o[0, 0] = -1
    o[1:4, 1:4], _ = np.linalg.qr(rng.standard_normal((3, 3)))
    o[4, 4], o[5, 5] = 1, -1
    g1 = O.canonical_rotation(w @ o, groups, 9, 3, 1)
    assert np.abs(w @ g0 - w @ o @ g1).max() < 1e-13
    assert np.abs(g0.T @ g0 - np.eye(6)).max() < 1e-13


# ------------------------------------------------------------------------------------------------ initial tensor
def test_w_matrix_is_sqrt_of_boltzmann_weight():
    """Eq. 3.2 :246: (W W^T)_{ab} = cosh b + s_a s_b sinh b = exp(beta s_a s_b)."""
    beta = 0.37
    w = O.w_matrix(beta)
    spin = np.array([1.0, -1.0])
    assert np.allclose(w @ w.T, np.exp(beta * np.outer(spin, spin)), atol=1e-15)


@pytest.mark.parametrize("h", [0.0, 1e-3, 0.4])
def test_init_tensor_spectrum_closed_form(h):
    """T0 = Phi0 Psi0^T (16x16) has two non-zero singular values; for h=0 they are 2cosh(4b), 2sinh(4b)
    (eigenvalues of [[e^{4b}, e^{-4b}],[e^{-4b}, e^{4b}]] dressed by e^{+-bh})."""
    beta = 0.14
    phi, psi = O.init_tensor(beta, h)
    t = phi.reshape(16, 2) @ psi.reshape(16, 2).T
    s = np.linalg.svd(t, compute_uv=False)
    # T0 = sum_a e^{bh s_a} w_a w_a^T, w_a = W[a]^{x4}; in the (non-orthogonal) basis {w_a} with Gram matrix
    # g_ab = (W W^T)_ab^4 = e^{4 b s_a s_b}, the non-zero spectrum of T0 is that of diag(e^{bh s}) g
    gm = np.array([[math.exp(4 * beta), math.exp(-4 * beta)], [math.exp(-4 * beta), math.exp(4 * beta)]])
    dm = np.diag([math.exp(beta * h), math.exp(-beta * h)])
    ev = np.sort(np.abs(np.linalg.eigvals(dm @ gm)))[::-1]
    # T0 is not symmetric for h != 0, but sqrt(d) g sqrt(d) is, with the same spectrum; singular values agree
    # with |eigenvalues| because T0 is similar to a symmetric matrix only for h = 0 -> compare h = 0 exactly
    if h == 0.0:
        assert np.allclose(s[:2], [2 * math.cosh(4 * beta), 2 * math.sinh(4 * beta)], atol=1e-14)
        assert abs(math.log(s[0]) - 0.842377876007976) < 1e-14          # BASELINE.md pin ln c0
        assert abs(s[1] / s[0] - math.tanh(0.56)) < 1e-14
        assert np.allclose(ev, s[:2], atol=1e-14)
    assert s[2:].max() < 1e-14
    # 1-site periodic lattice: tTr T0 = sum_a e^{bh s_a} e^{4b}
    ttr = np.einsum("ijkla,ijkla->", phi, psi)
    assert abs(ttr - math.exp(4 * beta) * 2 * math.cosh(beta * h)) < 1e-13


# ------------------------------------------------------------------------------------------------ enumeration
def enumerate_lnz_per_site(dims, beta, h):
    """Brute force ln Z / V of H = -sum_<ij> s_i s_j - h sum_i s_i on the periodic lattice `dims` (4 axes);
    an axis of length 2 has its two sites joined by two bonds, an axis of length 1 gives s_i s_i = 1."""
    sites = list(itertools.product(*[range(d) for d in dims]))
    idx = {s: k for k, s in enumerate(sites)}
    v = len(sites)
    conf = ((np.arange(2 ** v)[:, None] >> np.arange(v)) & 1) * 2.0 - 1.0       # all spin configurations
    energy = h * conf.sum(axis=1)
    for s in sites:
        for mu in range(4):
            nb = list(s)
            nb[mu] = (nb[mu] + 1) % dims[mu]
            energy = energy + conf[:, idx[s]] * conf[:, idx[tuple(nb)]]
    x = beta * energy
    return (x.max() + math.log(np.exp(x - x.max()).sum())) / v


def test_enumeration_matches_closed_forms():
    """The enumerator itself is pinned by the closed forms of SURVEY/BASELINE: Z(2x1x1x1) = 4 e^{6b} cosh 2b."""
    beta = 0.14
    assert abs(enumerate_lnz_per_site((2, 1, 1, 1), beta, 0.0) - math.log(4 * math.exp(6 * beta) * math.cosh(2 * beta)) / 2) < 1e-14
    assert abs(enumerate_lnz_per_site((2, 1, 1, 1), beta, 0.0) - 1.132496303952126) < 1e-14
    h = 1e-3
    z = math.exp(6 * beta) * (2 * math.exp(2 * beta) * math.cosh(2 * beta * h) + 2 * math.exp(-2 * beta))
    assert abs(enumerate_lnz_per_site((2, 1, 1, 1), beta, h) - math.log(z) / 2) < 1e-14
    assert abs(enumerate_lnz_per_site((2, 2, 2, 2), beta, 0.0) - 0.783166715793510) < 1e-13


@pytest.mark.parametrize("beta,h", [(0.14, 0.0), (0.14, 1e-3), (0.1497, 0.0), (0.5, 0.2)])
def test_one_step_is_exact(beta, h):
    """fn 1 :82,:111: Eq. 2.4 is exact when D > 2^d; ranks after one step (T0: 2, swap: 4, pairs: 4) fit D=4,
    so ln Z/V of the 2x1x1x1 lattice must equal brute-force enumeration."""
    for D, p in [(4, 4), (6, 2)]:
        o = O.TatrgOracle(beta, h, D, p, 1234, n_pow=1).step()
        assert abs(o.lnZ_per_site() - enumerate_lnz_per_site((2, 1, 1, 1), beta, h)) < 2e-14


@pytest.mark.parametrize("beta,h", [(0.14, 0.0), (0.14, 1e-3), (0.3, -0.1)])
def test_two_steps_are_exact_for_D16(beta, h):
    o = O.TatrgOracle(beta, h, 16, 16, 7, n_pow=2)
    o.step().step()
    assert abs(o.lnZ_per_site() - enumerate_lnz_per_site((2, 2, 1, 1), beta, h)) < 1e-13
    # no-truncation identity: spectrum of T^(2) as an f x b matrix == bond-swap spectrum of step 1
    o1 = O.TatrgOracle(beta, h, 16, 16, 7, n_pow=2).step()
    n = min(len(o.last["s"]), len(o1.last["sigma"]))
    assert n >= 4 and np.abs(o.last["s"][:4] - o1.last["sigma"][:4]).max() < 1e-13


def test_truncated_runs_approach_enumeration_with_D():
    """3 and 4 steps cannot be exact at feasible D (would need D=256); the truncation error against the exact
    2x2x2x1 / 2^4 enumeration must shrink as D grows (Fig. 9 trend :286-288) and stay small."""
    beta = 0.14
    ex3 = enumerate_lnz_per_site((2, 2, 2, 1), beta, 0.0)
    ex4 = enumerate_lnz_per_site((2, 2, 2, 2), beta, 0.0)
    err3, err4 = [], []
    for D in (4, 8, 12):
        o = O.TatrgOracle(beta, 0.0, D, D, 1, n_pow=2)
        o.step().step().step()
        err3.append(abs(o.lnZ_per_site() - ex3))
        o.step()
        err4.append(abs(o.lnZ_per_site() - ex4))
    assert err3[0] > err3[1] > err3[2] and err3[0] < 0.1
    assert err4[0] > err4[2] and err4[0] < 2e-2


def test_limits_beta_large_and_small():
    """beta -> infinity: ln Z/V = 4 beta + ln 2 / V exactly at finite V (two ground states);
    beta -> 0: ln Z/V = ln 2 + 4 ln cosh(beta) + O(beta^4)."""
    o = O.TatrgOracle(2.0, 0.0, 4, 4, 1234, n_pow=1)
    for _ in range(16):
        o.step()
    assert abs(o.lnZ_per_site() - 8.0 - math.log(2) / 2 ** 16) < 1e-12
    o = O.TatrgOracle(1e-3, 0.0, 4, 4, 1234, n_pow=1)
    for _ in range(16):
        o.step()
    assert abs(o.lnZ_per_site() - math.log(2) - 4 * math.log(math.cosh(1e-3))) < 1e-11


def test_high_temperature_series_band():
    """Thermodynamic value at beta = 0.14 from the high-T series ln2 + 4 ln cosh b + 6 t^4 + 76 t^6, t = tanh b."""
    beta = 0.14
    t = math.tanh(beta)
    series = math.log(2) + 4 * math.log(math.cosh(beta)) + 6 * t ** 4 + 76 * t ** 6
    lnz, _, _ = O.run(beta, 0.0, 4, 4, 1234, 16, n_pow=1)
    assert abs(lnz[-1] - series) < 3e-3 and lnz[-1] < series


# ------------------------------------------------------------------------------------------------ stages
def _state_after(n, D=4, p=4, beta=0.1497, h=0.0, seed=11, n_pow=1):
    o = O.TatrgOracle(beta, h, D, p, seed, n_pow=n_pow)
    for _ in range(n):
        o.step()
    return o


def test_decomposition_reconstructs_T_and_is_isometric():
    """Eq. 2.4 :76 with :137 'A ... D are all isometric': T/c_m = A c Dt^T up to the truncation at D."""
    o = _state_after(2, D=16, p=16)                      # still untruncated
    a, dt, core, s, lnc = O.decompose(o.phi, o.psi, 16, 11, 3)
    chi = a.shape[-1]
    am, dm = a.reshape(-1, chi), dt.reshape(-1, chi)
    assert np.abs(am.T @ am - np.eye(chi)).max() < 1e-12 and np.abs(dm.T @ dm - np.eye(chi)).max() < 1e-12
    t = o.phi.reshape(-1, o.phi.shape[-1]) @ o.psi.reshape(-1, o.psi.shape[-1]).T
    assert np.abs(am @ core @ dm.T * math.exp(lnc) - t).max() < 1e-12 * np.abs(t).max()
    assert abs(math.exp(lnc) - np.linalg.svd(t, compute_uv=False)[0]) < 1e-12


def test_bond_swap_exact_mode_is_the_definition():
    """Eq. 2.5 :90 / A.1 :335: sum_i1 B C = X sig Y when nothing is truncated; X, Y isometric (:93)."""
    o = _state_after(1, D=16, p=16)
    a, dt, core, s, _ = O.decompose(o.phi, o.psi, 16, 11, 2)
    x, y, sig, _ = O.bond_swap(a, dt, core, 64, 0, 0, 11, 2, exact=True)
    b = np.einsum("ijklc,ac->ijkla", dt, core)
    c = np.einsum("ijklc,cb->ijklb", a, core)
    lhs = np.einsum("ijkla,imnob->amnobjkl", b, c)
    rhs = np.einsum("amnog,g,bjklg->amnobjkl", x, sig, y)
    assert np.abs(lhs - rhs).max() < 1e-13
    g = x.shape[-1]
    xm, ym = x.reshape(-1, g), y.reshape(-1, g)
    assert np.abs(xm.T @ xm - np.eye(g)).max() < 1e-12 and np.abs(ym.T @ ym - np.eye(g)).max() < 1e-12


def test_rsvd_converges_to_exact_swap():
    """App. A :350-379: with many passes (paper: q = 20, :258) the RSVD result equals the truncated SVD."""
    o = _state_after(3, D=4, p=4)
    a, dt, core, s, _ = O.decompose(o.phi, o.psi, 4, 11, 4)
    _, _, sig_ex, all_ex = O.bond_swap(a, dt, core, 4, 4, 0, 11, 4, exact=True)
    _, _, sig_20, _ = O.bond_swap(a, dt, core, 4, 4, 19, 11, 4)
    _, _, sig_1, _ = O.bond_swap(a, dt, core, 4, 4, 1, 11, 4)
    assert np.abs(sig_20 - sig_ex).max() < 1e-10
    assert np.abs(sig_1 - sig_ex).max() < 5e-2 and np.all(sig_1 <= sig_ex + 1e-12)     # Ritz values from below


def test_rsvd_on_random_lowrank_matrix_vs_full_svd():
    """The same loop (A.4-A.6) written for a plain matrix, against the full Jacobi SVD (north_star pin)."""
    s_mat = inputs.lowrank_plus_noise(60, 45, 12, 1e-9, 3)
    omega = philox.gaussians(5, 1, 0, 0, 45 * 16).reshape(45, 16)
    for _ in range(4):
        q, _ = O.orth(s_mat @ omega)
        yt = s_mat.T @ q
        omega, _ = O.orth(yt)
    _, sig, _ = O.jacobi_svd(yt)
    _, ref, _ = O.jacobi_svd(s_mat)
    assert np.abs(sig[:12] - ref[:12]).max() < 1e-10


def test_triad_full_rank_equals_untriaded_contraction():
    """':179 when r = D is chosen ... recovers ATRG': with K = chi2*chi3 the isometries are square orthogonal
    matrices and Eq. 2.18 must equal the direct contraction A X sig M2 M3 M4 (Eq. 2.7 form)."""
    o = _state_after(2, D=4, p=4)
    a, dt, core, s, _ = O.decompose(o.phi, o.psi, 4, 11, 3)
    x, y, sig, _ = O.bond_swap(a, dt, core, 4, 4, 1, 11, 3)
    (ua, ux, uy, ud), _ = O.triad_isometries(a, dt, x, y, sig, 16)
    # pad to square if the Gram matrices are rank deficient: use a complete orthonormal basis
    for u in (ua, ux, uy, ud):
        assert u.shape[-1] <= 16
    e, f, g, h = O.triad_tensors(a, dt, x, y, sig, ua, ux, uy, ud)
    rng = np.random.default_rng(0)
    m2, m3, m4 = (rng.standard_normal((a.shape[mu], x.shape[mu], 3)) for mu in (1, 2, 3))
    phi_triad = O.contract_half(e, f, ua, ux, m2, m3, m4)
    # projectors U U^T act as identity on A and X only if they span the range: check through the Gram spectra
    pa = np.einsum("jkm,nom->jkno", ua, ua)
    px = np.einsum("jkm,nom->jkno", ux, ux)
    a_p = np.einsum("ijkla,jkno->inola", a, pa)
    x_p = np.einsum("ajklg,jkno->anolg", x, px)
    direct = np.einsum("iuvwa,axyzg,g,uxb,vyc,wzd->ibcdg", a_p, x_p, sig, m2, m3, m4, optimize=True)
    assert np.abs(phi_triad - direct).max() < 1e-12 * np.abs(direct).max()
    psi_triad = O.contract_psi(g, h, uy, ud, m2, m3, m4)
    py = np.einsum("jkm,nom->jkno", uy, uy)
    pd = np.einsum("jkm,nom->jkno", ud, ud)
    y_p = np.einsum("bjklg,jkno->bnolg", y, py)
    d_p = np.einsum("ijklb,jkno->inolb", dt, pd)
    direct = np.einsum("buvwg,jxyzb,uxc,vyd,wze->jcdeg", y_p, d_p, m2, m3, m4, optimize=True)
    assert np.abs(psi_triad - direct).max() < 1e-12 * np.abs(direct).max()


def test_triad_isometries_are_top_eigenvectors_of_the_definition():
    """Eq. 2.9 :135: U^A spans the dominant eigenspace of the Gram matrix of Gamma^ATRG = A X sig Y D on the
    legs (i2,i3) of the upper site, computed here from the FULL Gamma (no canonical-form shortcut)."""
    o = _state_after(2, D=3, p=3)
    a, dt, core, s, _ = O.decompose(o.phi, o.psi, 3, 11, 3)
    x, y, sig, _ = O.bond_swap(a, dt, core, 3, 3, 1, 11, 3)
    (ua, ux, uy, ud), spec = O.triad_isometries(a, dt, x, y, sig, 4)
    half_u = np.einsum("ijkla,amnog,g->ijklmnog", a, x, sig)           # upper half of Gamma (f_u, i'_l, g)
    half_l = np.einsum("bjklg,imnob->gjklimno", y, dt)                  # lower half (g, j'_u, b_l)
    d2, d3 = a.shape[1], a.shape[2]
    gram_a = np.einsum("ijklmnog,iuvlmnoh,gpqrstwx,hpqrstwx->jkuv", half_u, half_u, half_l, half_l, optimize=True)
    lam = np.linalg.eigvalsh(gram_a.reshape(d2 * d3, -1))[::-1]
    assert np.abs(lam - spec[0]).max() < 1e-12 * lam[0]
    k = ua.shape[-1]
    um = ua.reshape(d2 * d3, k)
    assert np.abs(um.T @ um - np.eye(k)).max() < 1e-12
    resid = gram_a.reshape(d2 * d3, -1) @ um - um * lam[:k]
    assert np.abs(resid).max() < 1e-10 * lam[0]
    gram_y = np.einsum("ijklmnog,ijklmnoh,gpqrstwx,huvrstwx->pquv", half_u, half_u, half_l, half_l, optimize=True)
    lam_y = np.linalg.eigvalsh(gram_y.reshape(d2 * d3, -1))[::-1]
    assert np.abs(lam_y - spec[2]).max() < 1e-12 * lam_y[0]
    # ":137 the other isometries ... in the same manner": U^X on the legs (i2,i3) of X (= forward legs of the lower site),
    # U^D on the legs (j2,j3) of D (backward legs of the lower site); each eigenvector set checked against the full Gamma
    gram_x = np.einsum("ijklmnog,ijkluvoh,gpqrstwx,hpqrstwx->mnuv", half_u, half_u, half_l, half_l, optimize=True)
    gram_d = np.einsum("ijklmnog,ijklmnoh,gpqrstwx,hpqrsuvx->twuv", half_u, half_u, half_l, half_l, optimize=True)
    for gram, iso, sp in ((gram_x, ux, spec[1]), (gram_y, uy, spec[2]), (gram_d, ud, spec[3])):
        gm = gram.reshape(d2 * d3, -1)
        lam_i = np.linalg.eigvalsh(gm)[::-1]
        assert np.abs(lam_i - sp).max() < 1e-12 * lam_i[0]
        ki = iso.shape[-1]
        im = iso.reshape(d2 * d3, ki)
        assert np.abs(im.T @ im - np.eye(ki)).max() < 1e-12
        assert np.abs(gm @ im - im * lam_i[:ki]).max() < 1e-10 * lam_i[0]
    # the four Gram matrices are genuinely different objects (a swapped pair would fail the lines above)
    assert abs(spec[0][1] / spec[0][0] - spec[1][1] / spec[1][0]) > 1e-6 or abs(spec[2][1] / spec[2][0] - spec[3][1] / spec[3][0]) > 1e-6


def test_squeezer_grams_staged_equals_direct():
    """R6: the staged Gram matrices equal the direct contraction of the half unit cell with itself."""
    rng = np.random.default_rng(5)
    e = rng.standard_normal((2, 3, 2, 3))        # E[i1,kA,i4u,al]
    f = rng.standard_normal((3, 4, 3, 2))        # F[al,kX,i4l,g]
    i_, _ = np.linalg.qr(rng.standard_normal((6, 3)))
    j_, _ = np.linalg.qr(rng.standard_normal((6, 4)))
    i_, j_ = i_.reshape(2, 3, 3), j_.reshape(3, 2, 4)
    half = np.einsum("ikua,axlg,bck,dex->ibdceulg", e, f, i_, j_)      # [i1,i2u,i2l,i3u,i3l,i4u,i4l,g]
    d2 = np.einsum("ibdceulg,iBDceulg->bdBD", half, half)
    d3 = np.einsum("ibdceulg,ibdCEulg->ceCE", half, half)
    d4 = np.einsum("ibdceulg,ibdceULg->ulUL", half, half)
    assert np.abs(O.squeezer_grams(e, f, i_, j_, 2) - d2).max() < 1e-12
    assert np.abs(O.squeezer_grams(e, f, i_, j_, 3) - d3).max() < 1e-12
    assert np.abs(O.squeezer_grams(e, f, i_, j_, 4) - d4).max() < 1e-12
    # lower half: Gs[be,kY,j4u,g], H[j1,kD,j4l,be], K[j2u,j3u,kY], L[j2l,j3l,kD]
    gs = rng.standard_normal((3, 3, 2, 2))
    h = rng.standard_normal((2, 4, 3, 3))
    half = np.einsum("byug,jdlb,acy,etd->gjaecTul".replace("T", "t"), gs, h, i_, j_)
    d2 = np.einsum("gjaectul,gjAEctul->aeAE", half, half)
    d3 = np.einsum("gjaectul,gjaeCTul->ctCT", half, half)
    d4 = np.einsum("gjaectul,gjaectUL->ulUL", half, half)
    assert np.abs(O.squeezer_grams_lower(gs, h, i_, j_, 2) - d2).max() < 1e-12
    assert np.abs(O.squeezer_grams_lower(gs, h, i_, j_, 3) - d3).max() < 1e-12
    assert np.abs(O.squeezer_grams_lower(gs, h, i_, j_, 4) - d4).max() < 1e-12


def test_squeezer_pair_is_the_optimal_oblique_projector():
    """R6 / :113: N^T M = 1 and G1 M N^T G2 is the best rank-k approximation of G1 G2 (Eckart-Young)."""
    rng = np.random.default_rng(8)
    g1 = inputs.lowrank_plus_noise(30, 12, 12, 0.0, 1)
    g2 = inputs.lowrank_plus_noise(12, 25, 12, 0.0, 2)
    th_f = (g1.T @ g1).reshape(3, 4, 3, 4)
    th_b = (g2 @ g2.T).reshape(3, 4, 3, 4)
    m, n, s = O.squeezer_pair(th_f, th_b, 5, 1, 1, 2)
    k = m.shape[-1]
    mm, nn = m.reshape(12, k), n.reshape(12, k)
    assert k == 5 and np.abs(nn.T @ mm - np.eye(k)).max() < 1e-11
    sv = np.linalg.svd(g1 @ g2, compute_uv=False)
    err = np.linalg.norm(g1 @ g2 - g1 @ mm @ nn.T @ g2)
    assert abs(err - math.sqrt((sv[k:] ** 2).sum())) < 1e-10 * sv[0]
    assert np.abs(s[:k] * sv[0] - sv[:k]).max() < 1e-12 * sv[0]


def _unit_cell_halves(last):
    """Upper half  U[i1, i2u,i2l, i3u,i3l, i4u,i4l, g] = sum E F I J  (F carries sigma, Eq. 2.11 :151) and lower half
    L[g, j1, j2u,j2l, j3u,j3l, j4u,j4l] = sum G H K L (Eq. 2.12-2.13, 2.16-2.17) of Gamma^Triad, written out in full."""
    e, f, g, h = last["efgh"]
    ua, ux, uy, ud = last["u"]
    up = np.einsum("ikua,axlg,bck,dex->ibdceulg", e, f, ua, ux)
    lo = np.einsum("byug,jdlb,acy,etd->gjaectul", g, h, uy, ud)
    return up, lo


@pytest.mark.parametrize("D,p,h,steps", [(2, 2, 0.0, 4), (3, 2, 0.05, 4), (3, 3, 0.0, 5)])
def test_step_wires_the_squeezers_as_the_optimal_projectors_between_adjacent_cells(D, p, h, steps):
    """:113 'squeezers ... achieving the lower bound of the Frobenius norm with the adjacent unit cell', :171 'derived from
    Gamma^Triad' (reading R6), in the TRUNCATED regime (k = D < rank).  With G1 = upper half of the cell as a matrix
    [rest, forward pair alpha] and G2 = sigma-weighted lower half of the neighbouring cell [backward pair alpha, rest], the pair
    (M, N) that TatrgOracle.step() returns for direction alpha must reach the Eckart-Young bound
    ||G1 G2 - G1 M N^T G2||_F^2 = sum_{i>k} s_i(G1 G2)^2, and a mis-wired step (M <-> N, sigma weight dropped, the
    (upper, lower) legs of the doubled bond transposed) must not."""
    o = O.TatrgOracle(0.1497, h, D, p, 5, n_pow=2)
    for _ in range(steps):
        o.step()
    last = o.last
    up, lo = _unit_cell_halves(last)
    los = lo * last["sig"][:, None, None, None, None, None, None, None]
    for mu in (2, 3, 4):
        au, al = 2 * mu - 3, 2 * mu - 2                       # axes of the forward pair in `up`
        g1 = np.moveaxis(up, (au, al), (-2, -1))
        du, dl = g1.shape[-2:]
        g1 = g1.reshape(-1, du * dl)
        lo_t = np.moveaxis(lo, (au + 1, al + 1), (0, 1)).reshape(du * dl, -1)
        g2 = np.moveaxis(los, (au + 1, al + 1), (0, 1)).reshape(du * dl, -1)
        m, n = last["m"][mu], last["n"][mu]
        k = m.shape[-1]
        mm, nn = m.reshape(du * dl, k), n.reshape(du * dl, k)
        assert np.abs(nn.T @ mm - np.eye(k)).max() < 1e-10
        sv = np.linalg.svd(g1 @ g2, compute_uv=False)
        assert k <= D and sv[k] > 1e-4 * sv[0]               # something IS discarded: the truncated regime
        best = (sv[k:] ** 2).sum()
        err = lambda a, b, rhs: np.linalg.norm(g1 @ rhs - g1 @ a @ b.T @ rhs) ** 2
        assert abs(err(mm, nn, g2) - best) < 1e-9 * sv[0] ** 2
        assert np.abs(last["squeezer_spectra"][mu][:k] * sv[0] - sv[:k]).max() < 1e-10 * sv[0]
        # mis-wirings
        assert err(nn, mm, g2) > best * (1 + 1e-3)                                   # M <-> N
        mt = m.transpose(1, 0, 2).reshape(du * dl, k)
        nt = n.transpose(1, 0, 2).reshape(du * dl, k)
        assert err(mt, nt, g2) > best * (1 + 1e-3)                                   # (upper, lower) transposed
        sv_t = np.linalg.svd(g1 @ lo_t, compute_uv=False)
        assert err(mm, nn, lo_t) > (sv_t[k:] ** 2).sum() * (1 + 1e-3)                # sigma weight dropped: not optimal there
    # M goes to Phi' (Eq. 2.18 :175), N to Psi' (Eq. 2.19), sigma enters once (through F); then the rotation R5
    m2, m3, m4 = (last["m"][mu] for mu in (2, 3, 4))
    n2, n3, n4 = (last["n"][mu] for mu in (2, 3, 4))
    phi_new = np.einsum("ibdceulg,bdx,cey,ulz->ixyzg", up, m2, m3, m4, optimize=True)
    psi_new = np.einsum("gjaectul,aex,cty,ulz->jxyzg", lo, n2, n3, n4, optimize=True)
    assert np.abs(o.phi - phi_new.transpose(1, 2, 3, 0, 4)).max() < 1e-12 * np.abs(phi_new).max()
    assert np.abs(o.psi - psi_new.transpose(1, 2, 3, 0, 4)).max() < 1e-12 * np.abs(psi_new).max()


@pytest.mark.parametrize("D,p", [(2, 2), (3, 6)])
def test_squeezer_grams_are_the_grams_of_the_whole_unit_cell_without_triad_truncation(D, p):
    """R6's canonical-form shortcut (:137): with K = the full pair dimension nothing is lost in the triad split, the lower half
    is isometric and the upper half is (isometry) x sigma, so the Gram matrix of the WHOLE cell Gamma^ATRG = A X sigma Y D
    (Eq. 2.6 :98) on a forward pair equals Theta_f (upper half only) and on a backward pair equals Theta_b (sigma-weighted lower half)."""
    o = O.TatrgOracle(0.1497, 0.02, D, p, 9, n_pow=2, K=D * D)
    for _ in range(4):
        o.step()
    last = o.last
    a, dt, x, y, sig = last["a"], last["dt"], last["x"], last["y"], last["sig"]
    # Gamma[i1, i2u,i3u,i4u, i2l,i3l,i4l, j2u,j3u,j4u, j1, j2l,j3l,j4l]
    gam = np.einsum("iuvwa,axyzg,g,bpqrg,jstcb->iuvwxyzpqrjstc", a, x, sig, y, dt, optimize=True)
    e, f, g, h = last["efgh"]
    ua, ux, uy, ud = last["u"]
    for mu in (2, 3, 4):
        fu, fl = mu - 1, mu + 2
        gf = np.moveaxis(gam, (fu, fl), (-2, -1))
        du, dl = gf.shape[-2:]
        gf = gf.reshape(-1, du * dl)
        th_f = O.squeezer_grams(e, f, ua, ux, mu).reshape(du * dl, du * dl)
        assert np.abs(gf.T @ gf - th_f).max() < 1e-11 * np.abs(th_f).max()
        bu, bl = mu + 5, mu + 9
        gb = np.moveaxis(gam, (bu, bl), (0, 1)).reshape(du * dl, -1)
        th_b = O.squeezer_grams_lower(g * sig, h, uy, ud, mu).reshape(du * dl, du * dl)
        assert np.abs(gb @ gb.T - th_b).max() < 1e-11 * np.abs(th_b).max()


def test_z2_symmetry_in_exact_swap_mode():
    """R1: ln Z(+h) = ln Z(-h); holds to rounding when the bond swap is the exact SVD (no sketch noise)."""
    vals = []
    for h in (1e-2, -1e-2):
        o = O.TatrgOracle(0.1497, h, 4, 4, 3, n_pow=1, exact_swap=True)
        for _ in range(8):
            o.step()
        vals.append(o.lnZ_per_site())
    assert abs(vals[0] - vals[1]) < 1e-12


def test_gamma_gauge_invariance_of_a_step():
    """T = Phi Psi^T is unchanged by Phi -> Phi R, Psi -> Psi R^-T: one full step must give the same ln Z and
    spectra (checks that no stage depends on the factor-bond basis)."""
    o1 = _state_after(3, D=4, p=4)
    o2 = _state_after(3, D=4, p=4)
    rng = np.random.default_rng(3)
    r = rng.standard_normal((o2.phi.shape[-1],) * 2) + 2 * np.eye(o2.phi.shape[-1])
    o2.phi = o2.phi @ r
    o2.psi = o2.psi @ np.linalg.inv(r).T
    o1.step(), o2.step()
    assert abs(o1.lnZ_per_site() - o2.lnZ_per_site()) < 1e-12
    assert np.abs(o1.last["sigma"][:4] - o2.last["sigma"][:4]).max() < 1e-11


def test_noise_stability_of_the_gauge_fixing():
    """R7+R10+R12: 1e-13 relative noise on the state at every step changes ln Z/V by ~1e-13, not 1e-5."""
    def go(noise):
        rng = np.random.default_rng(1)
        o = O.TatrgOracle(0.1497, 0.0, 4, 4, 5, n_pow=1)
        for _ in range(12):
            if noise:
                o.phi = o.phi * (1 + noise * rng.standard_normal(o.phi.shape))
                o.psi = o.psi * (1 + noise * rng.standard_normal(o.psi.shape))
            o.step()
        return o.lnZ_per_site()
    assert abs(go(0.0) - go(1e-13)) < 5e-12


# ---- X ratio, Eq. 3.3 :298-303 ---------------------------------------------------------------------------------
@pytest.mark.parametrize("beta", [0.14, 0.1497, 0.7])
def test_x_ratio_of_the_initial_tensor_closed_form(beta):
    """A[k,l] = e^{3 beta} sum_a w_a[k] w_a[l] with w_a = (sqrt cosh, +-sqrt sinh):  X = e^{2 beta} / cosh(2 beta)."""
    phi, psi = O.init_tensor(beta, 0.0)
    assert abs(O.x_ratio(phi, psi) - math.exp(2 * beta) / math.cosh(2 * beta)) <= 1e-14


@pytest.mark.parametrize("beta,h", [(0.14, 0.0), (0.3, 0.05)])
def test_x_ratio_after_one_exact_step_is_a_ratio_of_partition_functions(beta, h):
    """After one (exact, D >= 4) step the open axis is the coarse-grained one: Tr A = Z(2x1x1x1) and
    Tr A^2 = Z(4x1x1x1) up to the same normalisation squared, both by brute-force enumeration."""
    o = O.TatrgOracle(beta, h, 4, 4, 1, n_pow=1)
    o.step()
    z2 = math.exp(2 * enumerate_lnz_per_site((2, 1, 1, 1), beta, h))
    z4 = math.exp(4 * enumerate_lnz_per_site((4, 1, 1, 1), beta, h))
    assert abs(o.x_ratio() - z2 * z2 / z4) <= 1e-12 * (z2 * z2 / z4)


def test_x_ratio_counts_the_ground_state_degeneracy():
    """X -> 2 in the ordered phase, X -> 1 in the disordered phase (:303)."""
    lo = O.TatrgOracle(1.0, 0.0, 4, 4, 3, n_pow=1)
    hi = O.TatrgOracle(0.05, 0.0, 4, 4, 3, n_pow=1)
    for m in range(16):
        hi.step()
        if m < 8:
            lo.step()
    assert abs(lo.x_ratio() - 2.0) <= 1e-6 and abs(hi.x_ratio() - 1.0) <= 1e-2


# ---- plain ATRG (Eq. 2.7-2.8 :104-113) -----------------------------------------------------------------------------------
@pytest.mark.parametrize("beta,h", [(0.14, 0.0), (0.1497, 1e-3)])
def test_atrg_one_and_two_steps_are_exact(beta, h):
    """Same enumeration pins as the triad method: nothing is truncated in step 1 at D >= 4 and in step 2 at D >= 16."""
    o = O.TatrgOracle(beta, h, 16, 0, 1, n_pow=1, method="atrg")
    o.step()
    assert abs(o.lnZ_per_site() - enumerate_lnz_per_site((2, 1, 1, 1), beta, h)) <= 1e-13
    o.step()
    assert abs(o.lnZ_per_site() - enumerate_lnz_per_site((2, 2, 1, 1), beta, h)) <= 1e-12


def test_triad_with_full_internal_dimension_recovers_atrg():
    """PAPER.md :179 "r = D recovers ATRG": the triad run with K = chi2*chi3 and the plain ATRG run agree (up to the
    1e-6 numerical-rank cut of the triad isometries, reading R14)."""
    t = O.TatrgOracle(0.1497, 0.0, 4, 4, 9, n_pow=1, K=16)
    a = O.TatrgOracle(0.1497, 0.0, 4, 4, 9, n_pow=1, method="atrg")
    for _ in range(6):
        t.step()
        a.step()
        assert abs(t.lnZ_per_site() - a.lnZ_per_site()) <= 1e-8


def test_atrg_staged_gram_equals_definition_on_random_tensors():
    """atrg_grams is one einsum of four operands; check it against the explicit half-cell tensor."""
    p = inputs.random_tensor((2, 3, 2, 3, 2), 1)
    q = inputs.random_tensor((2, 2, 3, 2, 3), 2)
    half = np.einsum("iucda,alefg->iuclefdg", p, q)               # [o1,u2,u3,l2,l3,l4,u4,o2]
    th2 = np.einsum("iuclefdg,ivcwefdg->ulvw", half, half)
    assert np.abs(O.atrg_grams(p, q, 2) - th2).max() <= 1e-12


# ------------------------------------------------------------------------------------------------ ILO Triad-ATRG (section 2.3)
def test_ilo_bond_rank_equal_D_is_plain_triad_atrg():
    """':331 When r_bond = 1 is set, it returns to the conventional ATRG bond-swapping process.'"""
    o0 = O.TatrgOracle(0.1497, 0.0, 4, 4, 3, n_pow=1)
    o1 = O.TatrgOracle(0.1497, 0.0, 4, 4, 3, n_pow=1, bond_rank=4)
    for _ in range(5):
        o0.step(); o1.step()
        assert o0.lnZ_per_site() == o1.lnZ_per_site()


def test_ilo_shapes_follow_footnote_5():
    """fn 5 :203: with overspanning, X and Y become (r_bond D) x D x D x D x (r_bond D) once the overspanned gamma of one step
    has become the alpha, beta of the next; the squeezed legs stay at D; sigma has r_bond D entries (Eq. A.1 :337)."""
    D, Db = 3, 6
    o = O.TatrgOracle(0.1497, 0.0, D, D, 5, n_pow=2, bond_rank=Db)
    for _ in range(6):
        o.step()
    assert o.phi.shape == (D, D, D, D, Db) and o.psi.shape == (D, D, D, D, Db)
    assert o.last["x"].shape == (Db, D, D, D, Db) and o.last["y"].shape == (Db, D, D, D, Db)
    assert len(o.last["sig"]) == Db and o.last["a"].shape == (D, D, D, D, Db)
    for t in (o.last["x"], o.last["y"], o.last["a"], o.last["dt"]):      # still isometries (:137, :339)
        m = t.reshape(-1, t.shape[-1])
        assert np.abs(m.T @ m - np.eye(m.shape[1])).max() < 1e-12


def test_ilo_decomposition_keeps_the_whole_overspanned_bond():
    """fn 5: 'the subscripts alpha and beta in Eq. (2.4) are also overspanned': T = Phi Psi^T of an ILO state (factor bond
    r_bond D) is reproduced exactly by A c Dt^T -- the decomposition at rank r_bond D truncates nothing."""
    D, Db = 3, 6
    o = O.TatrgOracle(0.1497, 0.0, D, D, 5, n_pow=2, bond_rank=Db)
    for _ in range(5):
        o.step()
    a, dt, core, s, lnc = O.decompose(o.phi, o.psi, Db, 5, 6)
    chi = a.shape[-1]
    t = o.phi.reshape(-1, Db) @ o.psi.reshape(-1, Db).T
    assert chi == Db and np.abs(a.reshape(-1, chi) @ core @ dt.reshape(-1, chi).T * math.exp(lnc) - t).max() < 1e-12 * np.abs(t).max()
    a3, dt3, core3, _, lnc3 = O.decompose(o.phi, o.psi, D, 5, 6)             # rank D would truncate it
    assert np.abs(a3.reshape(-1, D) @ core3 @ dt3.reshape(-1, D).T * math.exp(lnc3) - t).max() > 1e-6 * np.abs(t).max()


def test_ilo_bond_swap_is_the_best_rank_rbondD_approximation():
    """App. A :339 'this decomposition ... yields an optimal low-rank approximation of the unit-cell tensor in terms of the
    Frobenius norm' (Eckart-Young): at rank r_bond D the squared error of X sigma Y against sum_i1 B C is the sum of the
    discarded squared singular values, and it is smaller than at rank D."""
    o = _state_after(2, D=4, p=4)
    a, dt, core, s, _ = O.decompose(o.phi, o.psi, 4, 11, 3)
    b = np.einsum("ijklc,ac->ijkla", dt, core)
    c = np.einsum("ijklc,cb->ijklb", a, core)
    lhs = np.einsum("ijkla,imnob->amnobjkl", b, c)
    errs = []
    for rank in (4, 8, 12):
        x, y, sig, sig_all = O.bond_swap(a, dt, core, rank, 0, 0, 11, 3, exact=True)
        assert len(sig) == rank
        rhs = np.einsum("amnog,g,bjklg->amnobjkl", x, sig, y)
        err2 = float(((lhs - rhs) ** 2).sum())
        tail2 = float(((sig_all[rank:] * sig[0]) ** 2).sum())
        assert abs(err2 - tail2) < 1e-12 * float((lhs ** 2).sum())
        errs.append(err2)
    assert errs[0] > errs[1] > errs[2]


@pytest.mark.parametrize("beta,h", [(0.14, 0.0), (0.1497, 1e-3)])
def test_ilo_first_steps_stay_exact(beta, h):
    """Overspanning never truncates more: one and two steps remain exact against brute-force enumeration."""
    o = O.TatrgOracle(beta, h, 16, 16, 2, n_pow=2, bond_rank=32)
    o.step()
    assert abs(o.lnZ_per_site() - enumerate_lnz_per_site((2, 1, 1, 1), beta, h)) < 2e-14
    o.step()
    assert abs(o.lnZ_per_site() - enumerate_lnz_per_site((2, 2, 1, 1), beta, h)) < 1e-13


# ------------------------------------------------------------------------------------------------ ILO without X, Y (:394, :201)
def _swap_factors(D=3, Db=6, steps=4, seed=5):
    """An overspanned state after `steps` ILO steps and the factors of its next bond swap, stopped at Eq. A.9."""
    o = O.TatrgOracle(0.1497, 0.0, D, D, seed, n_pow=2, bond_rank=Db)
    for _ in range(steps):
        o.step()
    a, dt, core, s, _ = O.decompose(o.phi, o.psi, Db, seed, steps + 1)
    ub, vb, qc, qb, sig, sig_all = O.bond_swap(a, dt, core, Db, D, 2, seed, steps + 1, lift=False)
    x, y, sig2, _ = O.bond_swap(a, dt, core, Db, D, 2, seed, steps + 1)
    return a, dt, ub, vb, qc, qb, sig, x, y, sig2


def test_implicit_factors_are_the_lift_of_eq_A10_A11():
    """lift=False returns exactly the operands of Eq. A.10-A.11 :389-392: contracting them gives the X, Y of the explicit route,
    Q^C and Q^B are isometries (Eq. A.2-A.3 :345-348), and U^bond, V^bond are isometries on (al q) resp. (be p) (Eq. A.9 :379)."""
    a, dt, ub, vb, qc, qb, sig, x, y, sig2 = _swap_factors()
    assert np.array_equal(sig, sig2)
    assert np.abs(np.einsum("aqg,jklq->ajklg", ub, qc) - x).max() < 1e-14
    assert np.abs(np.einsum("bpg,jklp->bjklg", vb, qb) - y).max() < 1e-14
    for q in (qc, qb):
        m = q.reshape(-1, q.shape[-1])
        assert np.abs(m.T @ m - np.eye(m.shape[1])).max() < 1e-13
    for u in (ub, vb):
        m = u.reshape(-1, u.shape[-1])
        assert np.abs(m.T @ m - np.eye(m.shape[1])).max() < 1e-12


def test_implicit_triad_grams_equal_the_definition_on_explicit_x_y():
    """:394 'we work directly with U^bond, sigma, and V^*bond to create isometries of the triad representation': the four Gram
    matrices of Eq. 2.9 :135 formed without X, Y have the spectra of the ones formed from X, Y (all D^2 eigenvalues, not only the
    kept ones), and the projectors U U^T on the kept subspaces agree wherever the cut does not fall inside a multiplet."""
    a, dt, ub, vb, qc, qb, sig, x, y, _ = _swap_factors()
    K = 6
    iso_i, spec_i = O.triad_isometries_implicit(a, dt, ub, vb, qc, qb, sig, K)
    iso_e, spec_e = O.triad_isometries(a, dt, x, y, sig, K)
    for li, le in zip(spec_i, spec_e):
        assert np.abs(li - le).max() <= 1e-12 * le[0]
    for ui, ue, lam in zip(iso_i, iso_e, spec_e):
        assert ui.shape == ue.shape
        k = ui.shape[-1]
        if k < len(lam) and lam[k - 1] - lam[k] < 1e-6 * lam[0]:
            continue
        pi, pe = ui.reshape(-1, k), ue.reshape(-1, k)
        assert np.abs(pi @ pi.T - pe @ pe.T).max() < 1e-8
    # the definition itself, written out on the explicit X (not through triad_isometries): G^X and kappa^A of Eq. 2.9 / :137
    xs = x * sig
    gx_def = np.einsum("ajklg,amnlg->jkmn", xs, xs).reshape(9, 9)
    lam_def = np.sort(np.linalg.eigvalsh(gx_def))[::-1]
    assert np.abs(lam_def - spec_i[1]).max() <= 1e-12 * lam_def[0]
    # a wrong weight (sigma instead of sigma^2) or a dropped Q^C would not survive this: change sigma and the spectrum must move
    _, spec_w = O.triad_isometries_implicit(a, dt, ub, vb, qc, qb, np.sqrt(sig), K)
    assert np.abs(spec_w[1] - lam_def).max() > 1e-3 * lam_def[0]


def test_implicit_triad_tensors_equal_eq_2_11_2_12_on_explicit_x_y():
    """F and G of Eq. 2.11-2.12 :151-155 from (U^bond, Q^C), (V^bond, Q^B) equal those from X, Y for the same isometries; E, H do
    not involve the swapped bond."""
    a, dt, ub, vb, qc, qb, sig, x, y, _ = _swap_factors(D=3, Db=6, steps=5, seed=9)
    (ua, ux, uy, ud), _ = O.triad_isometries(a, dt, x, y, sig, 6)
    e0, f0, g0, h0 = O.triad_tensors(a, dt, x, y, sig, ua, ux, uy, ud)
    e1, f1, g1, h1 = O.triad_tensors_implicit(a, dt, ub, vb, qc, qb, sig, ua, ux, uy, ud)
    assert np.array_equal(e0, e1) and np.array_equal(h0, h1)
    assert f1.shape == f0.shape and g1.shape == g0.shape
    assert np.abs(f1 - f0).max() < 1e-13 and np.abs(g1 - g0).max() < 1e-13


@pytest.mark.parametrize("D,Db,p,n_pow", [(3, 6, 3, 2), (4, 8, 4, 1), (4, 4, 4, 1)])
def test_implicit_run_equals_explicit_run(D, Db, p, n_pow):
    """The whole ILO run without X, Y gives the explicit route's ln Z/V and spectra step by step (rounding order only differs);
    X and Y are never stored.  (4, 4) is the plain Triad-ATRG of section 2.2: the implicit form does not need r_bond > 1."""
    o0 = O.TatrgOracle(0.1497, 0.0, D, p, 7, n_pow=n_pow, bond_rank=Db)
    o1 = O.TatrgOracle(0.1497, 0.0, D, p, 7, n_pow=n_pow, bond_rank=Db, implicit_xy=True)
    for m in range(8):
        o0.step(); o1.step()
        assert o1.last["x"] is None and o1.last["y"] is None
        assert abs(o0.lnZ_per_site() - o1.lnZ_per_site()) <= 1e-12 * abs(o0.lnZ_per_site()), m
        assert np.abs(o0.last["sigma"] - o1.last["sigma"]).max() <= 1e-10
        assert np.abs(o0.last["s"] - o1.last["s"]).max() <= 1e-10


def test_implicit_xy_is_a_triad_feature():
    with pytest.raises(ValueError):
        O.TatrgOracle(0.1497, 0.0, 3, 3, 1, method="atrg", implicit_xy=True)
