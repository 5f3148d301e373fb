"""GPU parity tests of the kernels the Triad-ATRG path is made of, through the C ABI, against the CPU oracle's
routines (oracle/) or their plain numpy definition in FP64.  Sizes span several tiles and a ragged tail.

Tolerances: a K-term FP64 dot product accumulated in a different order differs by at most
~K * 2^-53 * sum|a_k b_k|; the tests bound that by 64 * eps * K * max|a| * max|b| ... integers are bit-exact."""
import numpy as np
import pytest

import paper_2507_21909_b200 as T
from tests import inputs

pytestmark = pytest.mark.gpu
EPS = 2.0 ** -52


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


# ---- Philox (bit-exact integers, Gaussians to a few ulp) --------------------------------------------------------------
@pytest.mark.parametrize("seed,call,stream,start,count", [(0, 0, 0, 0, 1), (1234, 7, 0, 0, 4099), (2 ** 63 + 5, 3, 1, 2 ** 32 - 3, 1000),
                                                          (42, 60, 4, 123456789012, 257)])
def test_philox_integers_bit_exact(torch, seed, call, stream, start, count):
    from oracle import philox
    raw = T.philox_raw(seed, call, stream, start, count)
    e = np.arange(start, start + count, dtype=np.uint64)
    ref = philox.philox4x32_10(e & np.uint64(0xFFFFFFFF), e >> np.uint64(32), call, stream, seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)
    assert np.array_equal(raw, np.stack(ref, axis=1))


def test_philox_known_answer_on_device(torch):
    assert [hex(v) for v in T.philox_raw(0, 0, 0, 0, 1)[0]] == ["0x6627e8d5", "0xe169c58d", "0xbc57ac4c", "0x9b00dbd8"]


def test_philox_gaussians_match_oracle(torch):
    from oracle import philox
    z = T.philox_gaussian(1234, 5, 0, 1000, 200003)
    ref = philox.gaussians(1234, 5, 0, 1000, 200003)
    # libm vs CUDA math: log, sqrt, cos(2 pi u) differ by a few ulp of the result scale (|z| <= ~9)
    assert np.abs(z - ref).max() <= 64 * EPS
    assert T.philox_gaussian(1, 1, 1, 0, 0).size == 0


# ---- DGEMM --------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("M,N,K", [(1, 1, 1), (128, 128, 16), (129, 257, 33), (300, 70, 1000), (64, 2048, 7), (5, 5, 100003), (1024, 3, 64)])
@pytest.mark.parametrize("ta,tb", [(False, False), (True, False), (False, True), (True, True)])
def test_dgemm_matches_definition(torch, M, N, K, ta, tb):
    a = inputs.random_tensor((M, K), 1)
    b = inputs.random_tensor((K, N), 2)
    ref = a @ b
    A = dev(torch, a.T if ta else a)
    B = dev(torch, b.T if tb else b)
    C = T.dgemm(A, B, transa=ta, transb=tb).cpu().numpy()
    bound = 8 * EPS * K * np.abs(a).max() * np.abs(b).max()
    assert np.abs(C - ref).max() <= bound


def test_dgemm_batched_alpha_beta(torch):
    a = inputs.random_tensor((5, 70, 40), 3)
    b = inputs.random_tensor((5, 40, 90), 4)
    c0 = inputs.random_tensor((5, 70, 90), 5)
    C = dev(torch, c0)
    T.dgemm(dev(torch, a), dev(torch, b), alpha=0.5, beta=-2.0, C=C)
    ref = 0.5 * np.einsum("bik,bkj->bij", a, b) - 2.0 * c0
    assert np.abs(C.cpu().numpy() - ref).max() <= 8 * EPS * 40 * 25


@pytest.mark.parametrize("M,N,K", [(1666, 1538, 70), (2050, 1300, 16), (1280, 1920, 130)])
@pytest.mark.parametrize("ta,tb", [(False, False), (True, False), (False, True), (True, True)])
def test_dgemm_multiwave(torch, M, N, K, ta, tb):
    """More than 148 tiles of 128 x 128 (several waves of CTAs) with 16-byte-aligned operands: ragged last tiles in M and N, K not a
    multiple of the 16-deep k-step, a K of exactly one k-step (shorter than the cp.async pipeline)."""
    a = inputs.random_tensor((M, K), 11)
    b = inputs.random_tensor((K, N), 12)
    ref = a @ b
    C = T.dgemm(dev(torch, a.T if ta else a), dev(torch, b.T if tb else b), transa=ta, transb=tb).cpu().numpy()
    assert np.abs(C - ref).max() <= 8 * EPS * K * np.abs(a).max() * np.abs(b).max()


def test_dgemm_multiwave_batched_alpha_beta(torch):
    a = inputs.random_tensor((3, 1100, 48), 13)
    b = inputs.random_tensor((3, 48, 1000), 14)
    c0 = inputs.random_tensor((3, 1100, 1000), 15)
    C = dev(torch, c0)
    T.dgemm(dev(torch, a), dev(torch, b), alpha=-1.5, beta=0.25, C=C)
    ref = -1.5 * np.einsum("bik,bkj->bij", a, b) + 0.25 * c0
    assert np.abs(C.cpu().numpy() - ref).max() <= 8 * EPS * 48 * np.abs(a).max() * np.abs(b).max() * 2


@pytest.mark.parametrize("M,N,K", [(128, 128, 16), (1, 1, 1), (130, 70, 33), (1666, 1538, 70), (2050, 1300, 16), (1280, 1920, 131), (300, 260, 1000)])
@pytest.mark.parametrize("ta,tb", [(False, False), (True, False), (False, True), (True, True)])
def test_dgemm_tma_variant_matches_definition(torch, M, N, K, ta, tb):
    """The TMA-fed 128 x 128 x 16 tile (tensor maps with zero fill instead of predicates, 128B-swizzled tiles, permuted atom rows):
    all four storage orders, ragged M, N, K (K odd, K shorter than one k-step, K longer than the 6-stage ring), several waves."""
    ld_a = (M if ta else K) + ((M if ta else K) & 1)            # tensor maps need even leading dimensions
    ld_b = (K if tb else N) + ((K if tb else N) & 1)
    a = inputs.random_tensor((M, K), 21)
    b = inputs.random_tensor((K, N), 22)
    A = torch.zeros((K if ta else M, ld_a), dtype=torch.float64, device="cuda")
    B = torch.zeros((N if tb else K, ld_b), dtype=torch.float64, device="cuda")
    A[:, :(M if ta else K)] = dev(torch, a.T if ta else a)
    B[:, :(K if tb else N)] = dev(torch, b.T if tb else b)
    C = torch.full((M, N), float("nan"), dtype=torch.float64, device="cuda")
    import ctypes
    rc = T.lib().tatrg_dgemm_variant(ctypes.c_void_p(torch.cuda.current_stream().cuda_stream), 1, int(ta), int(tb), M, N, K, 1.0,
                                     ctypes.c_void_p(A.data_ptr()), ld_a, ctypes.c_void_p(B.data_ptr()), ld_b, 0.0, ctypes.c_void_p(C.data_ptr()), N, 1, 0, 0, 0)
    assert rc == T.OK
    assert np.abs(C.cpu().numpy() - a @ b).max() <= 8 * EPS * K * np.abs(a).max() * np.abs(b).max()


def test_dgemm_tma_variant_batched_broadcast_alpha_beta(torch):
    a = inputs.random_tensor((3, 1100, 48), 13)
    b = inputs.random_tensor((3, 48, 1000), 14)
    c0 = inputs.random_tensor((3, 1100, 1000), 15)
    C = dev(torch, c0)
    T.dgemm(dev(torch, a), dev(torch, b), alpha=-1.5, beta=0.25, C=C, variant=1)
    ref = -1.5 * np.einsum("bik,bkj->bij", a, b) + 0.25 * c0
    assert np.abs(C.cpu().numpy() - ref).max() <= 8 * EPS * 48 * np.abs(a).max() * np.abs(b).max() * 2
    # broadcast B (batch stride 0), transposed A
    import ctypes
    at = dev(torch, np.ascontiguousarray(np.transpose(a, (0, 2, 1))))
    b0 = dev(torch, b[0])
    out = torch.empty((3, 1100, 1000), dtype=torch.float64, device="cuda")
    rc = T.lib().tatrg_dgemm_variant(ctypes.c_void_p(torch.cuda.current_stream().cuda_stream), 1, 1, 0, 1100, 1000, 48, 1.0, ctypes.c_void_p(at.data_ptr()), 1100,
                                     ctypes.c_void_p(b0.data_ptr()), 1000, 0.0, ctypes.c_void_p(out.data_ptr()), 1000, 3, 48 * 1100, 0, 1100 * 1000)
    assert rc == T.OK
    assert np.abs(out.cpu().numpy() - np.einsum("bik,kj->bij", a, b[0])).max() <= 8 * EPS * 48 * np.abs(a).max() * np.abs(b).max()


def test_dgemm_tma_variant_rejects_what_tensor_maps_cannot_address(torch):
    a = torch.zeros((64, 33), dtype=torch.float64, device="cuda")      # odd leading dimension
    b = torch.zeros((33, 64), dtype=torch.float64, device="cuda")
    with pytest.raises(T.TatrgError):
        T.dgemm(a, b, variant=1)
    assert T.dgemm(a, b, variant=0).shape == (64, 64)


# ---- permute ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,perm", [((3, 5, 7, 4, 6), (1, 2, 3, 0, 4)), ((3, 5, 7, 4, 6), (4, 3, 2, 1, 0)), ((33, 65), (1, 0)),
                                        ((2, 2, 2, 2, 2), (1, 2, 3, 0, 4)), ((8, 8, 8, 8, 8), (0, 3, 4, 1, 2)), ((1, 7, 1, 5), (3, 2, 1, 0)),
                                        ((16, 16, 16, 16, 16), (1, 2, 3, 0, 4)), ((40, 3, 50), (2, 1, 0)), ((6,), (0,))])
def test_permute_bit_exact(torch, shape, perm):
    x = inputs.random_tensor(shape, 6)
    out = T.permute(dev(torch, x), perm).cpu().numpy()
    assert np.array_equal(out, np.transpose(x, perm))


# ---- contraction engine ---------------------------------------------------------------------------------------------------
SPECS = [("abc,cd->abd", (3, 4, 5), (5, 6)), ("ajklg,amnlg->jkmn", (3, 4, 5, 6, 7), (3, 2, 3, 6, 7)),
         ("mjk,Ijkla->Imla", (6, 3, 4), (5, 3, 4, 2, 3)), ("pia,bpm->iabm", (5, 3, 4), (4, 5, 6)),
         ("zul,axld->uaxzd", (3, 4, 5), (2, 6, 5, 3)), ("jp,Bjm->Bpm", (10, 4), (3, 10, 5)),
         ("ikua,ikvb->uavb", (3, 4, 5, 2), (3, 4, 5, 2)), ("Ikxzd,kxpq->Ipqzd", (4, 6, 5, 3, 2), (6, 5, 3, 4)),
         ("kmab,abxy->kmxy", (5, 5, 3, 3), (3, 3, 4, 4)), ("qib,iabm->aqm", (7, 2, 3), (2, 3, 3, 5)),
         ("a,a->", (1000,), (1000,)), ("ab,b->a", (200, 300), (300,))]


@pytest.mark.parametrize("spec,sa,sb", [s for s in SPECS if s[1] is not None])
def test_contract_matches_einsum(torch, spec, sa, sb):
    a = inputs.random_tensor(sa, 7)
    b = inputs.random_tensor(sb, 8)
    ref = np.einsum(spec.lower() if not any(ch.isupper() for ch in spec) else _lower_unique(spec), a, b)
    out = T.contract(spec, dev(torch, a), dev(torch, b)).cpu().numpy()
    k = a.size * b.size / max(ref.size, 1)
    assert out.shape == ref.shape
    assert np.abs(out - ref).max() <= 16 * EPS * max(k, 1) ** 0.5 * 25 * max(1.0, np.abs(ref).max())


def _lower_unique(spec):
    import string
    for ch in sorted(set(c for c in spec if c.isupper())):
        free = [c for c in string.ascii_lowercase if c not in spec][0]
        spec = spec.replace(ch, free)
    return spec


def test_contract_rejects_bad_specs(torch):
    a = dev(torch, inputs.random_tensor((3, 4), 1))
    with pytest.raises(T.TatrgError):
        T.contract("ab,cd->ad", a, a)          # b and c appear once
    with pytest.raises(T.TatrgError):
        T.contract("ab,bc->ac", a, a)          # extent mismatch on b


# ---- dot (tTr) ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 31, 1024, 1000003])
def test_dot(torch, n):
    x = inputs.random_tensor((n,), 9)
    y = inputs.random_tensor((n,), 10)
    ref = float(np.dot(x, y))
    assert abs(T.dot(dev(torch, x), dev(torch, y)) - ref) <= 8 * EPS * np.abs(x * y).sum()


# ---- eigen-decomposition vs the oracle's Jacobi ------------------------------------------------------------------------------
@pytest.mark.parametrize("n,rank", [(1, 1), (2, 2), (5, 3), (16, 16), (64, 40), (65, 65), (100, 30), (256, 256), (300, 120)])
def test_eigh_matches_oracle(torch, n, rank):
    from oracle import tatrg_oracle as O
    g = inputs.random_psd(n, rank, 11 + n)
    lam_o, v_o = O.jacobi_eigh(g)
    lam, vt = T.eigh(dev(torch, g))
    lam, vt = lam.cpu().numpy(), vt.cpu().numpy()
    assert np.abs(lam - lam_o).max() <= 64 * EPS * n * lam_o[0]
    assert np.abs(vt @ vt.T - np.eye(n)).max() <= 64 * EPS * n
    assert np.abs(vt.T @ (lam[:, None] * vt) - g).max() <= 64 * EPS * n * lam_o[0]
    # gauge-invariant: projector on the eigenvectors of the `rank` non-zero (geometric, simple) eigenvalues
    k = min(rank, 8)
    assert np.abs(vt[:k].T @ vt[:k] - v_o[:, :k] @ v_o[:, :k].T).max() <= 1e-10


def test_eigh_graded_gram_keeps_relative_accuracy_above_the_floor(torch):
    """Gram matrix with eigenvalues 1 .. 1e-12: every eigenvalue above the documented floor (1e-18 of the largest
    diagonal entry, two orders below GEMM rounding) must come out to FP64 absolute accuracy."""
    n = 96
    rng = np.random.default_rng(5)
    q, _ = np.linalg.qr(rng.standard_normal((n, n)))
    lam_true = 10.0 ** (-12 * np.arange(n) / (n - 1))
    g = (q * lam_true) @ q.T
    lam, vt = T.eigh(dev(torch, g))
    assert np.abs(lam.cpu().numpy() - lam_true).max() <= 64 * EPS * n


# ---- small SVD vs the oracle's one-sided Jacobi --------------------------------------------------------------------------------
@pytest.mark.parametrize("nv,ln", [(1, 1), (2, 5), (4, 4), (8, 16), (32, 32), (64, 64), (40, 96), (96, 96)])
def test_svd_rows_matches_oracle(torch, nv, ln):
    from oracle import tatrg_oracle as O
    x = inputs.lowrank_plus_noise(nv, ln, min(nv, ln, 6), 1e-3, 13 + nv)
    u_o, s_o, v_o = O.jacobi_svd(x)
    s, ut, va = T.svd_rows(dev(torch, x))
    s, ut, va = s.cpu().numpy(), ut.cpu().numpy(), va.cpu().numpy()
    assert np.abs(s - s_o[:nv]).max() <= 64 * EPS * max(nv, ln) * s_o[0]
    assert np.abs(va.T @ (s[:, None] * ut) - x).max() <= 64 * EPS * max(nv, ln) * s_o[0]
    assert np.abs(ut @ ut.T - np.eye(nv)).max() <= 64 * EPS * max(nv, ln)


def test_svd_rows_rank_deficient_gives_exact_zero_structure(torch):
    rng = np.random.default_rng(3)
    x = rng.standard_normal((8, 2)) @ rng.standard_normal((2, 12))
    s, ut, va = T.svd_rows(dev(torch, x))
    s = s.cpu().numpy()
    assert (s[2:] <= 1e-13 * s[0]).all() and s[1] > 1e-3 * s[0]


# ---- Cholesky QR (blocked Cholesky + triangular solve) ----------------------------------------------------------------------
@pytest.mark.parametrize("m,n,cond", [(7, 7, 1.0), (100, 7, 10.0), (1000, 64, 1e3), (3000, 130, 1e2), (2500, 200, 1e4), (4096, 257, 30.0)])
def test_cholqr_is_the_qr_factorisation(torch, m, n, cond):
    """X = Q R with Q^T Q = 1 and R upper triangular with positive diagonal is unique: the three properties pin the result.
    One pass of Cholesky QR loses orthogonality like cond(X)^2 eps, X = Q R holds to eps."""
    rng = np.random.default_rng(m + n)
    x = inputs.random_tensor((m, n), 11) * (cond ** (-np.arange(n) / max(n - 1, 1)))      # graded columns
    if n > 1:
        x = x @ np.linalg.qr(rng.standard_normal((n, n)))[0]                              # and mixed: cond(X) ~ cond
    q, r = T.cholqr(dev(torch, x))
    q, r = q.cpu().numpy(), r.cpu().numpy()
    assert np.all(np.diag(r) > 0) and np.abs(np.tril(r, -1)).max() == 0.0
    scale = np.abs(x).max()
    assert np.abs(q @ r - x).max() <= 64 * EPS * n * scale
    assert np.abs(q.T @ q - np.eye(n)).max() <= 64 * EPS * n * max(1.0, np.linalg.cond(x) ** 2)
    # against the definition through the oracle's LAPACK-free Jacobi: R^T R = X^T X has the eigenvalues of the Gram matrix
    from oracle import tatrg_oracle as O
    if n <= 130:
        lam = np.sort(O.jacobi_eigh(x.T @ x)[0])
        lam_r = np.sort(O.jacobi_eigh(r.T @ r)[0])
        assert np.abs(lam - lam_r).max() <= 64 * EPS * n * lam.max()


def test_cholqr_reports_rank_deficiency(torch):
    x = inputs.random_tensor((500, 40), 3)
    x[:, 17] = x[:, 3] - 2.0 * x[:, 5]
    with pytest.raises(T.TatrgError):
        T.cholqr(dev(torch, x))


def _pivoted_cholesky_by_definition(g, tol_rel):
    """Greedy definition: always eliminate the largest remaining diagonal entry (lowest index on ties) of the Schur
    complement, stop when its trace is <= tol_rel tr G.  Returns (pivot order, residual trace / trace)."""
    s = g.copy()
    n = len(g)
    alive = np.ones(n, bool)
    t0 = np.trace(g)
    piv = []
    while True:
        d = np.where(alive, np.diag(s), -1.0)
        tr = d[d > 0].sum()
        k = int(np.argmax(d))
        if len(piv) == n or not d[k] > 0 or not tr > tol_rel * t0:
            return piv, tr / t0
        col = s[:, k] / np.sqrt(d[k])
        col[~alive] = 0.0
        s -= np.outer(col, col)
        alive[k] = False
        piv.append(k)


@pytest.mark.parametrize("n,rank,decades", [(5, 5, 1.0), (64, 64, 3.0), (200, 37, 2.0), (256, 256, 14.0), (513, 300, 20.0), (1024, 1024, 0.5), (1024, 500, 24.0), (1500, 90, 6.0)])
def test_pivoted_cholesky_is_the_truncated_factorisation(torch, n, rank, decades):
    """G = L L^T + S with S positive semi-definite and tr S <= tol tr G; the pivots are those of the greedy definition
    (compared while the remaining diagonal is far above the rounding of the updates); L^T L has the eigenvalues of G."""
    rng = np.random.default_rng(n + rank)
    q = np.linalg.qr(rng.standard_normal((n, rank)))[0]
    lam = 10.0 ** (-decades * np.arange(rank) / max(rank - 1, 1))
    g = (q * lam) @ q.T
    g = 0.5 * (g + g.T)
    tol = 1e-14
    L, r, resid = T.pchol(dev(torch, g), tol)
    L = L.cpu().numpy()
    assert 1 <= r <= min(n, rank + 2) and L.shape == (n, r)
    s = g - L @ L.T
    assert np.abs(s).max() <= max(2 * tol * np.trace(g), 64 * EPS * n * np.abs(g).max())
    assert resid <= tol or r == n
    assert np.linalg.eigvalsh(s).min() >= -64 * EPS * n * np.abs(g).max()
    piv, resid_def = _pivoted_cholesky_by_definition(g, tol)
    # each column of L has its pivot entry as the largest entry: L[k_j, j]^2 is the pivot, |L[i, j]| <= L[k_j, j]
    mine = [int(np.argmax(np.abs(L[:, j]))) for j in range(r)]
    safe = sum(1 for j in range(min(r, len(piv))) if L[mine[j], j] ** 2 > 1e-9 * np.abs(g).max())
    assert mine[:safe] == piv[:safe]
    assert abs(r - len(piv)) <= max(2, r // 50)
    # rows that were pivots are zero in later columns (lower triangular in pivot order)
    for j in range(r):
        assert np.all(L[mine[:j], j] == 0.0)
    w = np.sort(np.linalg.eigvalsh(g))[::-1][:r]
    w1 = np.sort(np.linalg.eigvalsh(L.T @ L))[::-1]
    assert np.abs(w - w1).max() <= 2 * tol * np.trace(g) + 64 * EPS * n * w[0]


def test_pivoted_cholesky_edge_cases(torch):
    z = np.zeros((17, 17))
    L, r, resid = T.pchol(dev(torch, z))
    assert r == 0
    e = np.eye(3)
    L, r, resid = T.pchol(dev(torch, e))
    assert r == 3 and np.array_equal(L.cpu().numpy(), e)           # ties: lowest index first
    with pytest.raises(T.TatrgError):
        T.pchol(dev(torch, e), tol_rel=-1.0)


@pytest.mark.parametrize("m,n", [(5, 3), (1000, 64), (4096, 256), (33000, 300), (2048, 1024), (777, 513)])
def test_gram_symmetric_mode_matches_definition(torch, m, n):
    """X^T X with only the lower tiles computed (n >= 256), split along K, mirrored: against the definition, and exactly symmetric."""
    x = inputs.random_tensor((m, n), 5)
    g = T.gram(dev(torch, x)).cpu().numpy()
    ref = x.T @ x
    assert np.abs(g - ref).max() <= 8 * EPS * m * np.abs(x).max() ** 2
    if n >= 256:
        assert np.array_equal(g, g.T)
