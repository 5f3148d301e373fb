"""oracle/tatrg_oracle.py -- TEST INFRASTRUCTURE ONLY.

Plain, slow, CPU/FP64 restatement of one Triad-ATRG coarse-graining step of the 4D Ising tensor network
(Sugimoto & Sasaki, arXiv:2507.21909; all "PAPER.md:<line>" citations are to /root/reference/PAPER.md).
It follows the paper step by step (Fig. 5 a-f, :193): every contraction is one np.einsum whose subscript
string is the paper's equation; every truncated SVD / eigen-decomposition is a LAPACK-free Jacobi iteration
(oracle/jacobi.c); random numbers come from oracle/philox.py.  Nothing here is shared with, imported by or
generated from the CUDA path (paper_2507_21909_b200/), and the product path never imports this module:
only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may.

Readings of silent / garbled passages are numbered R1..R14 as in DESIGN.md.

Parity status: exact (untruncated) results are pinned by closed forms and brute-force enumeration
(tests/test_oracle_pins.py).  Truncated multi-step values at D >= 4 on large lattices have no external
reference: **parity unpinned** beyond "error vs enumeration shrinks with D".

Index names (rotated frame, axis 1 = axis being coarse-grained, Eq. 2.4 :76):
  upper site n+1^ : forward legs i1 i2 i3 i4 ("u"), backward legs j2 j3 j4 (its j1 is the contracted bond)
  lower site n    : forward legs i2 i3 i4 ("l"),    backward legs j1 j2 j3 j4
  Phi[i1,i2,i3,i4,g], Psi[j1,j2,j3,j4,g]  with  T[f,b] = sum_g Phi[f,g] Psi[b,g]   (Eq. 2.18-2.19 :175)
"""
import ctypes
import math
import os

import numpy as np

from . import philox

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

# ---- numerical readings; the CUDA path states the same constants independently ----
TAU_MULTIPLET = 1e-6   # R7: values whose relative gap is <= tau belong to one multiplet (never split, rotate jointly)
EPS_ORTH = 1e-6        # R14: orth() drops directions with sigma <= eps * sigma_max (numerical rank)
EPS_SV = 1e-12         # R14: singular values of small, accurately computed cores below this (relative) are zero
EPS_LAMBDA = 1e-12     # R14: eigenvalues of Gram matrices below this (relative) are zero
EPS_SQUEEZER = 1e-6    # R14: squeezer singular values below this (relative) are dropped
JACOBI_TOL = 1e-15
JACOBI_MAX_SWEEPS = 60
RHO_COLS = 64          # R10: reference vectors rho[:, j], j < 64


def _lib():
    global _LIB
    if _LIB is None:
        path = os.path.join(_HERE, "liborc_jacobi.so")
        if not os.path.exists(path):
            raise RuntimeError("oracle/liborc_jacobi.so missing: run __graft_entry__.build() (gcc oracle/jacobi.c)")
        _LIB = ctypes.CDLL(path)
        dp = ctypes.POINTER(ctypes.c_double)
        _LIB.orc_jacobi_svd.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp, dp, ctypes.c_double, ctypes.c_int]
        _LIB.orc_jacobi_svd.restype = ctypes.c_int
        _LIB.orc_jacobi_eigh.argtypes = [ctypes.c_int, dp, dp, dp, ctypes.c_double, ctypes.c_int]
        _LIB.orc_jacobi_eigh.restype = ctypes.c_int
    return _LIB


def _es(subscripts, *operands):
    """One contraction = one library einsum (BLAS-backed when it is a matrix product); no hand blocking."""
    return np.einsum(subscripts, *operands, optimize=True)


def _ptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


# --------------------------------------------------------------------------------------------------------
# dense decompositions (Jacobi)
# --------------------------------------------------------------------------------------------------------
def jacobi_svd(a):
    """Thin SVD a = U diag(s) V^T of an m x n matrix, m >= n or not; s descending; U m x r, V n x r, r=min(m,n).
    One-sided Jacobi on the columns of the taller orientation.  Columns of U belonging to s == 0 are zero."""
    a = np.asarray(a, dtype=np.float64)
    m, n = a.shape
    if m < n:
        v, s, u = jacobi_svd(a.T)
        return u, s, v
    at = np.array(a.T, dtype=np.float64, order="C", copy=True)   # row j = column j of a (always a copy)
    s = np.zeros(n)
    vt = np.zeros((n, n))
    rc = _lib().orc_jacobi_svd(m, n, _ptr(at), _ptr(s), _ptr(vt), JACOBI_TOL, JACOBI_MAX_SWEEPS)
    if rc < 0:
        raise RuntimeError("jacobi_svd did not converge")
    order = np.argsort(-s, kind="stable")
    s = s[order]
    us = at[order]                          # rows = s_j u_j
    vt = vt[order]
    u = np.zeros((m, n))
    nz = s > 0
    u[:, nz] = (us[nz] / s[nz, None]).T
    return u, s, np.ascontiguousarray(vt.T)


def jacobi_eigh(sym):
    """Eigen-decomposition of a symmetric matrix: returns (lam descending, V with eigenvectors as columns)."""
    sym = np.array(sym, dtype=np.float64, order="C")
    n = sym.shape[0]
    sym = 0.5 * (sym + sym.T)
    lam = np.zeros(n)
    vt = np.zeros((n, n))
    rc = _lib().orc_jacobi_eigh(n, _ptr(sym), _ptr(lam), _ptr(vt), JACOBI_TOL, JACOBI_MAX_SWEEPS)
    if rc < 0:
        raise RuntimeError("jacobi_eigh did not converge")
    order = np.argsort(-lam, kind="stable")
    return lam[order], np.ascontiguousarray(vt[order].T)


def orth(mat, eps=EPS_ORTH):
    """Orthonormal basis of the numerical column space: mat = Q R, Q^T Q = 1, R = Q^T mat  (R14).
    The paper's QR decompositions (Eq. A.2-A.3 :345-348, A.4-A.6 :359-365; "QR (or singular value)
    decompositions" :343) only need span(Q); the SVD form reveals the rank, which plain QR does not."""
    u, s, v = jacobi_svd(mat)
    r = int(np.sum(s > eps * s[0])) if s[0] > 0 else 0
    q = u[:, :r]
    rmat = s[:r, None] * v[:, :r].T
    return q, rmat


# --------------------------------------------------------------------------------------------------------
# rank selection and gauge fixing (R7, R10)
# --------------------------------------------------------------------------------------------------------
def select_rank(v, kmax, eps, tau=TAU_MULTIPLET):
    """Number of leading values of the descending list v to keep: at most kmax, only values > eps*v[0], and
    never cutting through a multiplet (relative gap <= tau): the whole multiplet is dropped instead (R7)."""
    v = np.asarray(v)
    if len(v) == 0 or not v[0] > 0:
        return 0
    n_pos = int(np.sum(v > eps * v[0]))
    if n_pos <= kmax:
        return n_pos
    k = kmax
    while k > 0 and (v[k - 1] - v[k]) <= tau * v[k - 1]:
        k -= 1
    return k if k > 0 else kmax


def multiplets(v, k, tau=TAU_MULTIPLET):
    """Partition 0..k-1 into runs of consecutive values with relative gap <= tau: [(start, stop), ...]."""
    out, start = [], 0
    for i in range(1, k + 1):
        if i == k or (v[i - 1] - v[i]) > tau * v[i - 1]:
            out.append((start, i))
            start = i
    return out


def rho(seed, step, stream, nrows, ncols):
    """Reference vectors rho[r, j] = Gaussian(counter e = r*RHO_COLS + j) of the reserved stream (R10)."""
    assert ncols <= RHO_COLS
    z = philox.gaussians(seed, step, stream, 0, nrows * RHO_COLS).reshape(nrows, RHO_COLS)
    return z[:, :ncols]


def canonical_rotation(w, groups, seed, step, stream):
    """Block-diagonal orthogonal G (k x k) fixing the gauge of the columns of w (n x k) (R10).
    For each multiplet c: C = w_c^T rho[:, :g]; C = Q R by modified Gram-Schmidt with diag(R) > 0; block = Q.
    w_c -> w_c Q is invariant under w_c -> w_c O for any orthogonal O (for g = 1: a sign flip)."""
    n, k = w.shape
    g = np.zeros((k, k))
    gmax = max(b - a for a, b in groups)
    ref = rho(seed, step, stream, n, gmax)
    for a, b in groups:
        c = w[:, a:b].T @ ref[:, : b - a]
        q = np.zeros_like(c)
        for j in range(b - a):                      # modified Gram-Schmidt, column by column
            col = c[:, j].copy()
            for i in range(j):
                col -= (q[:, i] @ col) * q[:, i]
            q[:, j] = col / np.sqrt(col @ col)
        g[a:b, a:b] = q
    return g


# --------------------------------------------------------------------------------------------------------
# (a0) initial tensor, Eq. 3.1-3.2 :241-246
# --------------------------------------------------------------------------------------------------------
def w_matrix(beta):
    """Eq. 3.2 :246.  Row a = spin state (a=0: +1, a=1: -1), column = bond index."""
    c, s = math.sqrt(math.cosh(beta)), math.sqrt(math.sinh(beta))
    return np.array([[c, s], [c, -s]])


def init_tensor(beta, h=0.0):
    """Eq. 3.1 :241 in factored form T[f,b] = sum_a Phi0[f,a] Psi0[b,a]; the site weight e^{beta h s_a} (R1)
    is attached to Phi0."""
    w = w_matrix(beta)
    spin = np.array([1.0, -1.0])
    psi0 = _es("ai,aj,ak,al->ijkla", w, w, w, w)
    phi0 = psi0 * np.exp(beta * h * spin)
    return phi0, psi0


# --------------------------------------------------------------------------------------------------------
# (a1) decomposition of T, Eq. 2.4 :72-80, Fig. 5(a)
# --------------------------------------------------------------------------------------------------------
def decompose(phi, psi, D, seed, step, tau=TAU_MULTIPLET):
    """T = Phi Psi^T = A c Dt^T with A, Dt isometric (f x chi, b x chi) and c = s/s1 rotated to the canonical
    gauge (symmetric, block diagonal).  Returns A[i1..i4,al], Dt[j1..j4,be], c, s (normalised, all), ln c_m."""
    dims_f, dims_b = phi.shape[:4], psi.shape[:4]
    qf, rf = orth(phi.reshape(-1, phi.shape[4]))
    qb, rb = orth(psi.reshape(-1, psi.shape[4]))
    u, s, v = jacobi_svd(rf @ rb.T)                       # core of T: (Q_Phi^T T Q_Psi)
    c_m = s[0]
    s = s / c_m
    chi = select_rank(s, D, EPS_SV, tau)
    a = qf @ u[:, :chi]
    dt = qb @ v[:, :chi]
    g = canonical_rotation(a, multiplets(s, chi, tau), seed, step, 1)
    a, dt = a @ g, dt @ g
    core = g.T @ (s[:chi, None] * g)
    return a.reshape(dims_f + (chi,)), dt.reshape(dims_b + (chi,)), core, s, math.log(c_m)


# --------------------------------------------------------------------------------------------------------
# (a2-a4) bond swapping, Eq. 2.5 :90 and App. A :329-394
# --------------------------------------------------------------------------------------------------------
def bond_swap(a, dt, core, D, oversample, n_pow, seed, step, tau=TAU_MULTIPLET, exact=False, lift=True):
    """sum_i1 B[i1,j',al] C[i1,i',be] ~ sum_g X[al,i',g] sig[g] Y[be,j',g]  (Eq. 2.5 / A.1).
    B[i1,j2,j3,j4,al] = sum_a' Dt[i1,j2,j3,j4,a'] c[al,a'],  C[i1,i2,i3,i4,be] = sum_a' A[i1,..,a'] c[a',be].
    lift=False stops at Eq. A.9 :379 and returns (U^bond[al,q,g], V^bond[be,p,g], Q^C[i',q], Q^B[j',p], sig, sig_all): the
    form in which the ILO method keeps the swapped bond (:394 "the tensors X and Y are not explicitly constructed")."""
    b = _es("ijklc,ac->ijkla", dt, core)
    c = _es("ijklc,cb->ijklb", a, core)
    chi1, chi_a = b.shape[0], b.shape[4]
    dj, di = b.shape[1:4], c.shape[1:4]
    # Eq. A.2-A.3 :345-348  B[(j'),(i1 al)] = QB[(j'),p] RB[p,i1,al],  C[(i'),(i1 be)] = QC[(i'),q] RC[q,i1,be]
    qb_, rb_ = orth(_es("ijkla->jklia", b).reshape(np.prod(dj), chi1 * chi_a))
    qc_, rc_ = orth(_es("ijklb->jklib", c).reshape(np.prod(di), chi1 * chi_a))
    npb, npc = qb_.shape[1], qc_.shape[1]
    QB, RB = qb_.reshape(dj + (npb,)), rb_.reshape(npb, chi1, chi_a)
    QC, RC = qc_.reshape(di + (npc,)), rc_.reshape(npc, chi1, chi_a)
    if exact:
        # the plain definition: full SVD of the core S[(al q),(be p)] = sum_i1 RC[q,i1,be] RB[p,i1,al]
        smat = _es("qib,pia->aqbp", RC, RB).reshape(chi_a * npc, chi_a * npb)
        u, sig, v = jacobi_svd(smat)
        ubond, vbond = u.reshape(chi_a, npc, -1), v.reshape(chi_a, npb, -1)
    else:
        l_eff = min(D + oversample, chi_a * npc, chi_a * npb)      # R3: sketch width l = D + p
        n_el = chi_a * int(np.prod(dj)) * l_eff
        om_phys = philox.gaussians(seed, step, philox.STREAM_OMEGA, 0, n_el).reshape((chi_a,) + dj + (l_eff,))
        omega = _es("jklp,bjklm->bpm", QB, om_phys)          # R12: drawn in the physical basis
        for k in range(n_pow + 1):                                 # R4: q = n_pow + 1 passes
            t = _es("pia,bpm->iabm", RB, omega)
            y = _es("qib,iabm->aqm", RC, t)                  # Eq. A.4 :356
            qk, _ = orth(y.reshape(chi_a * npc, -1))
            qk = qk.reshape(chi_a, npc, -1)
            t2 = _es("qib,aqm->ibam", RC, qk)
            yt = _es("pia,ibam->bpm", RB, t2)                # Eq. A.5 :361  (= (Q^T S)^T)
            if k < n_pow:
                qp, _ = orth(yt.reshape(chi_a * npb, -1))          # Eq. A.6 :365-368
                omega = qp.reshape(chi_a, npb, -1)
        # Eq. A.7-A.8 :373-376: SVD of the projected tensor Q^T S = yt^T = U~ sig Vbond^T
        vb, sig, ut = jacobi_svd(yt.reshape(chi_a * npb, -1))
        ubond = _es("aqm,mg->aqg", qk, ut)                   # Eq. A.9 :379
        vbond = vb.reshape(chi_a, npb, -1)
    sig_all = sig / sig[0]
    g = select_rank(sig, D, EPS_SV, tau)
    if not lift:
        return ubond[:, :, :g], vbond[:, :, :g], QC, QB, sig[:g], sig_all
    x = _es("aqg,jklq->ajklg", ubond[:, :, :g], QC)         # Eq. A.10 :389
    y = _es("bpg,jklp->bjklg", vbond[:, :, :g], QB)         # Eq. A.11 :392
    return x, y, sig[:g], sig_all


# --------------------------------------------------------------------------------------------------------
# (a5) triad isometries, Eq. 2.9 :133-137
# --------------------------------------------------------------------------------------------------------
def _top_eigvecs(gram, K, tau):
    lam, vec = jacobi_eigh(gram)
    lam = np.maximum(lam, 0.0)
    sv = np.sqrt(lam)                                  # multiplet rule is applied on the singular-value scale
    k = select_rank(sv, K, math.sqrt(EPS_LAMBDA), tau)
    return vec[:, :k], lam


def triad_isometries(a, dt, x, y, sig, K, tau=TAU_MULTIPLET):
    """Truncated HOSVD of Gamma^ATRG = A X sig Y D on the leg pair (2,3) of each of A, X, Y, D (Eq. 2.9),
    using the canonical form (:137): the isometric remainder contracts to the identity."""
    xs, ys = x * sig, y * sig
    d2, d3 = x.shape[1], x.shape[2]
    gx = _es("ajklg,amnlg->jkmn", xs, xs)
    ka = _es("ajklg,bjklg->ab", xs, xs)
    ga = _es("ijkla,ab,imnlb->jkmn", a, ka, a)
    gy = _es("ajklg,amnlg->jkmn", ys, ys)
    kd = _es("ajklg,bjklg->ab", ys, ys)
    gd = _es("ijkla,ab,imnlb->jkmn", dt, kd, dt)
    out, spectra = [], []
    for gram in (ga, gx, gy, gd):
        vec, lam = _top_eigvecs(gram.reshape(d2 * d3, d2 * d3), K, tau)
        out.append(vec.reshape(d2, d3, -1))
        spectra.append(lam)
    return out, spectra


# --------------------------------------------------------------------------------------------------------
# (a6) triad tensors, Eq. 2.10-2.17 :147-167
# --------------------------------------------------------------------------------------------------------
def triad_tensors(a, dt, x, y, sig, ua, ux, uy, ud):
    e = _es("ijkla,jkm->imla", a, ua)               # Eq. 2.10  E[i1,kA,i4,al]
    f = _es("ajklg,jkm->amlg", x, ux) * sig         # Eq. 2.11  F[al,kX,i4,g]  (sigma goes into F only)
    g = _es("bjklg,jkm->bmlg", y, uy)               # Eq. 2.12  G[be,kY,j4,g]
    h = _es("ijklb,jkm->imlb", dt, ud)              # Eq. 2.13  H[j1,kD,j4,be]
    return e, f, g, h                                     # Eq. 2.14-2.17: I,J,K,L = ua,ux,uy,ud


# --------------------------------------------------------------------------------------------------------
# (a5-a6) without X and Y, PAPER.md :394 / :201 (ILO Triad-ATRG)
# --------------------------------------------------------------------------------------------------------
def triad_isometries_implicit(a, dt, ubond, vbond, qc, qb, sig, K, tau=TAU_MULTIPLET):
    """Eq. 2.9 with Eq. A.10-A.11 substituted, X = U^bond Q^C and Y = V^bond Q^B never formed (:394 "we work directly with
    U^bond, sigma and V^*bond to create isometries of the triad representation"; :201 "QR decomposition is applied before
    the bond-swapping step ..., which allows us to avoid constructing large intermediate tensors X and Y").
      G^X[(i2 i3),(i2' i3')] = sum_{i4} sum_{q q'} Q^C[i2 i3 i4, q] w^C[q,q'] Q^C[i2' i3' i4, q'],
      w^C[q,q'] = sum_{al,g} sig_g^2 U^bond[al,q,g] U^bond[al,q',g]
      kappa^A[al,al'] = sum_{q,g} sig_g^2 U^bond[al,q,g] U^bond[al',q,g]      (Q^C^T Q^C = 1, Eq. A.3 :348)
    and the same with V^bond, Q^B for G^Y, kappa^D.  Nothing larger than Q^C, Q^B (chi^3 x r_bond D^2) appears."""
    us, vs = ubond * sig, vbond * sig
    d2, d3 = qc.shape[0], qc.shape[1]
    wc = _es("aqg,arg->qr", us, us)
    gx = _es("jklq,qr,mnlr->jkmn", qc, wc, qc)
    ka = _es("aqg,bqg->ab", us, us)
    ga = _es("ijkla,ab,imnlb->jkmn", a, ka, a)
    wb = _es("bpg,brg->pr", vs, vs)
    gy = _es("jklp,pr,mnlr->jkmn", qb, wb, qb)
    kd = _es("apg,bpg->ab", vs, vs)
    gd = _es("ijkla,ab,imnlb->jkmn", dt, kd, dt)
    out, spectra = [], []
    for gram in (ga, gx, gy, gd):
        vec, lam = _top_eigvecs(gram.reshape(d2 * d3, d2 * d3), K, tau)
        out.append(vec.reshape(d2, d3, -1))
        spectra.append(lam)
    return out, spectra


def triad_tensors_implicit(a, dt, ubond, vbond, qc, qb, sig, ua, ux, uy, ud):
    """Eq. 2.10-2.13 with Eq. A.10-A.11 substituted: the isometry meets Q^C (Q^B) first, a chi4 x K x r_bond D^2 object, and
    U^bond (V^bond) afterwards, so F and G come out without X and Y (:394)."""
    e = _es("ijkla,jkm->imla", a, ua)               # Eq. 2.10
    pc = _es("jklq,jkm->mlq", qc, ux)               # sum_{i2,i3} Q^C[i2,i3,i4,q] U^X[i2,i3,kX]
    f = _es("aqg,mlq->amlg", ubond, pc) * sig       # Eq. 2.11 with A.10: F[al,kX,i4,g]
    pb = _es("jklp,jkm->mlp", qb, uy)
    g = _es("bpg,mlp->bmlg", vbond, pb)             # Eq. 2.12 with A.11: G[be,kY,j4,g]
    h = _es("ijklb,jkm->imlb", dt, ud)              # Eq. 2.13
    return e, f, g, h


# --------------------------------------------------------------------------------------------------------
# (a7-a8) squeezers, PAPER.md :113, :171  (formula not printed: reading R6)
# --------------------------------------------------------------------------------------------------------
def squeezer_grams(e, f, i_, j_, direction):
    """Gram matrix of the half unit cell  U[i1,(i2u i2l),(i3u i3l),(i4u i4l),g] =
    sum_{al,kA,kX} E[i1,kA,i4u,al] F[al,kX,i4l,g] I[i2u,i3u,kA] J[i2l,i3l,kX]  on the bond pair `direction`
    (2, 3 or 4), all other indices contracted with a second copy.  Staged so that no D^8 object appears.
    Returned as theta[u,l,u',l'] (u = upper-site leg, l = lower-site leg)."""
    if direction == 4:
        ee = _es("ikua,ikvb->aubv", e, e)           # I^T I = J^T J = 1 removes legs 2,3
        ff = _es("akld,bkwd->albw", f, f)
        return _es("aubv,albw->ulvw", ee, ff)
    ee = _es("ikua,imub->akbm", e, e)               # sum i1, i4u
    ff = _es("axld,byld->axby", f, f)               # sum i4l, g
    ef = _es("akbm,axby->kxmy", ee, ff)             # [kA,kX,kA',kX']
    if direction == 2:
        ii = _es("uck,vcm->ukvm", i_, i_)           # sum over the other leg (3) of the upper site
        jj = _es("lcx,wcy->lxwy", j_, j_)
    else:
        ii = _es("cuk,cvm->ukvm", i_, i_)
        jj = _es("clx,cwy->lxwy", j_, j_)
    tmp = _es("ukvm,kxmy->uvxy", ii, ef)
    return _es("uvxy,lxwy->ulvw", tmp, jj)


def squeezer_pair(theta_f, theta_b, D, seed, step, direction, tau=TAU_MULTIPLET):
    """Rank-<=D oblique projector M N^T on a doubled bond (R6): with theta_f = R1^T R1 (Gram of the cell that
    owns the bond as a forward pair) and theta_b = R2 R2^T (Gram of the neighbouring cell that owns it as a
    backward pair), SVD R1 R2 = U s V^T, M = R2 V s^-1/2, N = R1^T U s^-1/2.  N^T M = 1 and M N^T minimises
    ||G1 G2 - G1 M N^T G2||_F (refs [64-67] of the paper, cited at :113)."""
    du, dl = theta_f.shape[0], theta_f.shape[1]
    n = du * dl
    lam1, w1 = jacobi_eigh(theta_f.reshape(n, n))
    lam2, w2 = jacobi_eigh(theta_b.reshape(n, n))
    k1 = int(np.sum(lam1 > EPS_LAMBDA * lam1[0]))
    k2 = int(np.sum(lam2 > EPS_LAMBDA * lam2[0]))
    r1 = np.sqrt(lam1[:k1, None]) * w1[:, :k1].T          # theta_f = R1^T R1
    r2 = w2[:, :k2] * np.sqrt(lam2[:k2])                  # theta_b = R2 R2^T
    u, s, v = jacobi_svd(r1 @ r2)
    k = select_rank(s, D, EPS_SQUEEZER, tau)
    m = (r2 @ v[:, :k]) / np.sqrt(s[:k])
    nn = (r1.T @ u[:, :k]) / np.sqrt(s[:k])
    g = canonical_rotation(m * np.sqrt(s[:k]), multiplets(s, k, tau), seed, step, direction)   # R10 on R2 V
    return (m @ g).reshape(du, dl, k), (nn @ g).reshape(du, dl, k), s / s[0]


# --------------------------------------------------------------------------------------------------------
# (a9) coarse-graining contraction, Eq. 2.18-2.19 :175
# --------------------------------------------------------------------------------------------------------
def contract_half(e, f, i_, j_, m2, m3, m4):
    """Phi'[i1,k2,k3,k4,g] of Eq. 2.18 (and Psi' of Eq. 2.19 with H,G,L,K,N in place of E,F,I,J,M: the lower
    site's tensors H, L play the role of E, I there -- see coarse_grain)."""
    em = _es("ikua,ulz->ikalz", e, m4)
    xi = _es("ikalz,axld->ikxzd", em, f)            # Xi[i1,kA,kX,k4,g]
    im = _es("uck,ulz->kclz", i_, m2)
    imm = _es("kclz,cwy->klwzy", im, m3)
    lam = _es("klwzy,lwx->kxzy", imm, j_)           # Lambda[kA,kX,k2,k3]
    return _es("ikxzd,kxab->iabzd", xi, lam)


def contract_psi(g, h, k_, l_, n2, n3, n4):
    """Psi'[j1,k2,k3,k4,g] of Eq. 2.19 :175.  Squeezer index order is (upper leg, lower leg, new leg)."""
    hn = _es("jdlb,ulz->jdbuz", h, n4)
    xi = _es("jdbuz,byug->jdyzg", hn, g)            # Xi'[j1,kD,kY,k4,g]
    kn = _es("ucy,ulz->yclz", k_, n2)
    knn = _es("yclz,cwv->ylwzv", kn, n3)
    lam = _es("ylwzv,lwd->ydzv", knn, l_)           # Lambda'[kY,kD,k2,k3]
    return _es("jdyzg,ydab->jabzg", xi, lam)


# --------------------------------------------------------------------------------------------------------
# one step and the RG driver
# --------------------------------------------------------------------------------------------------------
class TatrgOracle:
    """State = (Phi, Psi, [ln c_m], step counter).  step() = Fig. 5 (a)-(f) :193."""

    def __init__(self, beta, h, D, oversample, seed, n_pow=2, K=None, tau=TAU_MULTIPLET, exact_swap=False, method="triad",
                 bond_rank=None, implicit_xy=False):
        self.beta, self.h, self.D, self.p, self.seed = beta, h, D, oversample, seed
        self.method = method                                   # "triad" (Eq. 2.9-2.19) or "atrg" (Eq. 2.7-2.8)
        # ILO Triad-ATRG (section 2.3 :183-209, App. A :331-394): the bond swap keeps r_bond D values (the sum over gamma in
        # Eq. A.1 :337 runs to r_bond D) and, one step later, so does the decomposition of T (fn 5 :203: "the subscripts alpha and
        # beta in Eq. (2.4) are also overspanned"); the RSVD sketch is r_bond D + p wide (fn 9 :381).  bond_rank = r_bond D; the
        # squeezed legs stay at D.  bond_rank = D is the Triad-ATRG of section 2.2.
        self.bond_rank = bond_rank if bond_rank is not None else D
        # implicit_xy: the triad isometries and F, G straight from U^bond, sigma, V^bond, Q^C, Q^B (:394, :201); X and Y never exist.
        # The same numbers as the explicit route up to rounding (pinned in tests/test_oracle_pins.py).
        self.implicit_xy = implicit_xy
        if implicit_xy and method != "triad":
            raise ValueError("implicit_xy belongs to the triad representation (plain ATRG contracts X and Y themselves, Eq. 2.7-2.8)")
        self.n_pow, self.tau, self.exact_swap = n_pow, tau, exact_swap
        self.K = K if K is not None else D + oversample        # R3: triad internal-line dimension rD = D + p
        self.phi, self.psi = init_tensor(beta, h)
        self.lnc = []
        self.m = 0
        self.last = {}

    def step(self):
        D, tau, call = self.D, self.tau, self.m + 1
        a, dt, core, s_all, lnc = decompose(self.phi, self.psi, self.bond_rank, self.seed, call, tau)          # (a)
        if self.implicit_xy:
            ub, vb, qc, qb, sig, sig_all = bond_swap(a, dt, core, self.bond_rank, self.p, self.n_pow, self.seed, call, tau,
                                                     exact=self.exact_swap, lift=False)              # (b) up to Eq. A.9
            x = y = None
            (ua, ux, uy, ud), tri_spec = triad_isometries_implicit(a, dt, ub, vb, qc, qb, sig, self.K, tau)   # (c), :394
            e, f, g, h = triad_tensors_implicit(a, dt, ub, vb, qc, qb, sig, ua, ux, uy, ud)
        else:
            x, y, sig, sig_all = bond_swap(a, dt, core, self.bond_rank, self.p, self.n_pow, self.seed, call, tau,
                                           exact=self.exact_swap)                                    # (b)
        if self.method == "atrg":
            return self._finish_atrg(a, dt, core, s_all, lnc, x, y, sig, sig_all, call)
        if not self.implicit_xy:
            (ua, ux, uy, ud), tri_spec = triad_isometries(a, dt, x, y, sig, self.K, tau)           # (c)
            e, f, g, h = triad_tensors(a, dt, x, y, sig, ua, ux, uy, ud)
        ms, ns, sq_spec = {}, {}, {}
        for mu in (2, 3, 4):                                                                        # (d)
            th_f = squeezer_grams(e, f, ua, ux, mu)
            # lower half: G carries sigma^2 in its Gram (canonical form); H, L belong to the lower site.
            th_b = squeezer_grams_lower(g * sig, h, uy, ud, mu)
            ms[mu], ns[mu], sq_spec[mu] = squeezer_pair(th_f, th_b, D, self.seed, call, mu, tau)
        phi_new = contract_half(e, f, ua, ux, ms[2], ms[3], ms[4])                                  # (e)
        psi_new = contract_psi(g, h, uy, ud, ns[2], ns[3], ns[4])
        self.phi = np.ascontiguousarray(phi_new.transpose(1, 2, 3, 0, 4))                           # (f) R5
        self.psi = np.ascontiguousarray(psi_new.transpose(1, 2, 3, 0, 4))
        self.lnc.append(lnc)
        self.m += 1
        self.last = dict(s=s_all, sigma=sig_all, a=a, dt=dt, core=core, x=x, y=y, sig=sig, u=(ua, ux, uy, ud),
                         efgh=(e, f, g, h), m=ms, n=ns, triad_spectra=tri_spec, squeezer_spectra=sq_spec)
        return self

    def _finish_atrg(self, a, dt, core, s_all, lnc, x, y, sig, sig_all, call):
        """Steps (d)-(f) of plain ATRG: squeezers from Gamma^ATRG = A (X sigma) | (sigma Y) Dt, contraction by Eq. 2.7-2.8."""
        D, tau = self.D, self.tau
        xs, ys = x * sig, y * sig
        yp, ysp, dp = (t.transpose(4, 1, 2, 3, 0) for t in (y, ys, dt))          # lower half: upper site Y, lower site Dt
        ms, ns, sq_spec = {}, {}, {}
        for mu in (2, 3, 4):
            th_f = atrg_grams(a, xs, mu)
            th_b = atrg_grams(ysp, dp, mu)
            ms[mu], ns[mu], sq_spec[mu] = squeezer_pair(th_f, th_b, D, self.seed, call, mu, tau)
        phi_new = contract_atrg(a, xs, ms[2], ms[3], ms[4])                       # [i1,k2,k3,k4,g]
        psi_new = contract_atrg(yp, dp, ns[2], ns[3], ns[4])                      # [g,k2,k3,k4,j1]
        self.phi = np.ascontiguousarray(phi_new.transpose(1, 2, 3, 0, 4))
        self.psi = np.ascontiguousarray(psi_new.transpose(1, 2, 3, 4, 0))
        self.lnc.append(lnc)
        self.m += 1
        self.last = dict(s=s_all, sigma=sig_all, a=a, dt=dt, core=core, x=x, y=y, sig=sig, m=ms, n=ns, squeezer_spectra=sq_spec)
        return self

    def trace(self):
        """tTr of one tensor with itself on every axis: sum_{f,g} Phi[f,g] Psi[f,g]  (Eq. 2.1 :48, V = 2^m)."""
        return float(_es("ijklg,ijklg->", self.phi, self.psi))

    def lnZ_per_site(self):
        """R8: ln Z / V = sum_j 2^-j ln c_j + 2^-m ln tTr(T^(m)) for the periodic lattice of V = 2^m sites."""
        val = sum(l * 2.0 ** (-j) for j, l in enumerate(self.lnc))
        return val + 2.0 ** (-self.m) * math.log(self.trace())

    def singular_values(self, which="sigma"):
        return self.last[which]

    def x_ratio(self):
        return x_ratio(self.phi, self.psi)


# --------------------------------------------------------------------------------------------------------
# plain ATRG (no triad split), Eq. 2.7-2.8 :104-113  -- SURVEY A9, config 5's second half
# --------------------------------------------------------------------------------------------------------
_ATRG_GRAM = {2: "iucda,alefg,ivcdb,bwefg->ulvw", 3: "icuda,aelfg,icvdb,bewfg->ulvw", 4: "icdua,aeflg,icdvb,befwg->ulvw"}


def atrg_grams(p, q, direction):
    """Gram matrix of one half of Gamma^ATRG on the doubled bond `direction`: the half is
    P[o1,u2,u3,u4,b] (upper site) . Q[b,l2,l3,l4,o2] (lower site); every index but the pair (u_d, l_d) is contracted
    with a second copy.  One einsum = the definition (reading R6)."""
    return _es(_ATRG_GRAM[direction], p, q, p, q)


def contract_atrg(p, q, s2, s3, s4):
    """Eq. 2.7 :106 (and 2.8 with the other half): R[o1,k2,k3,k4,o2] = sum P Q S2 S3 S4, squeezers S[u,l,k]."""
    return _es("iuvda,amnlg,umx,vny,dlz->ixyzg", p, q, s2, s3, s4)


def x_ratio(phi, psi):
    """Eq. 3.3 :298-303 (Gu-Wen ratio): X = (Tr A)^2 / Tr A^2 with A[k,l] = sum T[i1 i2 i3 k, i1 i2 i3 l], written on the
    factored tensor T[f,b] = sum_g Phi[f,g] Psi[b,g].  X counts the ground-state degeneracy: 2 ordered, 1 disordered."""
    a = _es("ijkag,ijkbg->ab", phi, psi)
    return float(np.trace(a) ** 2 / np.trace(a @ a))


def squeezer_grams_lower(gs, h, k_, l_, direction):
    """Gram of the lower half  L[g,j1,(j2u j2l),(j3u j3l),(j4u j4l)] =
    sum_{be,kY,kD} Gs[be,kY,j4u,g] H[j1,kD,j4l,be] K[j2u,j3u,kY] L[j2l,j3l,kD]  on the pair `direction`.
    Same staging as squeezer_grams with (H, Gs, L, K) <-> (E, F, I, J) and upper/lower legs exchanged."""
    if direction == 4:
        gg = _es("bkug,ckvg->bucv", gs, gs)
        hh = _es("jklb,jkwc->blcw", h, h)
        return _es("bucv,blcw->ulvw", gg, hh)
    gg = _es("byug,czug->bycz", gs, gs)              # sum j4u, g
    hh = _es("jdlb,jelc->bdce", h, h)                # sum j1, j4l
    gh = _es("bycz,bdce->ydze", gg, hh)              # [kY,kD,kY',kD']
    if direction == 2:
        kk = _es("ucy,vcz->uyvz", k_, k_)
        ll = _es("lcd,wce->ldwe", l_, l_)
    else:
        kk = _es("cuy,cvz->uyvz", k_, k_)
        ll = _es("cld,cwe->ldwe", l_, l_)
    tmp = _es("uyvz,ydze->uvde", kk, gh)
    return _es("uvde,ldwe->ulvw", tmp, ll)


def run(beta, h, D, oversample, seed, n_steps, n_pow=2, **kw):
    """Convenience driver: returns (list of ln Z/V after each step, list of sigma spectra, list of s spectra)."""
    o = TatrgOracle(beta, h, D, oversample, seed, n_pow=n_pow, **kw)
    lnz, sig, ss = [], [], []
    for _ in range(n_steps):
        o.step()
        lnz.append(o.lnZ_per_site())
        sig.append(o.last["sigma"].copy())
        ss.append(o.last["s"].copy())
    return lnz, sig, ss
