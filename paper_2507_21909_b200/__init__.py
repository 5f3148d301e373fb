"""paper_2507_21909_b200 -- thin Python binding of libtatrg (include/tatrg.h): the B200-native Triad-ATRG hot path.

Argument marshalling only.  Every arithmetic step runs in the hand-written sm_100a kernels behind the C ABI; PyTorch
provides device memory (the workspace) and the CUDA stream.  There is no CPU fallback: importing works without a GPU
(so that the build and the symbol table can be checked), but any compute call without the extension or without a
CUDA device raises.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtatrg.so")
_lib = None

OK, EINVAL, ENOMEM, ECUDA, ENUMERIC, ESTATE = 0, -1, -2, -3, -4, -5
OPT_POWER_ITERS, OPT_K_TRIAD, OPT_TAU, OPT_STAGE_TIMING, OPT_KEEP_TENSORS, OPT_METHOD, OPT_SUBSPACE, OPT_BOND_RANK = 1, 2, 3, 4, 5, 6, 7, 8
OPT_OVERLAP, OPT_GRAPHS, OPT_VERBOSE, OPT_DGEMM_TMA, OPT_IMPLICIT_XY, OPT_CHEBYSHEV = 9, 10, 11, 12, 13, 14
METHOD_TRIAD, METHOD_ATRG = 0, 1
SV_SIGMA, SV_S = 0, 1
STAGES = ["decompose", "qr", "rsvd", "lift", "triad", "triad_tensors", "squeezer_grams", "squeezers", "contract",
          "rotate_trace"]

_c = ctypes
_dp = _c.POINTER(_c.c_double)
_SIGNATURES = {
    "tatrg_workspace_bytes": (_c.c_size_t, [_c.c_int, _c.c_int]),
    "tatrg_workspace_bytes_atrg": (_c.c_size_t, [_c.c_int, _c.c_int]),
    "tatrg_workspace_bytes_ilo": (_c.c_size_t, [_c.c_int, _c.c_int, _c.c_int]),
    "tatrg_create": (_c.c_int, [_c.c_double, _c.c_double, _c.c_int, _c.c_int, _c.c_uint64, _c.c_void_p, _c.c_size_t,
                                _c.POINTER(_c.c_void_p)]),
    "tatrg_set_option": (_c.c_int, [_c.c_void_p, _c.c_int, _c.c_double]),
    "tatrg_step": (_c.c_int, [_c.c_void_p, _c.c_void_p]),
    "tatrg_lnZ_per_site": (_c.c_double, [_c.c_void_p]),
    "tatrg_singular_values": (_c.c_int, [_c.c_void_p, _c.c_int, _c.c_int, _dp]),
    "tatrg_x_ratio": (_c.c_int, [_c.c_void_p, _c.c_void_p, _dp]),
    "tatrg_steps_done": (_c.c_int, [_c.c_void_p]),
    "tatrg_last_error": (_c.c_char_p, [_c.c_void_p]),
    "tatrg_destroy": (None, [_c.c_void_p]),
    "tatrg_stage_ms": (_c.c_int, [_c.c_void_p, _dp]),
    "tatrg_stage_flops": (_c.c_int, [_c.c_void_p, _dp]),
    "tatrg_last_step_launches": (_c.c_longlong, [_c.c_void_p]),
    "tatrg_last_step_host_syncs": (_c.c_longlong, [_c.c_void_p]),
    "tatrg_gemm_profile": (_c.c_int, [_c.c_void_p, _dp, _dp, _c.POINTER(_c.c_longlong)]),
    "tatrg_gemm_profile_large": (_c.c_int, [_c.c_void_p, _dp, _dp, _c.POINTER(_c.c_longlong)]),
    "tatrg_permute_profile": (_c.c_int, [_c.c_void_p, _dp, _dp, _c.POINTER(_c.c_longlong)]),
    "tatrg_permute_profile_large": (_c.c_int, [_c.c_void_p, _dp, _dp, _c.POINTER(_c.c_longlong)]),
    "tatrg_workspace_peak": (_c.c_size_t, [_c.c_void_p]),
    "tatrg_get_tensor": (_c.c_longlong, [_c.c_void_p, _c.c_char_p, _dp, _c.c_longlong, _c.POINTER(_c.c_int),
                                         _c.POINTER(_c.c_longlong)]),
    "tatrg_set_state": (_c.c_int, [_c.c_void_p, _dp, _dp, _c.POINTER(_c.c_longlong)]),
    "tatrg_dgemm": (_c.c_int, [_c.c_void_p, _c.c_int, _c.c_int, _c.c_longlong, _c.c_longlong, _c.c_longlong, _c.c_double,
                               _c.c_void_p, _c.c_longlong, _c.c_void_p, _c.c_longlong, _c.c_double, _c.c_void_p,
                               _c.c_longlong, _c.c_int, _c.c_longlong, _c.c_longlong, _c.c_longlong]),
    "tatrg_dgemm_variant": (_c.c_int, [_c.c_void_p, _c.c_int, _c.c_int, _c.c_int, _c.c_longlong, _c.c_longlong, _c.c_longlong, _c.c_double,
                            _c.c_void_p, _c.c_longlong, _c.c_void_p, _c.c_longlong, _c.c_double, _c.c_void_p, _c.c_longlong,
                            _c.c_int, _c.c_longlong, _c.c_longlong, _c.c_longlong]),
    "tatrg_permute": (_c.c_int, [_c.c_void_p, _c.c_int, _c.POINTER(_c.c_longlong), _c.POINTER(_c.c_int), _c.c_void_p,
                                 _c.c_void_p]),
    "tatrg_contract": (_c.c_int, [_c.c_void_p, _c.c_char_p, _c.c_void_p, _c.POINTER(_c.c_longlong), _c.c_void_p,
                                  _c.POINTER(_c.c_longlong), _c.c_void_p, _c.c_void_p, _c.c_size_t]),
    "tatrg_philox_raw": (_c.c_int, [_c.c_void_p, _c.c_uint64, _c.c_uint32, _c.c_uint32, _c.c_uint64, _c.c_longlong,
                                    _c.c_void_p]),
    "tatrg_philox_gaussian": (_c.c_int, [_c.c_void_p, _c.c_uint64, _c.c_uint32, _c.c_uint32, _c.c_uint64, _c.c_longlong,
                                         _c.c_void_p]),
    "tatrg_eigh_work_bytes": (_c.c_size_t, [_c.c_int]),
    "tatrg_eigh": (_c.c_int, [_c.c_void_p, _c.c_int, _c.c_void_p, _c.c_void_p, _c.c_void_p, _c.c_void_p]),
    "tatrg_svd_work_bytes": (_c.c_size_t, [_c.c_int, _c.c_int]),
    "tatrg_svd": (_c.c_int, [_c.c_void_p, _c.c_int, _c.c_int, _c.c_void_p, _c.c_void_p, _c.c_void_p, _c.c_void_p,
                             _c.c_void_p]),
    "tatrg_gram_scratch_bytes": (_c.c_size_t, [_c.c_longlong, _c.c_int]),
    "tatrg_gram": (_c.c_int, [_c.c_void_p, _c.c_longlong, _c.c_int, _c.c_void_p, _c.c_void_p, _c.c_void_p]),
    "tatrg_gram_static_max_scratch_bytes": (_c.c_size_t, []),
    "tatrg_gram_static": (_c.c_int, [_c.c_void_p, _c.c_longlong, _c.c_int, _c.c_void_p, _c.c_void_p, _c.c_char_p, _c.c_size_t]),
    "tatrg_pchol_work_bytes": (_c.c_size_t, [_c.c_int]),
    "tatrg_pchol": (_c.c_int, [_c.c_void_p, _c.c_int, _c.c_void_p, _c.c_void_p, _c.c_double, _c.c_void_p, _c.POINTER(_c.c_int), _c.POINTER(_c.c_double)]),
    "tatrg_cholqr_work_bytes": (_c.c_size_t, [_c.c_int]),
    "tatrg_cholqr": (_c.c_int, [_c.c_void_p, _c.c_longlong, _c.c_int, _c.c_void_p, _c.c_void_p, _c.c_void_p, _c.c_void_p]),
    "tatrg_dot": (_c.c_int, [_c.c_void_p, _c.c_longlong, _c.c_void_p, _c.c_void_p, _c.c_void_p]),
    "tatrg_dmma_issue_rate": (_c.c_int, [_c.c_void_p, _c.c_int, _c.c_int, _dp, _c.c_void_p]),
    "tatrg_dmma_tile_rate": (_c.c_int, [_c.c_void_p, _c.c_int, _c.c_int, _dp, _c.c_void_p]),
}


class TatrgError(RuntimeError):
    pass


def lib():
    """The loaded C-ABI library.  Fails loudly when it has not been built: there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise TatrgError("libtatrg.so is missing: run `python -m paper_2507_21909_b200.build` (needs nvcc)")
        _lib = ctypes.CDLL(_LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(_lib, name)
            fn.restype, fn.argtypes = res, args
    return _lib


def exported_symbols():
    return sorted(_SIGNATURES)


def _check(rc, what, handle=None):
    if rc < 0:
        msg = lib().tatrg_last_error(handle).decode() if handle else ""
        raise TatrgError("%s failed with status %d %s" % (what, rc, msg))
    return rc


def _torch_cuda():
    import torch
    if not torch.cuda.is_available():
        raise TatrgError("no CUDA device: the Triad-ATRG path has no CPU fallback")
    return torch


def _stream_ptr(stream=None):
    torch = _torch_cuda()
    s = stream if stream is not None else torch.cuda.current_stream()
    return ctypes.c_void_p(s.cuda_stream)


def workspace_bytes(D, oversample):
    return lib().tatrg_workspace_bytes(D, oversample)


class Tatrg:
    """One 4D Ising tensor network being coarse-grained on one GPU (tatrg_create .. tatrg_destroy)."""

    def __init__(self, beta, h, D, oversample, seed, power_iters=2, K=None, tau=None, device="cuda:0", workspace=None,
                 method=METHOD_TRIAD, bond_rank=None):
        torch = _torch_cuda()
        L = lib()
        need = L.tatrg_workspace_bytes_atrg(D, oversample) if method == METHOD_ATRG else L.tatrg_workspace_bytes(D, oversample)
        if bond_rank is not None and bond_rank != D:      # ILO Triad-ATRG (section 2.3): bond_rank = r_bond * D
            need = max(need, L.tatrg_workspace_bytes_ilo(D, oversample, bond_rank)) if L.tatrg_workspace_bytes_ilo(D, oversample, bond_rank) else 0
        if need == 0:
            raise TatrgError("unsupported (D, oversample, bond_rank) = (%d, %d, %s)" % (D, oversample, bond_rank))
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.workspace = workspace if workspace is not None else torch.empty(need, dtype=torch.uint8, device=self.device)
            h_ = ctypes.c_void_p()
            rc = L.tatrg_create(beta, h, D, oversample, seed, ctypes.c_void_p(self.workspace.data_ptr()),
                                self.workspace.numel(), ctypes.byref(h_))
        if rc != OK:
            raise TatrgError("tatrg_create failed with status %d" % rc)
        self._h = h_
        self.D = D
        self.set_option(OPT_POWER_ITERS, power_iters)
        if K is not None:
            self.set_option(OPT_K_TRIAD, K)
        if tau is not None:
            self.set_option(OPT_TAU, tau)
        if method != METHOD_TRIAD:
            self.set_option(OPT_METHOD, method)
        if bond_rank is not None and bond_rank != D:
            self.set_option(OPT_BOND_RANK, bond_rank)

    def set_option(self, key, value):
        _check(lib().tatrg_set_option(self._h, key, float(value)), "tatrg_set_option", self._h)

    def step(self, stream=None):
        torch = _torch_cuda()
        with torch.cuda.device(self.device):
            _check(lib().tatrg_step(self._h, _stream_ptr(stream)), "tatrg_step", self._h)
        return self

    def lnZ_per_site(self):
        v = lib().tatrg_lnZ_per_site(self._h)
        if v != v:
            raise TatrgError("tatrg_lnZ_per_site: " + lib().tatrg_last_error(self._h).decode())
        return v

    def singular_values(self, which=SV_SIGMA, k=None):
        k = k if k is not None else 128
        out = np.zeros(k)
        n = _check(lib().tatrg_singular_values(self._h, which, k, out.ctypes.data_as(_dp)), "tatrg_singular_values", self._h)
        return out[:n]

    def x_ratio(self, stream=None):
        torch = _torch_cuda()
        x = ctypes.c_double()
        with torch.cuda.device(self.device):
            _check(lib().tatrg_x_ratio(self._h, _stream_ptr(stream), ctypes.byref(x)), "tatrg_x_ratio", self._h)
        return x.value

    def steps_done(self):
        return lib().tatrg_steps_done(self._h)

    def stage_ms(self):
        out = np.zeros(len(STAGES))
        _check(lib().tatrg_stage_ms(self._h, out.ctypes.data_as(_dp)), "tatrg_stage_ms")
        return out

    def stage_flops(self):
        out = np.zeros(len(STAGES))
        _check(lib().tatrg_stage_flops(self._h, out.ctypes.data_as(_dp)), "tatrg_stage_flops")
        return out

    def launches(self):
        return lib().tatrg_last_step_launches(self._h)

    def host_syncs(self):
        return lib().tatrg_last_step_host_syncs(self._h)

    def gemm_profile(self):
        ms, fl, n = ctypes.c_double(), ctypes.c_double(), ctypes.c_longlong()
        _check(lib().tatrg_gemm_profile(self._h, ctypes.byref(ms), ctypes.byref(fl), ctypes.byref(n)), "tatrg_gemm_profile")
        return ms.value, fl.value, n.value

    def gemm_profile_large(self):
        ms, fl, n = ctypes.c_double(), ctypes.c_double(), ctypes.c_longlong()
        _check(lib().tatrg_gemm_profile_large(self._h, ctypes.byref(ms), ctypes.byref(fl), ctypes.byref(n)), "tatrg_gemm_profile_large")
        return ms.value, fl.value, n.value

    def permute_profile(self):
        ms, by, n = ctypes.c_double(), ctypes.c_double(), ctypes.c_longlong()
        _check(lib().tatrg_permute_profile(self._h, ctypes.byref(ms), ctypes.byref(by), ctypes.byref(n)), "tatrg_permute_profile")
        return ms.value, by.value, n.value

    def permute_profile_large(self):
        ms, by, n = ctypes.c_double(), ctypes.c_double(), ctypes.c_longlong()
        _check(lib().tatrg_permute_profile_large(self._h, ctypes.byref(ms), ctypes.byref(by), ctypes.byref(n)), "tatrg_permute_profile_large")
        return ms.value, by.value, n.value

    def workspace_peak(self):
        return lib().tatrg_workspace_peak(self._h)

    def get_tensor(self, name):
        nd = ctypes.c_int()
        dims = (ctypes.c_longlong * 8)()
        n = _check(lib().tatrg_get_tensor(self._h, name.encode(), None, 0, ctypes.byref(nd), dims), "tatrg_get_tensor", self._h)
        out = np.zeros(n)
        _check(lib().tatrg_get_tensor(self._h, name.encode(), out.ctypes.data_as(_dp), n, ctypes.byref(nd), dims), "tatrg_get_tensor")
        return out.reshape([dims[i] for i in range(nd.value)])

    def set_state(self, phi, psi):
        phi = np.ascontiguousarray(phi, dtype=np.float64)
        psi = np.ascontiguousarray(psi, dtype=np.float64)
        dims = (ctypes.c_longlong * 5)(*phi.shape)
        _check(lib().tatrg_set_state(self._h, phi.ctypes.data_as(_dp), psi.ctypes.data_as(_dp), dims), "tatrg_set_state", self._h)

    def set_state_host(self, phi_t, psi_t):
        """Same as set_state, from (pinned) torch CPU float64 tensors, without a numpy copy."""
        dims = (ctypes.c_longlong * 5)(*phi_t.shape)
        _check(lib().tatrg_set_state(self._h, ctypes.cast(phi_t.data_ptr(), _dp), ctypes.cast(psi_t.data_ptr(), _dp), dims),
               "tatrg_set_state", self._h)

    def get_tensor_into(self, name, out_t):
        """Copies tensor `name` into the (pinned) torch CPU float64 tensor out_t; returns its shape."""
        nd = ctypes.c_int()
        dims = (ctypes.c_longlong * 8)()
        n = _check(lib().tatrg_get_tensor(self._h, name.encode(), ctypes.cast(out_t.data_ptr(), _dp), out_t.numel(),
                                          ctypes.byref(nd), dims), "tatrg_get_tensor", self._h)
        if n > out_t.numel():
            raise TatrgError("get_tensor_into: buffer too small")
        return [dims[i] for i in range(nd.value)]

    def close(self):
        if getattr(self, "_h", None):
            lib().tatrg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- primitives on torch CUDA tensors (float64, contiguous) -------------------------------------------------------
def _p(t):
    return ctypes.c_void_p(t.data_ptr())


def dgemm(A, B, transa=False, transb=False, alpha=1.0, beta=0.0, C=None, variant=None):
    """C = alpha*op(A)@op(B) + beta*C for 2-D or batched 3-D row-major tensors.  variant: None = the library's choice,
    0 = cp.async-fed kernels, 1 = the TMA-fed 128 x 128 tile (tatrg_dgemm_variant)."""
    torch = _torch_cuda()
    batched = A.dim() == 3
    a2, b2 = A.shape[-2:], B.shape[-2:]
    M, K = (a2[1], a2[0]) if transa else a2
    N = b2[0] if transb else b2[1]
    nb = A.shape[0] if batched else 1
    if C is None:
        C = torch.empty((nb, M, N) if batched else (M, N), dtype=torch.float64, device=A.device)
    rest = (int(transa), int(transb), M, N, K, alpha, _p(A), a2[1], _p(B), b2[1], beta, _p(C), N,
            nb, a2[0] * a2[1] if batched else 0, b2[0] * b2[1] if batched else 0, M * N if batched else 0)
    if variant is None:
        _check(lib().tatrg_dgemm(_stream_ptr(), *rest), "tatrg_dgemm")
    else:
        _check(lib().tatrg_dgemm_variant(_stream_ptr(), int(variant), *rest), "tatrg_dgemm_variant")
    return C


def permute(x, perm):
    torch = _torch_cuda()
    out = torch.empty([x.shape[p] for p in perm], dtype=torch.float64, device=x.device)
    dims = (ctypes.c_longlong * x.dim())(*x.shape)
    pm = (ctypes.c_int * x.dim())(*perm)
    _check(lib().tatrg_permute(_stream_ptr(), x.dim(), dims, pm, _p(x), _p(out)), "tatrg_permute")
    return out


def contract(spec, A, B):
    torch = _torch_cuda()
    ins, out = spec.split("->")
    sa, sb = ins.split(",")
    ext = {}
    for s, t in ((sa, A), (sb, B)):
        for ch, d in zip(s, t.shape):
            ext[ch] = d
    C = torch.empty([ext[ch] for ch in out], dtype=torch.float64, device=A.device)
    nbytes = 8 * (A.numel() + B.numel() + C.numel()) + (64 << 20)
    scratch = torch.empty(nbytes, dtype=torch.uint8, device=A.device)
    da = (ctypes.c_longlong * A.dim())(*A.shape)
    db = (ctypes.c_longlong * B.dim())(*B.shape)
    _check(lib().tatrg_contract(_stream_ptr(), spec.encode(), _p(A), da, _p(B), db, _p(C), _p(scratch), nbytes), "tatrg_contract")
    torch.cuda.current_stream().synchronize()
    return C


def philox_raw(seed, call, stream_id, start, count):
    torch = _torch_cuda()
    out = torch.empty(4 * count, dtype=torch.int32, device="cuda")
    _check(lib().tatrg_philox_raw(_stream_ptr(), seed, call, stream_id, start, count, _p(out)), "tatrg_philox_raw")
    return out.cpu().numpy().view(np.uint32).reshape(count, 4)


def philox_gaussian(seed, call, stream_id, start, count):
    torch = _torch_cuda()
    out = torch.empty(count, dtype=torch.float64, device="cuda")
    _check(lib().tatrg_philox_gaussian(_stream_ptr(), seed, call, stream_id, start, count, _p(out)), "tatrg_philox_gaussian")
    return out.cpu().numpy()


def eigh(G):
    """(lam descending, Vt with eigenvectors as rows) of a symmetric matrix (torch CUDA float64)."""
    torch = _torch_cuda()
    n = G.shape[0]
    g = G.clone().contiguous()
    lam = torch.empty(n, dtype=torch.float64, device=G.device)
    vt = torch.empty((n, n), dtype=torch.float64, device=G.device)
    work = torch.empty(lib().tatrg_eigh_work_bytes(n), dtype=torch.uint8, device=G.device)
    _check(lib().tatrg_eigh(_stream_ptr(), n, _p(g), _p(lam), _p(vt), _p(work)), "tatrg_eigh")
    return lam, vt


def svd_rows(X):
    """X = Vacc^T diag(s) Ut for a small matrix (rows orthogonalised by one-sided Jacobi)."""
    torch = _torch_cuda()
    nv, ln = X.shape
    x = X.contiguous()
    s = torch.empty(nv, dtype=torch.float64, device=X.device)
    ut = torch.empty((nv, ln), dtype=torch.float64, device=X.device)
    va = torch.empty((nv, nv), dtype=torch.float64, device=X.device)
    work = torch.empty(lib().tatrg_svd_work_bytes(nv, ln), dtype=torch.uint8, device=X.device)
    _check(lib().tatrg_svd(_stream_ptr(), nv, ln, _p(x), _p(s), _p(ut), _p(va), _p(work)), "tatrg_svd")
    return s, ut, va


def gram(X):
    """X^T X (torch CUDA float64, m x n) through the symmetric mode of the DGEMM (lower tiles + mirror)."""
    torch = _torch_cuda()
    m, n = X.shape
    x = X.contiguous()
    g = torch.empty((n, n), dtype=torch.float64, device=X.device)
    nb = lib().tatrg_gram_scratch_bytes(m, n)
    scratch = torch.empty(max(nb, 8), dtype=torch.uint8, device=X.device)
    _check(lib().tatrg_gram(_stream_ptr(), m, n, _p(x), _p(g), _p(scratch)), "tatrg_gram")
    return g


def gram_static(X, out=None):
    """X^T X like gram(), through tatrg_gram_static: no device allocation inside the call (split-K scratch in the library's
    16 MiB static array).  `out` (n x n, float64, CUDA) lets the caller provide the result buffer too."""
    torch = _torch_cuda()
    m, n = X.shape
    x = X.contiguous()
    g = out if out is not None else torch.empty((n, n), dtype=torch.float64, device=X.device)
    err = ctypes.create_string_buffer(512)
    rc = lib().tatrg_gram_static(_stream_ptr(), m, n, _p(x), _p(g), err, 512)
    if rc < 0:
        raise TatrgError("tatrg_gram_static failed with status %d: %s" % (rc, err.value.decode()))
    return g


def cholqr(X):
    """X = Q R by Cholesky QR (torch CUDA float64, m x n with m >= n): (Q, R), R upper triangular with positive diagonal."""
    torch = _torch_cuda()
    m, n = X.shape
    x = X.clone().contiguous()
    q = torch.empty((m, n), dtype=torch.float64, device=X.device)
    r = torch.empty((n, n), dtype=torch.float64, device=X.device)
    work = torch.empty(lib().tatrg_cholqr_work_bytes(n), dtype=torch.uint8, device=X.device)
    _check(lib().tatrg_cholqr(_stream_ptr(), m, n, _p(x), _p(q), _p(r), _p(work)), "tatrg_cholqr")
    return q, r


def pchol(G, tol_rel=1e-14):
    """G = L L^T + S by truncated Cholesky with diagonal pivoting (torch CUDA float64, n x n): (L[:, :rank], rank, tr S / tr G)."""
    torch = _torch_cuda()
    n = G.shape[0]
    g = G.contiguous()
    L = torch.zeros((n, n), dtype=torch.float64, device=G.device)
    work = torch.empty(lib().tatrg_pchol_work_bytes(n), dtype=torch.uint8, device=G.device)
    rank, resid = ctypes.c_int(), ctypes.c_double()
    _check(lib().tatrg_pchol(_stream_ptr(), n, _p(g), _p(L), tol_rel, _p(work), ctypes.byref(rank), ctypes.byref(resid)), "tatrg_pchol")
    return L[:, :rank.value], rank.value, resid.value


def dot(x, y):
    torch = _torch_cuda()
    res = torch.empty(1200, dtype=torch.float64, device=x.device)
    _check(lib().tatrg_dot(_stream_ptr(), x.numel(), _p(x), _p(y), _p(res)), "tatrg_dot")
    return float(res[0].item())


def dmma_tile_rate(iters=5000, order=0):
    """DMMA rate of the DGEMM register tile (8 x 4 atoms per warp, one CTA per SM) without memory traffic, TFLOP/s."""
    torch = _torch_cuda()
    scratch = torch.zeros(8, dtype=torch.float64, device="cuda")
    out = ctypes.c_double()
    _check(lib().tatrg_dmma_tile_rate(_stream_ptr(), iters, order, ctypes.byref(out), _p(scratch)), "tatrg_dmma_tile_rate")
    return out.value


def dmma_issue_rate(iters=20000, ctas_per_sm=2):
    """Register-resident DMMA issue rate of the device in TFLOP/s (calibration of the FP64 tensor ceiling)."""
    torch = _torch_cuda()
    scratch = torch.zeros(8, dtype=torch.float64, device="cuda")
    out = ctypes.c_double()
    _check(lib().tatrg_dmma_issue_rate(_stream_ptr(), iters, ctas_per_sm, ctypes.byref(out), _p(scratch)), "tatrg_dmma_issue_rate")
    return out.value
