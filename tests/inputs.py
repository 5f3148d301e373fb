"""Seeded input generators shared by the oracle tests and the CUDA parity tests.
Holds none of the method's arithmetic: only plain random matrices / tensors with a prescribed spectrum shape."""
import numpy as np


def lowrank_plus_noise(m, n, rank, noise, seed):
    """m x n matrix with `rank` geometrically decaying singular values plus white noise of relative size `noise`."""
    rng = np.random.default_rng(seed)
    u, _ = np.linalg.qr(rng.standard_normal((m, rank)))
    v, _ = np.linalg.qr(rng.standard_normal((n, rank)))
    s = 0.7 ** np.arange(rank)
    return (u * s) @ v.T + noise * rng.standard_normal((m, n))


def random_tensor(shape, seed):
    return np.random.default_rng(seed).standard_normal(shape)


def random_psd(n, rank, seed, decay=0.6):
    """Symmetric positive semi-definite n x n of the given rank with geometric spectrum (Gram-matrix-like)."""
    rng = np.random.default_rng(seed)
    q, _ = np.linalg.qr(rng.standard_normal((n, n)))
    lam = np.zeros(n)
    lam[:rank] = decay ** np.arange(rank)
    return (q * lam) @ q.T


def configs():
    """BASELINE.json configs[0..4] as (name, beta, h, D, oversample, n_pow, seed, n_steps)."""
    return {
        "c1": (0.14, 0.0, 4, 4, 1, 1234, 16),
        "c2": (0.1497, 0.0, 8, 8, 2, 3, 40),
        "c3": (0.1497, 1e-3, 16, 16, 2, 7, 48),
        "c4": (0.1497, 0.0, 32, 32, 2, 42, 60),
        "c5": (0.1497, 0.0, 48, 48, 2, 99, 60),
    }
