"""oracle/philox.py -- TEST INFRASTRUCTURE ONLY (part of the CPU oracle; never imported by the product path).

Philox4x32-10 counter-based generator (Salmon et al., "Parallel random numbers: as easy as 1, 2, 3", SC'11)
restated in numpy, and the Gaussian stream the Triad-ATRG oracle draws its RSVD test tensor from.

PAPER.md only says "Omega is a random tensor" (App. A, :371); BASELINE.json fixes "Gaussian test matrices from
Philox4x32-10".  The stream layout is reading R11 of DESIGN.md:

    key     = (seed & 0xffffffff, seed >> 32)
    counter = (e & 0xffffffff, e >> 32, call, stream)     e = element index, call = RG step, stream = 0 Omega / 1 rho
    (x0,x1,x2,x3) = philox4x32_10(counter, key)
    u1 = ((x0 >> 6) * 2^27 + (x1 >> 5) + 0.5) * 2^-53      in (0,1]
    u2 = ((x2 >> 6) * 2^27 + (x3 >> 5) + 0.5) * 2^-53
    z  = sqrt(-2 ln u1) * cos(2 pi u2)                     one Gaussian per counter

The CUDA path implements the same generator independently (no shared code); integers must agree bit for bit,
Gaussians to a few ulp (libm vs CUDA math).
"""
import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = 0x9E3779B9
_W1 = 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)

STREAM_OMEGA = 0
STREAM_RHO = 1


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Ten rounds of Philox-4x32.  All arguments are array-likes of 32-bit values; returns four uint32 arrays."""
    c0 = np.asarray(c0, dtype=np.uint64) & _MASK
    c1 = np.asarray(c1, dtype=np.uint64) & _MASK
    c2 = np.asarray(c2, dtype=np.uint64) & _MASK
    c3 = np.asarray(c3, dtype=np.uint64) & _MASK
    c0, c1, c2, c3 = np.broadcast_arrays(c0, c1, c2, c3)
    k0 = int(k0) & 0xFFFFFFFF
    k1 = int(k1) & 0xFFFFFFFF
    for _ in range(10):
        p0 = _M0 * c0                      # 32x32 -> 64 bit products
        p1 = _M1 * c2
        hi0, lo0 = p0 >> _S32, p0 & _MASK
        hi1, lo1 = p1 >> _S32, p1 & _MASK
        n0 = hi1 ^ c1 ^ np.uint64(k0)
        n1 = lo1
        n2 = hi0 ^ c3 ^ np.uint64(k1)
        n3 = lo0
        c0, c1, c2, c3 = n0, n1, n2, n3
        k0 = (k0 + _W0) & 0xFFFFFFFF       # key schedule (Weyl sequence)
        k1 = (k1 + _W1) & 0xFFFFFFFF
    return (c0.astype(np.uint32), c1.astype(np.uint32), c2.astype(np.uint32), c3.astype(np.uint32))


def uniforms53(x0, x1):
    """(x0>>6)*2^27 + (x1>>5) is a 53-bit integer k; (k + 0.5) 2^-53 lies in (0,1]: never 0 (the logarithm is finite); for
    k = 2^53 - 1 the sum rounds to 2^53 and u = 1 exactly, which gives z = 0."""
    a = (np.asarray(x0, dtype=np.uint64) >> np.uint64(6)).astype(np.float64)
    b = (np.asarray(x1, dtype=np.uint64) >> np.uint64(5)).astype(np.float64)
    return (a * 134217728.0 + b + 0.5) * (1.0 / 9007199254740992.0)


def gaussians(seed, call, stream, start, count):
    """z[e] for e = start .. start+count-1 (float64), one Box-Muller cosine branch per counter."""
    e = np.arange(start, start + count, dtype=np.uint64)
    x0, x1, x2, x3 = philox4x32_10(e & _MASK, e >> _S32, call, stream, seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)
    u1 = uniforms53(x0, x1)
    u2 = uniforms53(x2, x3)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
