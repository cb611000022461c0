"""Philox4x32-10 for the *primary generator stream* only.

The transport RNG lives twice elsewhere (CUDA library, oracle), each written on its own;
this numpy version only draws primary attributes, which are then plain inputs for both.
"""
import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = np.uint32(0x9E3779B9)
_W1 = np.uint32(0xBB67AE85)
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)


def philox4x32_10(ctr, key):
    """ctr: (...,4) uint32, key: (...,2) uint32 -> (...,4) uint32."""
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    c0, c1, c2, c3 = (c[..., i].copy() for i in range(4))
    k0, k1 = k[..., 0].copy(), k[..., 1].copy()
    with np.errstate(over="ignore"):
        for _ in range(10):
            p0 = c0.astype(np.uint64) * _M0
            p1 = c2.astype(np.uint64) * _M1
            n0 = ((p1 >> _S32) & _MASK).astype(np.uint32) ^ c1 ^ k0
            n1 = (p1 & _MASK).astype(np.uint32)
            n2 = ((p0 >> _S32) & _MASK).astype(np.uint32) ^ c3 ^ k1
            n3 = (p0 & _MASK).astype(np.uint32)
            c0, c1, c2, c3 = n0, n1, n2, n3
            k0 = (k0 + _W0).astype(np.uint32)
            k1 = (k1 + _W1).astype(np.uint32)
    return np.stack([c0, c1, c2, c3], axis=-1)


def to_uniform(hi, lo):
    """53-bit uniform in (0,1), open at both ends (R2)."""
    hi = np.asarray(hi, dtype=np.uint64)
    lo = np.asarray(lo, dtype=np.uint64)
    mant = ((hi >> np.uint64(5)) << np.uint64(26)) + (lo >> np.uint64(6))
    return (mant.astype(np.float64) + 0.5) * 2.0 ** -53


def uniforms(event, seed, track_id, step, n):
    """First n uniforms of the stream (event, track_id, step): shape (n,)."""
    nb = (n + 1) // 2
    ctr = np.zeros((nb, 4), dtype=np.uint32)
    ctr[:, 0] = np.uint32(track_id & 0xFFFFFFFF)
    ctr[:, 1] = np.uint32((track_id >> 32) & 0xFFFFFFFF)
    ctr[:, 2] = np.uint32(step)
    ctr[:, 3] = np.arange(nb, dtype=np.uint32)
    key = np.zeros((nb, 2), dtype=np.uint32)
    key[:, 0] = np.uint32(event)
    key[:, 1] = np.uint32(seed)
    w = philox4x32_10(ctr, key)
    u = np.empty(2 * nb)
    u[0::2] = to_uniform(w[:, 0], w[:, 1])
    u[1::2] = to_uniform(w[:, 2], w[:, 3])
    return u[:n]
