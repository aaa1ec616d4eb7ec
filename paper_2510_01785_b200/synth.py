"""Seeded synthetic inputs shared by the CUDA path's tests/bench and the CPU oracle's tests.

This module holds NONE of the method's arithmetic (no geometry, no Legendre, no DFT): only a
counter-based random generator and the workload recipes of BASELINE.json's configs (DESIGN.md
"Input recipe").  Values depend only on (seed, tag, element index): a fixed 64-bit integer mix
(splitmix64 finaliser) -> two 53-bit uniforms -> Box-Muller, so they are identical on any
machine, thread count or library version.
"""
from __future__ import annotations

import numpy as np

_MASK = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on uint64 arrays (wrap-around arithmetic)."""
    x = x.astype(np.uint64, copy=True)
    with np.errstate(over="ignore"):
        x += np.uint64(0x9E3779B97F4A7C15)
        x ^= x >> np.uint64(30)
        x *= np.uint64(0xBF58476D1CE4E5B9)
        x ^= x >> np.uint64(27)
        x *= np.uint64(0x94D049BB133111EB)
        x ^= x >> np.uint64(31)
    return x


def _key(seed: int, tag: int) -> np.uint64:
    k = _mix64(np.array([seed & 0xFFFFFFFFFFFFFFFF], dtype=np.uint64))
    with np.errstate(over="ignore"):
        k = _mix64(k ^ (np.uint64(tag) * np.uint64(0xD1342543DE82EF95)))
    return k[0]


def uniform(seed: int, tag: int, n: int, offset: int = 0) -> np.ndarray:
    """n uniforms in (0, 1), element i depends only on (seed, tag, offset + i)."""
    idx = np.arange(offset, offset + n, dtype=np.uint64)
    with np.errstate(over="ignore"):
        bits = _mix64(idx * np.uint64(0x2545F4914F6CDD1D) ^ _key(seed, tag))
    return ((bits >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed: int, tag: int, n: int, offset: int = 0) -> np.ndarray:
    """n standard normals by Box-Muller from two independent uniform streams."""
    out = np.empty(n, dtype=np.float64)
    chunk = 1 << 24
    for s in range(0, n, chunk):
        c = min(chunk, n - s)
        u1 = uniform(seed, 2 * tag, c, offset + s)
        u2 = uniform(seed, 2 * tag + 1, c, offset + s)
        out[s:s + c] = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    return out


# ---------------------------------------------------------------------------- layout helpers
# (index bookkeeping of the C-ABI's packed alm layout; no transform arithmetic)

def npix(nside: int) -> int:
    return 12 * nside * nside


def alm_count(lmax: int, mmax: int) -> int:
    return (mmax + 1) * (lmax + 1) - mmax * (mmax + 1) // 2


def alm_lm(lmax: int, mmax: int):
    """(l, m) of every packed coefficient, m-major: index(l,m) = m(2 lmax+1-m)/2 + l."""
    ms = np.repeat(np.arange(mmax + 1), lmax + 1 - np.arange(mmax + 1))
    start = np.arange(mmax + 1) * (2 * lmax + 1 - np.arange(mmax + 1)) // 2 + np.arange(mmax + 1)
    ls = np.arange(alm_count(lmax, mmax)) - np.repeat(start, lmax + 1 - np.arange(mmax + 1)) + ms
    return ls.astype(np.int64), ms.astype(np.int64)


# ---------------------------------------------------------------------------- workload recipes

def gaussian_map(seed: int, nside: int, batch: int = 1, tag: int = 1) -> np.ndarray:
    """[batch, npix] i.i.d. N(0,1) pixels (configs 1 and 3)."""
    n = npix(nside)
    return normal(seed, tag, batch * n).reshape(batch, n)


def powerlaw_alm(seed: int, lmax: int, mmax: int, batch: int = 1, tag: int = 2) -> np.ndarray:
    """[batch, nalm] complex Gaussian with E|a_lm|^2 = (l+1)^-2; m>0: Re, Im ~ N(0, (l+1)^-2 / 2);
    m = 0: real N(0, (l+1)^-2), Im = 0 (configs 1, 2, 4, 5)."""
    na = alm_count(lmax, mmax)
    ls, ms = alm_lm(lmax, mmax)
    re = normal(seed, tag, batch * na).reshape(batch, na)
    im = normal(seed, tag + 100, batch * na).reshape(batch, na)
    sig = 1.0 / (ls + 1.0)
    scale = np.where(ms == 0, sig, sig / np.sqrt(2.0))
    out = (re + 1j * im) * scale
    out[:, ms == 0] = out[:, ms == 0].real
    return out


def white_alm(seed: int, lmax: int, mmax: int, batch: int = 1, tag: int = 3) -> np.ndarray:
    """[batch, nalm] complex N(0,1) cotangents (Re, Im ~ N(0,1)); Im a_l0 is left non-zero on purpose:
    the C-ABI must ignore it."""
    na = alm_count(lmax, mmax)
    re = normal(seed, tag, batch * na).reshape(batch, na)
    im = normal(seed, tag + 100, batch * na).reshape(batch, na)
    return re + 1j * im


def ring_weights(seed: int, nside: int, tag: int = 4) -> np.ndarray:
    """Synthetic non-symmetric ring weights w_i = (4 pi / Npix)(1 + 0.1 u_i), u ~ U(-1,1)."""
    u = 2.0 * uniform(seed, tag, 4 * nside - 1) - 1.0
    return (4.0 * np.pi / npix(nside)) * (1.0 + 0.1 * u)


CONFIGS = {
    # name: BASELINE.json configs[k]
    "cfg1": dict(nside=32, lmax=64, mmax=64, batch=1, dtype="f64", seed=101),
    "cfg2": dict(nside=256, lmax=511, mmax=511, batch=1, dtype="f64", seed=202),
    "cfg3": dict(nside=64, lmax=128, mmax=128, batch=256, dtype="f32", seed=303),
    "cfg4": dict(nside=1024, lmax=2047, mmax=2047, batch=8, dtype="f32", seed=404),
    "cfg5": dict(nside=4096, lmax=8191, mmax=8191, batch=1, dtype="f64", seed=505),
}
