"""Counter-based uniform / normal generator keyed by (seed, stream, index).

Reading G25: "from seed" in BASELINE.json:configs is realised as a
stateless hash so any slice of any coordinate can be regenerated independently and in
any chunking.  The hash is the splitmix64 finaliser applied to a Weyl sequence; normals
come from Box-Muller on two independent streams.  Values are produced ONCE on the host
and handed as bytes to both the oracle and the CUDA path.
"""
from __future__ import annotations

import numpy as np

SEED_BASE = 1710073500  # + config index (G25)

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_K_SEED = np.uint64(0xD1342543DE82EF95)
_K_STREAM = np.uint64(0xA24BAED4963EE407)
_CHUNK = 1 << 22


def _mix(z: np.ndarray) -> np.ndarray:
    z ^= z >> np.uint64(30)
    z *= _M1
    z ^= z >> np.uint64(27)
    z *= _M2
    z ^= z >> np.uint64(31)
    return z


def _uniform_chunk(seed: int, stream: int, lo: int, hi: int) -> np.ndarray:
    with np.errstate(over="ignore"):
        i = np.arange(lo + 1, hi + 1, dtype=np.uint64)
        z = i * _GOLDEN
        z += np.uint64(seed & 0xFFFFFFFFFFFFFFFF) * _K_SEED
        z += np.uint64(stream) * _K_STREAM
        z = _mix(z)
        z += _GOLDEN
        z = _mix(z)
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def uniform01(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    """n uniforms in [0,1) for indices start..start+n-1 of (seed, stream)."""
    out = np.empty(n, dtype=np.float64)
    for lo in range(0, n, _CHUNK):
        hi = min(n, lo + _CHUNK)
        out[lo:hi] = _uniform_chunk(seed, stream, start + lo, start + hi)
    return out


def normal01(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    """n standard normals (Box-Muller, no truncation) for (seed, stream)."""
    out = np.empty(n, dtype=np.float64)
    for lo in range(0, n, _CHUNK):
        hi = min(n, lo + _CHUNK)
        u1 = _uniform_chunk(seed, 2 * stream + 1000, start + lo, start + hi)
        u2 = _uniform_chunk(seed, 2 * stream + 1001, start + lo, start + hi)
        np.subtract(1.0, u1, out=u1)          # (0,1]
        np.log(u1, out=u1)
        u1 *= -2.0
        np.sqrt(u1, out=u1)
        u2 *= 2.0 * np.pi
        np.cos(u2, out=u2)
        u1 *= u2
        out[lo:hi] = u1
    return out
