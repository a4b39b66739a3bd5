"""Seeded synthetic input generators (SURVEY.md §8(d) "Synthetic inputs").

This module is shared by the tests, ``bench.py`` and ``__graft_entry__.smoke()`` to feed the SAME
values to the CUDA path and to the CPU oracle. It holds none of the skeletons' arithmetic: it only
draws numbers. It imports neither the oracle nor the CUDA binding.

The paper (arxiv 1405.2915) measures the skeletons on no public dataset (its only experiment is an
application whose inputs are not described); BASELINE.json L7-L11 fixes the synthetic
shapes and value distributions that these generators produce.

Generator: stateless, counter based.
    key  = mix64(seed * GAMMA)
    u64  = mix64(key + (i + 1) * GAMMA)             (mix64 = the splitmix64 finaliser)
    u    = (u64 >> 40) * 2**-24   in [0, 1)          exactly representable in fp32
"""
from __future__ import annotations

import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_CHUNK = 1 << 24

BASE_SEED = 14052915


def _mix64(z: np.ndarray) -> np.ndarray:
    z = z.copy()
    z ^= z >> np.uint64(30)
    z *= _M1
    z ^= z >> np.uint64(27)
    z *= _M2
    z ^= z >> np.uint64(31)
    return z


def raw_u64(seed: int, n: int, start: int = 0) -> np.ndarray:
    """u64 draw i for i in [start, start+n)."""
    with np.errstate(over="ignore"):
        key = _mix64(np.array([np.uint64(seed & 0xFFFFFFFFFFFFFFFF) * _GAMMA], dtype=np.uint64))[0]
        out = np.empty(n, dtype=np.uint64)
        for lo in range(0, n, _CHUNK):
            hi = min(n, lo + _CHUNK)
            i = np.arange(start + lo + 1, start + hi + 1, dtype=np.uint64)
            out[lo:hi] = _mix64(key + i * _GAMMA)
    return out


def _unit24(seed: int, n: int) -> np.ndarray:
    """float64 array of u = (u64 >> 40) * 2^-24 in [0,1)."""
    out = np.empty(n, dtype=np.float64)
    for lo in range(0, n, _CHUNK):
        hi = min(n, lo + _CHUNK)
        out[lo:hi] = (raw_u64(seed, hi - lo, lo) >> np.uint64(40)).astype(np.float64) * 2.0 ** -24
    return out


def uniform01_f32(seed: int, n: int) -> np.ndarray:
    """fp32 uniform on [0,1) (BJ:L9-L11 'uniform[0,1]')."""
    return _unit24(seed, n).astype(np.float32)


def uniform_pm1_f32(seed: int, n: int) -> np.ndarray:
    """fp32 uniform on [-1,1) (BJ:L7-L8 'uniform[-1,1]'); 2u-1 is exact in fp32."""
    return (2.0 * _unit24(seed, n) - 1.0).astype(np.float32)


def uniform_pm1_f64(seed: int, n: int) -> np.ndarray:
    """fp64 uniform on [-1,1) with a full 53-bit significand (fp64 element tests; not a BASELINE.json config)."""
    out = np.empty(n, dtype=np.float64)
    for lo in range(0, n, _CHUNK):
        hi = min(n, lo + _CHUNK)
        out[lo:hi] = (raw_u64(seed, hi - lo, lo) >> np.uint64(11)).astype(np.float64) * 2.0 ** -52 - 1.0
    return out


def uniform_int_i32(seed: int, n: int, hi_inclusive: int) -> np.ndarray:
    """int32 uniform on {0..hi_inclusive} (BJ:L8 'uniform[0,1000]', BJ:L11 'uniform[0,15]')."""
    out = np.empty(n, dtype=np.int32)
    m = np.uint64(hi_inclusive + 1)
    for lo in range(0, n, _CHUNK):
        hi = min(n, lo + _CHUNK)
        out[lo:hi] = ((raw_u64(seed, hi - lo, lo) >> np.uint64(32)) % m).astype(np.int32)
    return out


def full_range_i32(seed: int, n: int) -> np.ndarray:
    """int32 over the whole 32-bit range (wrap-around tests)."""
    return (raw_u64(seed, n) >> np.uint64(32)).astype(np.uint32).view(np.int32)


def positive_weights_f32(seed: int, count: int) -> np.ndarray:
    """`count` positive weights, normalised to sum 1 in fp64, then rounded to fp32 (BJ:L9;
    SURVEY §8(c).5 iv). Both the oracle and the CUDA path consume these rounded fp32 values."""
    u = _unit24(seed, count) + 2.0 ** -24
    return (u / u.sum()).astype(np.float32)


def signed_weights_f32(seed: int, count: int) -> np.ndarray:
    """Weights of mixed sign in [-1,1) (not a config; used by the tolerance tests)."""
    return uniform_pm1_f32(seed, count)


def permutation(seed: int, n: int) -> np.ndarray:
    """A seeded permutation of 0..n-1 (argsort of the draws)."""
    return np.argsort(raw_u64(seed, n), kind="stable").astype(np.int64)


def config_seed(config: int, operand: int) -> int:
    """Seed recipe of SURVEY §8(d): 14052915 + 1000*config + operand index."""
    return BASE_SEED + 1000 * config + operand
