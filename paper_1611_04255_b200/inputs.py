"""Seeded synthetic inputs shared by the tests, bench.py and the smoke check.

This module holds NONE of the method's arithmetic: it only draws the random
vectors that stand in for the paper's CNN gradient / parameter messages
(AlexNet, GoogLeNet on ImageNet; VGG-16 is BASELINE.json's
addition).  Sizes and value scales only -- the real networks, weights and
dataset are not used.  Both the CPU oracle (through the tests) and the CUDA
path are fed the arrays produced here, byte for byte.

Recipe: rank r of config c draws from
``numpy.random.default_rng([c, r])``; uniform = ``random(float32) * 2 - 1``
(exact in fp32), normal = ``standard_normal(float32) * float32(sigma)``.
"""
from __future__ import annotations

import numpy as np

# BASELINE.json "configs", in order (index = seed).
CONFIGS = {
    0: dict(name="cfg0_P4_1Mi_uniform", P=4, n=1_048_576, block=65_536, dist="uniform",
            ops=("allreduce", "reduce", "broadcast"), root=0),
    1: dict(name="cfg1_P6_alexnet_61M", P=6, n=61_000_000, block=65_536, dist="normal",
            sigma=1e-3, ops=("allreduce",),
            block_sweep=(16_384, 65_536, 131_072, 262_144, 524_288, 1_048_576)),
    2: dict(name="cfg2_P8_googlenet_7M_sgd", P=8, n=7_000_000, block=65_536, dist="normal",
            sigma=1e-2, w_sigma=0.05, lr=0.01, iters=100, ops=("bsp_sgd_step",), root=0),
    3: dict(name="cfg3_sweep", P=(2, 4, 8, 16), n=tuple(2 ** e for e in range(10, 28)),
            block=65_536, dist="uniform", ops=("broadcast", "reduce", "allreduce")),
    4: dict(name="cfg4_P16_vgg16_138M", P=16, n=138_000_000, block=262_144, dist="normal",
            sigma=1e-3, ops=("allreduce",)),
}


def uniform(seed, rank: int, n: int) -> np.ndarray:
    """U[-1, 1) float32 vector for (seed, rank)."""
    rng = np.random.default_rng([*np.atleast_1d(seed).tolist(), rank])
    x = rng.random(n, dtype=np.float32)
    x *= np.float32(2.0)
    x -= np.float32(1.0)
    return x


def normal(seed, rank: int, n: int, sigma: float) -> np.ndarray:
    """N(0, sigma^2) float32 vector for (seed, rank)."""
    rng = np.random.default_rng([*np.atleast_1d(seed).tolist(), rank])
    x = rng.standard_normal(n, dtype=np.float32)
    x *= np.float32(sigma)
    return x


def rank_vectors(seed, P: int, n: int, dist: str = "uniform", sigma: float = 1.0):
    """The P virtual ranks' message vectors."""
    if dist == "uniform":
        return [uniform(seed, r, n) for r in range(P)]
    if dist == "normal":
        return [normal(seed, r, n, sigma) for r in range(P)]
    raise ValueError(f"unknown distribution {dist!r}")


def sgd_inputs(seed, P: int, n: int, g_sigma: float = 1e-2, w_sigma: float = 0.05):
    """Config-2 style inputs: per-rank gradients and one shared weight vector
    (rank index P in the seed sequence), copied into P replicas."""
    grads = [normal(seed, r, n, g_sigma) for r in range(P)]
    w = normal(seed, P, n, w_sigma)
    weights = [w.copy() for _ in range(P)]
    return grads, weights


def small_integers(seed, rank: int, n: int, lo: int = -8, hi: int = 8) -> np.ndarray:
    """Small-integer-valued float32 vector: every summation order is exact."""
    rng = np.random.default_rng([*np.atleast_1d(seed).tolist(), rank])
    return rng.integers(lo, hi + 1, size=n).astype(np.float32)


# ---- element types other than fp32 (U21) --------------------------------------------------------
# f16 vectors are numpy float16 arrays, bf16 vectors numpy uint16 arrays of bit patterns (numpy has no bfloat16),
# f64 vectors numpy float64.  The 16-bit values are drawn as BIT PATTERNS (random sign, exponent field in a band,
# random fraction), so nothing here rounds or converts a floating-point value.
DT_F32, DT_F16, DT_BF16, DT_F64 = 0, 1, 2, 3
DT_NAMES = {DT_F32: "f32", DT_F16: "f16", DT_BF16: "bf16", DT_F64: "f64"}
DT_NUMPY = {DT_F32: np.float32, DT_F16: np.float16, DT_BF16: np.uint16, DT_F64: np.float64}
_FRAC_BITS = {DT_F16: 10, DT_BF16: 7}
_EXP_BIAS = {DT_F16: 15, DT_BF16: 127}


def typed_vector(seed, rank: int, n: int, dt: int, kind: str = "sum") -> np.ndarray:
    """One rank's vector of element type `dt`.  kind "sum": magnitudes in [2^-4, 2) (sums over 32 ranks stay finite
    in every type); "prod": magnitudes in [0.5, 2) (products wander by a few binades, now and then out of f16's range
    -- both sides then produce the same infinities or zeros); "wide": any finite exponent, subnormals included."""
    rng = np.random.default_rng([*np.atleast_1d(seed).tolist(), rank, dt])
    if dt == DT_F32 or dt == DT_F64:
        ftype = np.float32 if dt == DT_F32 else np.float64
        if kind == "prod":
            x = rng.random(n, dtype=ftype) + ftype(0.5)          # [0.5, 1.5)
            x *= rng.integers(0, 2, size=n).astype(ftype) * ftype(2) - ftype(1)
            return x
        x = rng.random(n, dtype=ftype)
        x *= ftype(2.0)
        x -= ftype(1.0)
        return x
    fb, bias = _FRAC_BITS[dt], _EXP_BIAS[dt]
    if kind == "sum":
        e = rng.integers(bias - 4, bias + 1, size=n)
    elif kind == "prod":
        e = rng.integers(bias - 1, bias + 1, size=n)
    elif kind == "wide":
        e = rng.integers(0, 2 * bias + 1, size=n)                # 0 = zero / subnormal ... 2 * bias = largest binade
    else:
        raise ValueError(kind)
    bits = (rng.integers(0, 2, size=n) << 15) | (e << fb) | rng.integers(0, 1 << fb, size=n)
    bits = bits.astype(np.uint16)
    return bits.view(np.float16) if dt == DT_F16 else bits


def typed_rank_vectors(seed, P: int, n: int, dt: int, kind: str = "sum"):
    return [typed_vector(seed, r, n, dt, kind) for r in range(P)]
