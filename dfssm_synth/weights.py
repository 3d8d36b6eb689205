"""Seeded synthetic DF-SSM weights with the distributions BASELINE.json's config 0 states.

    scaffold signs      Bernoulli(0.5), packed 32 per uint32
    row scale           fp16(|N(0,1)| * 0.02)
    LoRA A, B           integer uniform in [-127, 127]; fp32 per-channel scales 1e-3
    A_log               log U[1, 16]
    dt_bias             softplus^-1(dt0), dt0 log-uniform in [1e-3, 1e-1]
    D                   1
    conv weights        N(0, std 0.2); conv bias 0
    norm weights        1
    embedding           integer uniform in [-127, 127]; row scale U[0.5, 1.5) / 127

`variant="varied"` is for tests only: it randomises everything BASELINE.json leaves
constant (LoRA scales, norm weights, conv bias, D) so that a kernel which ignores or
mis-indexes one of them cannot pass parity by luck.

One numpy Generator per tensor, seeded by (seed, layer, tensor index); the resulting
blob bytes are the contract, not the RNG.
"""
from __future__ import annotations

import numpy as np

from .shapes import Shape, FMT_SCAFFOLD17, FMT_LORA_INT4
from .blob import layer_tensor_specs, global_tensor_specs, write_blob, pack_levels, pack_int4


def _rng(seed: int, layer: int, tid: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([int(seed), int(layer) + 1, int(tid)])))


def _int8_uniform(g: np.random.Generator, shape) -> np.ndarray:
    return g.integers(-127, 128, size=shape, dtype=np.int8)


def _gen(name: str, dt: np.dtype, shp, g: np.random.Generator, varied: bool, fmt: int = 0) -> np.ndarray:
    base = name.split(".")[-1]
    if base == "sign":
        return g.integers(0, 1 << 32, size=shp, dtype=np.uint32).astype("<u4")
    if base == "lvl":           # 17 levels, uniform (the frozen scaffold of Eq. 3; no trained weights exist here)
        return pack_levels(g.integers(-8, 9, size=(shp[0], shp[1] * 32)))
    if base == "row_scale":     # with 17 levels the scale multiplies sum(level * q), |level| <= 8: keep the row outputs O(same)
        return (np.abs(g.standard_normal(shp)) * (0.02 / 5.0 if fmt & FMT_SCAFFOLD17 else 0.02)).astype(np.float16)
    if base in ("A", "B", "emb"):
        return _int8_uniform(g, shp)
    if base in ("A4", "B4"):
        return pack_int4(g.integers(-8, 8, size=(shp[0], shp[1] * 2)))
    if base in ("a_s", "b_s"):
        v = np.full(shp, 16e-3 if fmt & FMT_LORA_INT4 else 1e-3, dtype=np.float64)
        if varied:
            v = v * g.uniform(0.5, 1.5, size=shp)
        return v.astype(np.float32)
    if base in ("norm_w", "gnorm_w", "normf_w"):
        v = np.ones(shp, dtype=np.float64)
        if varied:
            v = g.uniform(0.5, 1.5, size=shp) * np.where(g.random(shp) < 0.1, -1.0, 1.0)
        return v.astype(np.float32)
    if base == "conv_w":
        return (g.standard_normal(shp) * 0.2).astype(np.float32)
    if base == "conv_b":
        v = np.zeros(shp, dtype=np.float64)
        if varied:
            v = g.standard_normal(shp) * 0.1
        return v.astype(np.float32)
    if base == "A_log":
        return np.log(g.uniform(1.0, 16.0, size=shp)).astype(np.float32)
    if base == "dt_bias":
        dt0 = np.exp(g.uniform(np.log(1e-3), np.log(1e-1), size=shp))
        return (dt0 + np.log(-np.expm1(-dt0))).astype(np.float32)  # inverse softplus
    if base == "D":
        v = np.ones(shp, dtype=np.float64)
        if varied:
            v = g.uniform(0.5, 1.5, size=shp)
        return v.astype(np.float32)
    if base == "emb_s":
        return (g.uniform(0.5, 1.5, size=shp) / 127.0).astype(np.float32)
    raise KeyError(name)


def make_tensors(s: Shape, seed: int, variant: str = "baseline") -> dict:
    assert variant in ("baseline", "varied")
    varied = variant == "varied"
    out = {}
    for l in range(s.n_layers):
        for tid, (name, dt, shp) in enumerate(layer_tensor_specs(s)):
            out[f"L{l}.{name}"] = _gen(name, dt, shp, _rng(seed, l, tid), varied, s.fmt)
    for tid, (name, dt, shp) in enumerate(global_tensor_specs(s)):
        out[f"G.{name}"] = _gen(name, dt, shp, _rng(seed, -1, tid), varied)
    return out


def make_blob(s: Shape, seed: int, variant: str = "baseline") -> np.ndarray:
    """uint8 array holding the canonical blob for shape `s`."""
    return write_blob(s, make_tensors(s, seed, variant))
