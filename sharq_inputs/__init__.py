"""Seeded synthetic inputs for SharQ.

Serves both the oracle and the CUDA path; holds none of the method's arithmetic: it only draws
random numbers, places outliers and rounds fp32 to bf16 bit patterns (uint16).  The paper's
activations come from Llama / Qwen / Wan2.2 models and public evaluation suites that are not
available here; these tensors stand in for them with the shapes and the
outlier structure BASELINE.json's configs prescribe ("a small number of large-magnitude
outliers").
"""
from __future__ import annotations

import numpy as np

BASE_SEED = 26587
TENSOR_X, TENSOR_GAMMA, TENSOR_W, TENSOR_CHANNELS, TENSOR_SPIKES, TENSOR_ROUTER, TENSOR_BETA = range(7)


def seed_for(config: int, tensor_id: int, extra: int = 0) -> int:
    return BASE_SEED * 1000 + 10 * config + tensor_id + 1000003 * extra


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(seed))


def to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit patterns (uint16), round-to-nearest-even; inputs are finite."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    return ((u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(u16: np.ndarray) -> np.ndarray:
    return (np.asarray(u16, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def activations(T: int, K: int, config: int = 1, outlier_mult: float = 50.0, extra: int = 0,
                n_outlier_channels: int = 8, spike_prob: float = 1e-3, spike_mult: float = 20.0) -> np.ndarray:
    """X bf16 bits [T, K]: N(0,1); `n_outlier_channels` seeded channels x outlier_mult; a
    Bernoulli(spike_prob) set of entries x spike_mult."""
    x = _rng(seed_for(config, TENSOR_X, extra)).standard_normal((T, K), dtype=np.float32)
    ch = _rng(seed_for(config, TENSOR_CHANNELS, extra)).choice(K, size=min(n_outlier_channels, K), replace=False)
    x[:, ch] *= np.float32(outlier_mult)
    spikes = _rng(seed_for(config, TENSOR_SPIKES, extra)).random((T, K), dtype=np.float32) < spike_prob
    x[spikes] *= np.float32(spike_mult)
    return to_bf16_bits(x)


def gamma(K: int, config: int = 1) -> np.ndarray:
    g = _rng(seed_for(config, TENSOR_GAMMA)).random(K, dtype=np.float32) + np.float32(0.5)
    return to_bf16_bits(g)


def beta(K: int, config: int = 1) -> np.ndarray:
    b = _rng(seed_for(config, TENSOR_BETA)).standard_normal(K, dtype=np.float32) * np.float32(0.1)
    return to_bf16_bits(b)


def weight(D: int, K: int, config: int = 1, extra: int = 0, std: float = 0.02) -> np.ndarray:
    w = _rng(seed_for(config, TENSOR_W, extra)).standard_normal((D, K), dtype=np.float32) * np.float32(std)
    return to_bf16_bits(w)


def moe_routing(tokens: int = 4096, experts: int = 128, top_k: int = 8, config: int = 5):
    """Seeded softmax router over N(0,1) logits; top-k with ties to the lower expert id.
    Returns (expert_ids [tokens, top_k] int32, offsets [experts+1] int32, order [tokens*top_k]
    int32 = routed (token, slot) pairs sorted by expert, stable)."""
    logits = _rng(seed_for(config, TENSOR_ROUTER)).standard_normal((tokens, experts), dtype=np.float32)
    p = np.exp(logits - logits.max(axis=1, keepdims=True))
    p /= p.sum(axis=1, keepdims=True)
    ids = np.argsort(-p, axis=1, kind="stable")[:, :top_k].astype(np.int32)
    flat = ids.reshape(-1)
    order = np.argsort(flat, kind="stable").astype(np.int32)
    counts = np.bincount(flat, minlength=experts)
    offsets = np.zeros(experts + 1, dtype=np.int32)
    offsets[1:] = np.cumsum(counts)
    return ids, offsets, order
