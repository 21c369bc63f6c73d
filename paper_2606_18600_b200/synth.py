"""Seeded synthetic inputs shared by the oracle-side and CUDA-side callers (tests, bench, smoke).

This module holds NONE of the method's arithmetic: it only draws random numbers, shapes them like the paper's
workloads and lays out block tables.  The recipe is stated in DESIGN.md "Input recipe" (= SURVEY.md §8(d)):

* lengths: ``clip(round(exp(N(ln median, 0.7))), lo, hi)`` from ``numpy.random.default_rng(seed)`` — sigma 0.7
  is the value for which a median of 600 gives the paper's mean input 763 (reading A17);
* tensors: per-tensor ``torch.Generator().manual_seed(seed*1_000_003 + 64*layer + tensor_idx)``,
  ``randn * sigma -> bf16``; projection / embedding / lm_head matrices N(0, 0.02) (BASELINE.json configs),
  gains 1 + N(0, 0.02), hidden inputs N(0,1), random KV pre-fill N(0,1) (reading A21);
* block tables: a random permutation of the pool's pages (BASELINE.json configs: "shuffled block table").

These stand in for the Azure Conversation trace and the Llama-3.1-70B / Qwen3-32B checkpoints the paper measures
with, neither of which is available offline.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import torch

SIGMA = 0.7
PAGE = 16

_TENSORS = ("ln1", "wq", "wk", "wv", "q_norm", "k_norm", "wo", "ln2", "w_gate", "w_up", "w_down")


@dataclass(frozen=True)
class ModelShape:
    name: str
    hidden: int
    n_q: int
    n_kv: int
    d: int
    ffn: int
    n_layers: int          # layers in the stage
    eps: float
    theta: float
    qk_norm: int
    vocab: int

    @property
    def hq(self):
        return self.n_q * self.d

    @property
    def hkv(self):
        return self.n_kv * self.d

    def layer_params(self) -> int:
        return self.hidden * (self.hq + 2 * self.hkv) + self.hq * self.hidden + 3 * self.hidden * self.ffn


# BASELINE.json configs[0..4]; eps per reading A8, vocab per reading A12
TINY = ModelShape("tiny-llama", 256, 4, 2, 64, 688, 2, 1e-5, 5e5, 0, 512)
TINY_QWEN = ModelShape("tiny-qwen", 256, 4, 2, 64, 688, 2, 1e-6, 1e6, 1, 512)
TINY128 = ModelShape("tiny-d128", 512, 8, 1, 128, 1024, 2, 1e-5, 5e5, 1, 640)
LLAMA70B = ModelShape("llama-3.1-70b-shaped", 8192, 64, 8, 128, 28672, 20, 1e-5, 5e5, 0, 128256)
QWEN32B = ModelShape("qwen3-32b-shaped", 5120, 64, 8, 128, 25600, 16, 1e-6, 1e6, 1, 151936)


def lognormal_lengths(rng: np.random.Generator, n: int, median: float, lo: int, hi: int) -> np.ndarray:
    x = np.exp(rng.normal(np.log(median), SIGMA, n))
    return np.clip(np.round(x), lo, hi).astype(np.int64)


def _gen(seed: int, layer: int, idx: int) -> torch.Generator:
    g = torch.Generator()
    g.manual_seed(seed * 1_000_003 + 64 * layer + idx)
    return g


def randn_bf16(shape, std: float, gen: torch.Generator, mean: float = 0.0) -> torch.Tensor:
    t = torch.randn(shape, generator=gen, dtype=torch.float32)
    if std != 1.0:
        t.mul_(std)
    if mean != 0.0:
        t.add_(mean)
    return t.to(torch.bfloat16)


def layer_weights(shape: ModelShape, layer: int, seed: int = 0, proj_std: float = 0.02, executor=None) -> dict:
    """CPU bf16 tensors of one decoder layer (no biases: reading A7).  `executor` (a concurrent.futures executor)
    only draws the tensors concurrently: each has its own generator, so the bytes are the same either way."""
    H, Hq, Hkv, F, d = shape.hidden, shape.hq, shape.hkv, shape.ffn, shape.d
    shp = {"ln1": (H,), "wq": (Hq, H), "wk": (Hkv, H), "wv": (Hkv, H), "q_norm": (d,), "k_norm": (d,),
           "wo": (H, Hq), "ln2": (H,), "w_gate": (F, H), "w_up": (F, H), "w_down": (H, F)}
    def draw(idx, name):
        g = _gen(seed, layer, idx)
        if name in ("ln1", "ln2", "q_norm", "k_norm"):
            return randn_bf16(shp[name], 0.02, g, mean=1.0)
        return randn_bf16(shp[name], proj_std, g)

    if executor is None:
        out = {name: draw(idx, name) for idx, name in enumerate(_TENSORS)}
    else:
        futs = {name: executor.submit(draw, idx, name) for idx, name in enumerate(_TENSORS)}
        out = {name: f.result() for name, f in futs.items()}
    if not shape.qk_norm:
        out["q_norm"] = None
        out["k_norm"] = None
    return out


def edge_weights(shape: ModelShape, seed: int = 0) -> dict:
    V, H = shape.vocab, shape.hidden
    return {"embed": randn_bf16((V, H), 0.02 * 50, _gen(seed, 1000, 0)),   # embeddings scaled to O(1) rows
            "final_norm": randn_bf16((H,), 0.02, _gen(seed, 1000, 1), mean=1.0),
            "lm_head": randn_bf16((V, H), 0.02, _gen(seed, 1000, 2))}


def hidden_rows(n: int, H: int, seed: int, idx: int = 0) -> torch.Tensor:
    return randn_bf16((n, H), 1.0, _gen(seed, 2000, idx))


@dataclass
class PagedBatch:
    """Block tables + lengths of one call; all numpy int32."""
    lens: np.ndarray            # tokens per sequence that the pages must cover (ctx_before + q_len)
    block_tables: np.ndarray    # [n_seqs, max_blocks]
    n_pages_pool: int
    max_blocks: int
    used_pages: np.ndarray = field(default=None)


def paged_batch(rng: np.random.Generator, lens, extra_tokens: int = 0, pool_factor: float = 1.0,
                min_max_blocks: int = 0, n_pages_pool: int | None = None) -> PagedBatch:
    """Random permutation of the pool's pages laid into block tables covering lens[s] + extra_tokens tokens."""
    lens = np.asarray(lens, dtype=np.int64)
    need = (lens + extra_tokens + PAGE - 1) // PAGE
    total = int(need.sum())
    if n_pages_pool is None:
        n_pages_pool = max(int(np.ceil(total * pool_factor)), total)
    assert n_pages_pool >= total
    perm = rng.permutation(n_pages_pool)[:total].astype(np.int32)
    max_blocks = max(int(need.max()), min_max_blocks)
    bt = np.full((len(lens), max_blocks), -1, dtype=np.int32)
    o = 0
    for s, n in enumerate(need):
        bt[s, :n] = perm[o:o + n]
        o += n
    # entries past the needed pages are "ignored" by contract; fill them with a valid id so a buggy reader
    # cannot fault, while the sentinel tests still see any stray write
    bt[bt < 0] = 0
    return PagedBatch(lens.astype(np.int32), bt, n_pages_pool, max_blocks, perm)


def bits(t: torch.Tensor) -> np.ndarray:
    """bf16 torch tensor -> numpy uint16 bit patterns (shares memory when possible)."""
    return t.contiguous().view(torch.int16).numpy().view(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << 16).view(np.float32)


# ---- the five BASELINE.json workloads (lengths only; tensors are drawn by the callers) ------------------------

def cfg1_contexts(seed=0):
    return np.random.default_rng(seed).integers(17, 131, 4)


def cfg2_contexts(seed=0):
    return lognormal_lengths(np.random.default_rng(seed), 64, 1024, 128, 8192)


def cfg3_contexts(seed=0):
    return lognormal_lengths(np.random.default_rng(seed), 128, 768, 64, 4096)


def cfg4_lengths(seed=0):
    return lognormal_lengths(np.random.default_rng(seed), 32, 1200, 256, 4096)
