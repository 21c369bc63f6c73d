"""Shared test helpers: build a seeded tiny problem and run the ORACLE side of it (no CUDA here)."""
from __future__ import annotations

import numpy as np
import torch

from oracle import Oracle, OracleDims
from paper_2606_18600_b200 import synth


def odims(shape: synth.ModelShape, rounding=0) -> OracleDims:
    return OracleDims(shape.hidden, shape.n_q, shape.n_kv, shape.d, shape.ffn, shape.vocab, shape.eps,
                      shape.theta, shape.qk_norm, rounding)


def weights_bits(shape: synth.ModelShape, seed=0, proj_std=0.02, n_layers=None):
    """list of per-layer dicts of torch bf16 tensors, and the same as numpy uint16 bit views."""
    L = shape.n_layers if n_layers is None else n_layers
    tl = [synth.layer_weights(shape, l, seed, proj_std) for l in range(L)]
    bl = [{k: (None if v is None else synth.bits(v)) for k, v in w.items()} for w in tl]
    return tl, bl


def new_pool(shape: synth.ModelShape, n_pages: int, L=None, fill="sentinel", seed=0) -> np.ndarray:
    """uint16 [L,2,pages,n_kv,16,d].  'sentinel' = 0x7FC1 (a NaN pattern no computation produces);
    'random' = N(0,1) bf16."""
    L = shape.n_layers if L is None else L
    shp = (L, 2, n_pages, shape.n_kv, 16, shape.d)
    if fill == "sentinel":
        return np.full(shp, 0x7FC1, dtype=np.uint16)
    g = torch.Generator()
    g.manual_seed(seed * 1_000_003 + 3000)
    t = torch.randn(shp, generator=g, dtype=torch.float32).to(torch.bfloat16)
    return synth.bits(t).copy()


def logical_kv(pool_layer_kv: np.ndarray, bt_row: np.ndarray, n_tokens: int) -> np.ndarray:
    """Gather one sequence's logical K (or V) [n_tokens, n_kv, d] out of a [pages,n_kv,16,d] pool."""
    pages = bt_row[: (n_tokens + 15) // 16]
    g = pool_layer_kv[pages]                      # [np, n_kv, 16, d]
    g = np.transpose(g, (0, 2, 1, 3)).reshape(-1, pool_layer_kv.shape[1], pool_layer_kv.shape[3])
    return g[:n_tokens]


def rel_err_rows(g: np.ndarray, r: np.ndarray) -> float:
    """Reading A15: per token row ||g-r||_inf / ||r||_inf, maximised over rows."""
    g = np.asarray(g, dtype=np.float64)
    r = np.asarray(r, dtype=np.float64)
    num = np.abs(g - r).max(axis=-1)
    den = np.abs(r).max(axis=-1)
    return float((num / np.maximum(den, 1e-30)).max())


def run_oracle_prefill(orc: Oracle, shape, wbits, pool, lens, bt, x_bits, ctx_before=None, rounding=0,
                       taps=False):
    """Prefill all sequences (q_len = lens - ctx_before) in one call. x_bits [T,H] uint16."""
    lens = np.asarray(lens, dtype=np.int32)
    ctx_before = np.zeros_like(lens) if ctx_before is None else np.asarray(ctx_before, dtype=np.int32)
    q_len = lens - ctx_before
    cu = np.concatenate([[0], np.cumsum(q_len)]).astype(np.int32)
    y, tp = orc.stage(odims(shape, rounding), wbits, pool, cu, ctx_before, bt, x_in_bf16=x_bits, taps=taps)
    return y, tp, cu


def run_oracle_decode(orc: Oracle, shape, wbits, pool, ctx, bt, x_bits, rounding=0, taps=False):
    """One decode step: each sequence has ctx[b] cached tokens, one new row each."""
    ctx = np.asarray(ctx, dtype=np.int32)
    cu = np.arange(len(ctx) + 1, dtype=np.int32)
    y, tp = orc.stage(odims(shape, rounding), wbits, pool, cu, ctx, bt, x_in_bf16=x_bits, taps=taps)
    return y, tp
