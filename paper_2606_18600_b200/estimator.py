"""The paper's static latency estimator for ONE stage, printed beside the measurements (report only).

L_op = max(FLOPs / FLOPS, MemScanCost * E / BW) summed over the Table-2 operations and the stage's layers
(Eq. 1; Table 2), D_TP = 1, E = 2 bytes.  Readings: A2 H_kv =
n_kv * d; A3 decode attention FLOPs = 4 * sum_b (ctx_b + 1) * Hq; A4 H^2 -> H * Hq where n_q * d != H; A5 the
memory term is elements * E / BW; A6 prefill attention keeps the paper's non-causal 4 * S^2 * H count.
Pure host arithmetic; not part of the hot path and not used by it.
"""
from __future__ import annotations

import numpy as np

E = 2.0


def _op(flops, mem_elems, FLOPS, BW):
    return max(flops / FLOPS, mem_elems * E / BW)


def decode_rows(shape, ctx, FLOPS, BW):
    """Per-layer seconds of each Table-2 'Decode' row for one iteration (S_out = 1, S_in -> ctx_b)."""
    ctx = np.asarray(ctx, dtype=np.float64)
    B = len(ctx)
    H, Hq, Hkv, F = shape.hidden, shape.hq, shape.hkv, shape.ffn
    tok = float((ctx + 1).sum())
    return {
        "qkv": _op(B * (2 * H * Hq + 4 * H * Hkv), B * H + H * Hq + 2 * H * Hkv, FLOPS, BW),
        "attention": _op(4 * tok * Hq, B * Hq + 2 * tok * Hkv, FLOPS, BW),
        "out_proj": _op(2 * B * Hq * H, B * Hq + Hq * H, FLOPS, BW),
        "up_gate": _op(4 * B * H * F, B * H + 2 * H * F, FLOPS, BW),
        "down": _op(2 * B * H * F, B * F + H * F, FLOPS, BW),
    }


def decode_step_ms(shape, ctx, FLOPS, BW) -> float:
    return 1e3 * shape.n_layers * sum(decode_rows(shape, ctx, FLOPS, BW).values())


def prefill_rows(shape, lens, FLOPS, BW):
    """Per-layer seconds of each Table-2 'Prefill' row with B*S_in -> sum(len), B*S_in^2 -> sum(len^2)."""
    lens = np.asarray(lens, dtype=np.float64)
    T, S2 = float(lens.sum()), float((lens * lens).sum())
    H, Hq, Hkv, F = shape.hidden, shape.hq, shape.hkv, shape.ffn
    return {
        "qkv": _op(T * (2 * H * Hq + 4 * H * Hkv), T * H + H * Hq + 2 * H * Hkv, FLOPS, BW),
        "attention": _op(4 * S2 * Hq, T * Hq + 2 * T * Hkv, FLOPS, BW),
        "out_proj": _op(2 * T * Hq * H, T * Hq + Hq * H, FLOPS, BW),
        "up_gate": _op(4 * T * H * F, T * H + 2 * H * F, FLOPS, BW),
        "down": _op(2 * T * H * F, T * F + H * F, FLOPS, BW),
    }


def prefill_ms(shape, lens, FLOPS, BW) -> float:
    return 1e3 * shape.n_layers * sum(prefill_rows(shape, lens, FLOPS, BW).values())
