"""placement_oracle.py — TEST INFRASTRUCTURE, not product.  A plain, slow restatement of ShuntServe's serving
performance estimator and of what its placement optimizer searches for (arxiv/paper_2606_18600 section 4), used only
by tests/ to check libshuntplace.so.  It shares no code with paper_2606_18600_b200/csrc/placement.cpp.

What it follows, in the paper's notation (Table 3):
  * Eq. 1: L_ops = max(FLOPs / FLOPS, MemScanCost * E / BW), summed over the operations;
  * Table 2, written out row by row below as (FLOPs, MemScanCost) pairs;
  * Eq. 2 / Eq. 3: L_PP = alpha + B S H E / beta; L_TP = 4 (alpha + B S H E / (D_TP beta)) (D_TP-1) l;
  * Eq. 5 / Eq. 4: L(B) = max_i L_prefill^i + max_i L_decode^i; RPS = B / L(B);
  * Eq. 6: B = min_i floor((M^i - M_weight^i - M_act) / (l^i (S_in + S_out) * bytes per token per layer));
  * Eq. 7: score = throughput / cost * (1 - gamma max(0, latency / SLO - 1)).
The optimizer's result is DEFINED as the placement with the best score; the oracle finds it by exhaustive enumeration
of every (stage count, layer split, instance assignment), which is what Algorithm 1 approximates with DP + beam.

Readings: A2 H_kv = n_kv d; A3 the decode attention row has a B; A4 H^2 -> H Hq; A5; A18 Eq. 6 needs the
KV bytes per token 2 H_kv E.  Pins: tests/test_placement.py (hand-computed Table-2 values, P14's numbers, monotonicity).
"""
from __future__ import annotations

import itertools
import math
from dataclasses import dataclass


@dataclass
class Model:
    hidden: int
    hq: int
    hkv: int
    ffn: int
    vocab: int
    n_layers: int
    elem_bytes: int = 2


@dataclass
class Instance:
    flops: float
    mem_bw: float
    mem_bytes: float
    n_gpus: int = 1
    alpha_intra: float = 0.0
    beta_intra: float = 1.0
    cost: float = 1.0


@dataclass
class Opts:
    s_in: float
    s_out: float
    alpha_inter: float = 0.0
    beta_inter: float = 1e30
    act_bytes: float = 0.0
    gamma: float = 0.0
    slo: float = 0.0
    max_stages: int = 64
    max_batch: int = 0


def table2(m: Model, B: float, s_in: float, s_out: float, D: float, phase: str):
    """Table 2 as {operation: (FLOPs, MemScanCost in elements)} for ONE layer (and the logits row), one stage."""
    H, Hq, Hkv, F, V = m.hidden, m.hq, m.hkv, m.ffn, m.vocab
    if phase == "prefill":
        S = s_in
        return {
            "qkv": (B * (2 * S * H * Hq + 4 * S * H * Hkv) / D, B * S * H + (H * Hq + 2 * H * Hkv) / D),
            "attention": (4 * B * S * S * Hq / D, (B * S * Hq + 2 * B * S * Hkv) / D),
            "output": (2 * B * S * Hq * H / D, (B * S * Hq + Hq * H) / D),
            "up_gate": (4 * B * S * H * F / D, B * S * H + 2 * H * F / D),
            "down": (2 * B * S * H * F / D, (B * S * F + H * F) / D),
            "logits": (2 * B * S * H * V / D, B * S * H + H * V / D),
        }
    att_f = sum(4 * B * (s_in + t) * Hq / D for t in range(1, int(s_out) + 1))
    att_m = sum((B * Hq + 2 * B * (s_in + t) * Hkv) / D for t in range(1, int(s_out) + 1))
    So = s_out
    return {
        "qkv": (B * So * (2 * H * Hq + 4 * H * Hkv) / D, So * (B * H + (H * Hq + 2 * H * Hkv) / D)),
        "attention": (att_f, att_m),
        "output": (2 * B * So * Hq * H / D, So * (B * Hq + Hq * H) / D),
        "up_gate": (4 * B * So * H * F / D, So * (B * H + 2 * H * F / D)),
        "down": (2 * B * So * H * F / D, So * (B * F + H * F) / D),
        "logits": (2 * B * So * H * V / D, So * (B * H + H * V / D)),
    }


def stage_latency(m: Model, g: Instance, o: Opts, layers: int, B: int, phase: str, is_last: bool, has_next: bool):
    D = g.n_gpus
    rows = table2(m, B, o.s_in, o.s_out, D, phase)
    lat_op = {k: max(f / g.flops, mem * m.elem_bytes / g.mem_bw) for k, (f, mem) in rows.items()}   # Eq. 1
    lat = layers * sum(v for k, v in lat_op.items() if k != "logits")
    if is_last and m.vocab > 0:
        lat += lat_op["logits"]
    S, n_msgs = (o.s_in, 1) if phase == "prefill" else (1, o.s_out)
    msg = B * S * m.hidden * m.elem_bytes
    if D > 1:
        lat += n_msgs * 4 * (g.alpha_intra + msg / (D * g.beta_intra)) * (D - 1) * layers            # Eq. 3
    if has_next:
        lat += n_msgs * (o.alpha_inter + msg / o.beta_inter)                                           # Eq. 2
    return lat


def max_batch(m: Model, types, o: Opts, inst, layers) -> int:
    per_layer_params = m.hidden * m.hq + 2 * m.hidden * m.hkv + m.hq * m.hidden + 3 * m.hidden * m.ffn
    kv = (o.s_in + o.s_out) * 2 * m.hkv * m.elem_bytes
    best = None
    for i, (t, l) in enumerate(zip(inst, layers)):
        g = types[t]
        w = l * per_layer_params * m.elem_bytes
        if i == 0:
            w += m.vocab * m.hidden * m.elem_bytes
        if i == len(inst) - 1:
            w += m.vocab * m.hidden * m.elem_bytes
        free = g.n_gpus * g.mem_bytes - w - o.act_bytes
        if free <= 0:
            return 0
        b = math.floor(free / (l * kv))                                                               # Eq. 6
        best = b if best is None else min(best, b)
    if best < 1:
        return 0
    if o.max_batch > 0:
        best = min(best, o.max_batch)
    return int(min(best, 10 ** 9))


def evaluate(m: Model, types, o: Opts, inst, layers):
    """A COMPLETE placement -> dict(batch, prefill_s, decode_s, rps, cost, score)."""
    assert sum(layers) == m.n_layers
    B = max_batch(m, types, o, inst, layers)
    cost = sum(types[t].cost for t in inst)
    if B <= 0:
        return dict(batch=0, prefill_s=0.0, decode_s=0.0, rps=0.0, cost=cost, score=0.0)
    n = len(inst)
    pre = max(stage_latency(m, types[t], o, l, B, "prefill", i == n - 1, i < n - 1) for i, (t, l) in enumerate(zip(inst, layers)))
    dec = max(stage_latency(m, types[t], o, l, B, "decode", i == n - 1, i < n - 1) for i, (t, l) in enumerate(zip(inst, layers)))
    lat = pre + dec                                                                                    # Eq. 5
    rps = B / lat                                                                                      # Eq. 4
    pen = 1.0
    if o.gamma > 0 and o.slo > 0:
        pen = 1 - o.gamma * max(0.0, lat / o.slo - 1)
    return dict(batch=B, prefill_s=pre, decode_s=dec, rps=rps, cost=cost, score=rps / cost * pen)     # Eq. 7


def compositions(n: int, k: int):
    """all ordered splits of n layers into k positive parts"""
    for cuts in itertools.combinations(range(1, n), k - 1):
        b = (0,) + cuts + (n,)
        yield tuple(b[i + 1] - b[i] for i in range(k))


def brute_force(m: Model, types, o: Opts, avail=None):
    """Exhaustive search: the best complete placement, or None if nothing fits."""
    best = None
    for s in range(1, min(o.max_stages, m.n_layers) + 1):
        for layers in compositions(m.n_layers, s):
            for inst in itertools.product(range(len(types)), repeat=s):
                if avail is not None and any(inst.count(t) > avail[t] for t in range(len(types))):
                    continue
                r = evaluate(m, types, o, inst, layers)
                if r["batch"] > 0 and (best is None or r["score"] > best[0]["score"]):
                    best = (r, inst, layers)
    return best


# ---- request dispatch (weighted round-robin on pipeline throughput; smooth variant) ----
def wrr_sequence(weights, n, changes=None):
    """The first n picks.  Each pick: credit_i += w_i for every pipeline with w_i > 0; choose the largest credit (lowest
    index on ties); credit_chosen -= sum of the positive weights.  `changes` = {pick index: (pipeline, new weight)} applied
    BEFORE that pick (the changed pipeline's credit restarts at 0).  -1 when no pipeline has a positive weight."""
    w = [float(x) for x in weights]
    credit = [0.0] * len(w)
    out = []
    for k in range(n):
        if changes and k in changes:
            i, nw = changes[k]
            w[i], credit[i] = float(nw), 0.0
        live = [i for i in range(len(w)) if w[i] > 0]
        if not live:
            out.append(-1)
            continue
        for i in live:
            credit[i] += w[i]
        best = live[0]
        for i in live:
            if credit[i] > credit[best]:
                best = i
        credit[best] -= sum(w[i] for i in live)
        out.append(best)
    return out
