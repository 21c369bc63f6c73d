"""Tensor parallelism inside a stage: how a decoder layer's tensors are
cut into D_TP shards by KV head, and the all-reduce a rank registers with its stage (ss_stage_set_allreduce).

Sharding (the standard Megatron cut the paper's Table 2 divides by D_TP): q/k/v and gate/up projections by output
rows (whole heads / FFN columns stay on one rank), o and down projections by input columns, so each rank computes a
partial [T, H] of the O and down projections and the ranks sum them — two all-reduces per layer (Eq. 3).  Norm gains
and the residual stream are replicated; each rank's KV pool holds only its kv heads.  No arithmetic of the method
lives here: only slicing, and the call into torch.distributed.
"""
from __future__ import annotations

import torch

from . import synth


def shard_shape(shape: synth.ModelShape, size: int) -> synth.ModelShape:
    if shape.n_kv % size or shape.n_q % size or shape.ffn % (8 * size):
        raise ValueError(f"D_TP = {size} does not divide n_kv = {shape.n_kv}, n_q = {shape.n_q} or ffn/8 = {shape.ffn // 8}")
    return synth.ModelShape(f"{shape.name}/tp{size}", shape.hidden, shape.n_q // size, shape.n_kv // size, shape.d,
                            shape.ffn // size, shape.n_layers, shape.eps, shape.theta, shape.qk_norm, shape.vocab)


def shard_layer_weights(w: dict, rank: int, size: int, shape: synth.ModelShape) -> dict:
    """The rank's shard of one layer's tensors (contiguous copies; `shape` is the FULL model's shape)."""
    hq, hkv, f = shape.hq // size, shape.hkv // size, shape.ffn // size
    rows = lambda t, n: t[rank * n:(rank + 1) * n].contiguous()
    cols = lambda t, n: t[:, rank * n:(rank + 1) * n].contiguous()
    return {"ln1": w["ln1"], "ln2": w["ln2"], "q_norm": w.get("q_norm"), "k_norm": w.get("k_norm"),
            "wq": rows(w["wq"], hq), "wk": rows(w["wk"], hkv), "wv": rows(w["wv"], hkv), "wo": cols(w["wo"], hq),
            "w_gate": rows(w["w_gate"], f), "w_up": rows(w["w_up"], f), "w_down": cols(w["w_down"], f)}


def nccl_allreduce(group=None):
    """The all-reduce of a real multi-GPU run: one process per GPU, torch.distributed initialised with the nccl
    backend; the SUM is enqueued on the stage's stream (so it is ordered between the stage's kernels) and returns
    without synchronising.  Use: stage.set_allreduce(tp.nccl_allreduce())."""
    import torch.distributed as dist

    def fn(partial: torch.Tensor, stream_ptr: int) -> None:
        with torch.cuda.stream(torch.cuda.ExternalStream(stream_ptr)):
            dist.all_reduce(partial, op=dist.ReduceOp.SUM, group=group)

    return fn
