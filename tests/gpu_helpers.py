"""GPU-side test helpers: build a Stage (CUDA path, through the C-ABI binding) from the same seeded tensors the
oracle side gets.  Nothing here computes any of the method's arithmetic."""
from __future__ import annotations

import numpy as np
import torch

from paper_2606_18600_b200 import binding, synth
from tests import helpers as hp

DEV = "cuda:0"


def to_dev(t):
    return None if t is None else t.to(DEV)


class Problem:
    """Weights (CPU bf16 + bit views for the oracle, device copies for the stage) + a stage."""

    def __init__(self, shape: synth.ModelShape, seed=0, proj_std=0.02, n_pages=64, max_tokens=512, max_seqs=16,
                 max_blocks=32, with_edge=False, n_layers=None, pool_fill="sentinel", inv_freq=None):
        self.shape = shape
        self.L = shape.n_layers if n_layers is None else n_layers
        self.tw, self.wb = hp.weights_bits(shape, seed, proj_std, self.L)
        self.dw = [{k: to_dev(v) for k, v in w.items()} for w in self.tw]
        self.edge_cpu = synth.edge_weights(shape, seed) if with_edge else None
        self.edge_dev = {k: to_dev(v) for k, v in self.edge_cpu.items()} if with_edge else None
        self.dims = binding.make_dims(shape, max_tokens, max_seqs, max_blocks, n_layers_total=self.L)
        # the oracle-side pool and the device pool start from the same bytes
        self.pool_cpu = hp.new_pool(shape, n_pages, self.L, fill=pool_fill, seed=seed)
        pool_dev = torch.from_numpy(self.pool_cpu.view(np.int16).copy()).view(torch.bfloat16).to(DEV).contiguous()
        self.stage = binding.Stage(self.dims, 0, self.L, self.dw, self.edge_dev, kv_pool=pool_dev.view(-1),
                                   device=DEV, inv_freq=inv_freq)
        assert self.stage.num_pages() == n_pages
        torch.cuda.synchronize()

    def pool_bits(self) -> np.ndarray:
        """device pool -> uint16 [L,2,pages,n_kv,16,d]"""
        self.stage.synchronize()
        return self.stage.pool_view().cpu().view(torch.int16).numpy().view(np.uint16)

    def i32(self, a):
        return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(DEV)

    def bf16(self, bits_u16):
        return torch.from_numpy(np.ascontiguousarray(bits_u16).view(np.int16).copy()).view(torch.bfloat16).to(DEV)

    def prefill(self, lens, bt, x_bits, ctx_before=None, logits=False):
        lens = np.asarray(lens, dtype=np.int32)
        ctx_before = np.zeros_like(lens) if ctx_before is None else np.asarray(ctx_before, dtype=np.int32)
        q_len = lens - ctx_before
        cu = np.concatenate([[0], np.cumsum(q_len)]).astype(np.int32)
        T = int(cu[-1])
        out = torch.empty((T, self.shape.hidden), dtype=torch.bfloat16, device=DEV)
        lg = am = None
        if logits:
            lg = torch.empty((len(lens), self.shape.vocab), dtype=torch.float32, device=DEV)
            am = torch.empty((len(lens),), dtype=torch.int32, device=DEV)
        args = (self.i32(cu), self.i32(ctx_before), self.i32(bt), self.bf16(x_bits))
        torch.cuda.synchronize()
        self.stage.prefill(len(lens), args[0], args[1], args[2], T, hidden=args[3], out_hidden=out, out_logits=lg,
                           out_argmax=am)
        self.stage.synchronize()
        res = synth.bf16_bits_to_f32(out.cpu().view(torch.int16).numpy().view(np.uint16))
        if logits:
            return res, lg.cpu().numpy(), am.cpu().numpy()
        return res

    def decode(self, ctx, bt, x_bits, logits=False):
        ctx = np.asarray(ctx, dtype=np.int32)
        B = len(ctx)
        out = torch.empty((B, self.shape.hidden), dtype=torch.bfloat16, device=DEV)
        lg = am = None
        if logits:
            lg = torch.empty((B, self.shape.vocab), dtype=torch.float32, device=DEV)
            am = torch.empty((B,), dtype=torch.int32, device=DEV)
        args = (self.i32(bt), self.i32(ctx), self.bf16(x_bits))
        torch.cuda.synchronize()
        self.stage.decode(B, args[0], args[1], hidden=args[2], out_hidden=out, out_logits=lg, out_argmax=am)
        self.stage.synchronize()
        res = synth.bf16_bits_to_f32(out.cpu().view(torch.int16).numpy().view(np.uint16))
        if logits:
            return res, lg.cpu().numpy(), am.cpu().numpy()
        return res

    def close(self):
        self.stage.destroy()


def bf16_ulp_distance(a_bits: np.ndarray, b_bits: np.ndarray) -> np.ndarray:
    """distance in bf16 steps between two bit patterns (sign-magnitude -> monotone integer)"""
    def mono(u):
        u = u.astype(np.int32)
        return np.where(u & 0x8000, -(u & 0x7FFF), u & 0x7FFF)
    return np.abs(mono(a_bits) - mono(b_bits))
