"""Pipeline of stages with micro-batching: one process per GPU, rank i owns the contiguous —
possibly uneven — layer range of stage i (Fig. 2), a `[rows, H]` bf16 tensor crosses each stage
boundary (Eq. 2), the last stage's greedy tokens go back to stage 0 for the next iteration, and M
micro-batches keep the stages busy (`b_t^j`, the t-th iteration of the j-th micro-batch, PAPER.md:255 / Fig. 6).

The schedule is lock-step: in tick tau every rank runs at most one item (t, j) and then all ranks do ONE grouped
exchange (send what I just produced to my successor, receive what my predecessor just produced).  Rank r runs item k
at tick start[k] + r, where start[] is the earliest schedule that respects the token feedback (item (t, j) needs the
tokens of (t - 1, j), which leave the last stage P - 1 ticks after stage 0 ran it).  With M >= P the pipeline is full:
one item per tick per rank, so a tick lasts max_i L^i (+ the hop) — the max of Eq. 5; with M < P
the schedule has P - M bubble ticks per iteration.  No arithmetic of the method lives here: the stage's work is the
`compute` callback (StagePipeline binds it to ss_stage_prefill / ss_stage_decode); this file is order and transport.

Transport: torch.distributed point-to-point, grouped per tick (batch_isend_irecv), so a send and a receive that
cross between the same two ranks cannot deadlock.  `wire="direct"` hands the device tensors to the backend (NCCL
over NVLink between B200s); `wire="host"` stages them through host memory (gloo: CPU tests, and the 2-process test on
one GPU).
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist


def item_starts(P: int, M: int, n_iters: int) -> list:
    """start[k] = tick in which stage 0 runs item k = t * M + j (stage r runs it at start[k] + r)."""
    start = []
    for k in range(n_iters * M):
        s = start[-1] + 1 if start else 0
        if k >= M:
            s = max(s, start[k - M] + P)      # tokens of (t - 1, j) reach stage 0 at the END of tick start + P - 1
        start.append(s)
    return start


def n_ticks(P: int, M: int, n_iters: int) -> int:
    return item_starts(P, M, n_iters)[-1] + P


class PipelineRank:
    """The driver loop of ONE stage.  compute(t, j, inp, out) runs item (t, j) of this stage: `inp` is a view of the
    token buffer (stage 0) or of the received hidden rows, `out` a view of the hidden rows to send on (or, on the last
    stage, of the int32 token buffer).  rows(t, j) = rows of the hidden tensor of item (t, j); n_tok(j) = tokens the
    last stage emits per item of micro-batch j (one per sequence)."""

    def __init__(self, rank, world, M, n_iters, hidden, rows, n_tok, compute, first_tokens, device="cpu",
                 hidden_dtype=torch.bfloat16, wire="direct", group=None, sync=None):
        self.r, self.P, self.M, self.n_iters = rank, world, M, n_iters
        self.rows, self.n_tok, self.compute, self.first_tokens = rows, n_tok, compute, first_tokens
        self.wire, self.group, self.sync = wire, group, sync or (lambda: None)
        self.start = item_starts(world, M, n_iters)
        self.at = {s: k for k, s in enumerate(self.start)}
        max_rows = max(rows(t, j) for t in range(n_iters) for j in range(M))
        self.hid_in = torch.empty((max_rows, hidden), dtype=hidden_dtype, device=device)
        self.hid_out = torch.empty((max_rows, hidden), dtype=hidden_dtype, device=device)
        self.tok = [torch.zeros((n_tok(j),), dtype=torch.int32, device=device) for j in range(M)]   # per micro-batch
        self.generated = {}                                    # last stage: (t, j) -> tokens (host copy)
        self.ticks = 0

    def _item(self, tick, r):
        return self.at.get(tick - r)

    def _send(self, ops, keep, x, dst):
        if self.wire == "host":
            self.sync()
            x = x.cpu()
        keep.append(x)
        ops.append(dist.P2POp(dist.isend, x, dst, self.group))

    def _recv(self, ops, post, x, src):
        if self.wire == "host" and x.device.type != "cpu":
            h = torch.empty(x.shape, dtype=x.dtype)
            post.append((x, h))
            x = h
        ops.append(dist.P2POp(dist.irecv, x, src, self.group))

    def run(self):
        r, P, M = self.r, self.P, self.M
        last = r == P - 1
        for tick in range(n_ticks(P, M, self.n_iters)):
            k = self._item(tick, r)
            out = None
            if k is not None:
                t, j = divmod(k, M)
                n = self.rows(t, j)
                inp = (self.first_tokens(j) if t == 0 else self.tok[j]) if r == 0 else self.hid_in[:n]
                out = self.tok[j] if last else self.hid_out[:n]
                self.compute(t, j, inp, out)
                if last:
                    self.sync()
                    self.generated[(t, j)] = out.cpu().clone()
            ops, keep, post = [], [], []
            if P > 1:
                if k is not None and (not last or t < self.n_iters - 1):
                    self._send(ops, keep, out, (r + 1) % P)
                prev = (r - 1) % P
                kp = self._item(tick, prev)
                if kp is not None:
                    tp_, jp = divmod(kp, M)
                    if r > 0:
                        self._recv(ops, post, self.hid_in[:self.rows(tp_, jp)], prev)
                    elif tp_ < self.n_iters - 1:
                        self._recv(ops, post, self.tok[jp], prev)
                if ops:
                    for w in dist.batch_isend_irecv(ops):
                        w.wait()
                    for dst, h in post:
                        dst.copy_(h)
            self.ticks += 1
        return self.generated


class StagePipeline:
    """PipelineRank bound to one ss_stage: item (0, j) is the prefill of micro-batch j's prompts, items (t >= 1, j)
    are decode steps.  `batches[j]` = dict(lens=int32[n] prompt lengths, block_tables=int32[n, max_blocks],
    prompt=int32[sum(lens)] token ids (used by stage 0 only)).  Every rank holds the same page mapping for its own
    layers' pool.  Greedy decoding: the last stage's argmax feeds stage 0."""

    def __init__(self, stage, rank, world, batches, n_iters, hidden, device, wire="direct", group=None):
        self.st, self.dev, self.batches = stage, device, batches
        i32 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(device)
        self.meta = []
        for b in batches:
            lens = np.asarray(b["lens"], dtype=np.int32)
            cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
            self.meta.append(dict(n=len(lens), T=int(lens.sum()), cu=i32(cu), zero=i32(np.zeros_like(lens)),
                                  bt=i32(b["block_tables"]), prompt=i32(b["prompt"]) if rank == 0 else None,
                                  ctx=[i32(lens + t - 1) for t in range(1, n_iters)]))
        self.first, self.last = rank == 0, rank == world - 1
        self.drv = PipelineRank(rank, world, len(batches), n_iters, hidden,
                                rows=lambda t, j: self.meta[j]["T"] if t == 0 else self.meta[j]["n"],
                                n_tok=lambda j: self.meta[j]["n"], compute=self._compute,
                                first_tokens=lambda j: self.meta[j]["prompt"], device=device, wire=wire, group=group,
                                sync=stage.synchronize)

    def _compute(self, t, j, inp, out):
        m = self.meta[j]
        kw = dict(token_ids=inp) if self.first else dict(hidden=inp)
        if self.last:
            kw.update(out_argmax=out)
        else:
            kw.update(out_hidden=out)
        if t == 0:
            self.st.prefill(m["n"], m["cu"], m["zero"], m["bt"], m["T"], **kw)
        else:
            self.st.decode(m["n"], m["bt"], m["ctx"][t - 1], **kw)

    def run(self):
        """The loop runs with the stage's stream current, so the transport (NCCL's stream, or the staging copies of
        the host wire) is ordered after the kernels that produced a tensor and before the ones that consume it."""
        if str(self.dev).startswith("cuda"):
            torch.cuda.synchronize()
            with torch.cuda.stream(self.st.stream):
                return self.drv.run()
        return self.drv.run()
