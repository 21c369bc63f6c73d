"""Online mixed-batch driver for BASELINE.json configs[4] ("cfg-5"): every iteration is ONE ss_stage_mixed call
(ss_stage_prefill plus the host hint "the first 96 sequences are decode rows") that combines 96 decode requests (q_len = 1 rows, first in the batch: reading A19) with up to 4 prefill chunks of
<= 512 tokens from new requests, over a page pool kept near 85% occupancy (reading A18), as in the paper's online
serving experiments (continuous batching of the Azure-trace-shaped load).

Host scheduling only — slots, lengths, the ready FIFO, page bookkeeping through the stage's allocator
(ss_kv_alloc / ss_kv_free) — no arithmetic of the method lives here; every step of the forward pass runs in the
CUDA kernels behind the C-ABI.  Recipe (DESIGN.md section 3 / SURVEY 8(d) cfg-5), all draws from one
numpy.random.default_rng(seed): decode slots start with ctx ~ LN(1024) in [16, 8192] and remaining output
~ LN(250) in [1, 2048]; prefill slots hold a new request with prompt ~ LN(600) in [16, 2048] (2048 = the paper's
prune), consumed <= 512 tokens per iteration; a finished prompt enters a ready FIFO (pages kept) and
its slot takes a new request; a decode slot whose remaining output hits 0 frees its pages and takes the FIFO head
(or, if the FIFO is empty, a fresh already-prefilled context); FIFO entries are dropped (pages freed) while the
occupancy exceeds 0.85.  A decode row always gets the page its next token needs: if the pool is out of pages, FIFO entries
and then prompts in mid-prefill are preempted (pages freed, the prompt starts over), and a prefill chunk is only admitted
while one free page per decode row remains.
"""
from __future__ import annotations

from collections import deque
from dataclasses import dataclass, field

import numpy as np
import torch

from . import synth

PAGE = synth.PAGE
N_DECODE, N_PREFILL, CHUNK = 96, 4, 512
OCCUPANCY = 0.85


@dataclass
class Req:
    pages: list = field(default_factory=list)
    ctx: int = 0          # tokens cached
    prompt: int = 0       # prefill slots: prompt length
    remaining: int = 0    # decode slots: output tokens still to produce


@dataclass
class Iteration:
    """What one call was given (host copies, for tests) and where its rows sit."""
    cu_q: np.ndarray
    ctx_before: np.ndarray
    block_tables: np.ndarray
    n_seqs: int
    T: int


class _CountingStage:
    """The allocator face of a stage for host-only dry runs of the scheduler: page ids off a free stack, no device."""

    def __init__(self, n_pages: int):
        self.n = n_pages
        self.free = list(range(n_pages - 1, -1, -1))

    def num_pages(self):
        return self.n

    def num_free(self):
        return len(self.free)

    def kv_alloc(self, n):
        out = self.free[-n:]
        del self.free[-n:]
        return out

    def kv_free(self, ids):
        self.free.extend(ids)


class OnlineDriver:
    def __init__(self, stage, shape: synth.ModelShape, seed: int = 0, max_blocks: int = 0, device="cuda:0",
                 use_mixed: bool = True):
        self.stage, self.shape, self.dev = stage, shape, torch.device(device)
        self.use_mixed = use_mixed   # False: plain ss_stage_prefill (decode rows as 1-row causal tiles)
        self.rng = np.random.default_rng(seed)
        self.max_blocks = max_blocks or (8192 + 2048 + CHUNK) // PAGE + 2
        self.n_pages = stage.num_pages()
        self.decode = [self._fresh_decode() for _ in range(N_DECODE)]
        self.prefill = [self._fresh_prefill() for _ in range(N_PREFILL)]
        self.fifo: deque = deque()
        self.stats = {"decode_tokens": 0, "prefill_tokens": 0, "dropped": 0, "preempted": 0, "evicted": 0, "finished": 0, "occupancy": []}
        self.h_bt = None  # staging buffers: made by the first step() (plan() / _advance() are host-only and testable without a GPU)

    def _staging(self):
        S = N_DECODE + N_PREFILL
        # pinned host staging + device copies of the per-call integer inputs
        self.h_bt = torch.zeros((S, self.max_blocks), dtype=torch.int32).pin_memory()
        self.h_cu = torch.zeros(S + 1, dtype=torch.int32).pin_memory()
        self.h_ctx = torch.zeros(S, dtype=torch.int32).pin_memory()
        self.d_bt = torch.zeros_like(self.h_bt, device=self.dev)
        self.d_cu = torch.zeros_like(self.h_cu, device=self.dev)
        self.d_ctx = torch.zeros_like(self.h_ctx, device=self.dev)

    # ---- sizing (reading A18): the pool whose mean occupancy over the run is 0.85 ----
    @staticmethod
    def _draw_decode(rng):
        ctx = int(synth.lognormal_lengths(rng, 1, 1024, 16, 8192)[0])
        rem = int(synth.lognormal_lengths(rng, 1, 250, 1, 2048)[0])
        return ctx, rem

    @staticmethod
    def initial_pages(seed: int) -> int:
        """Pages of the 96 initial decode contexts (same draws, same order as __init__) plus the prefill slots'
        first chunks, divided by 0.85: the pool that is 85% full at iteration 0."""
        rng = np.random.default_rng(seed)
        live = sum((OnlineDriver._draw_decode(rng)[0] + 1 + PAGE - 1) // PAGE for _ in range(N_DECODE))
        live += N_PREFILL * (CHUNK // PAGE)
        return int(np.ceil(live / OCCUPANCY))

    _POOL_CACHE: dict = {}

    @staticmethod
    def pool_pages(seed: int, iters: int = 500) -> int:
        """The pool size at which this scheduler, run for BASELINE.json's 500 iterations from `seed`, keeps the pool at
        85% occupancy ON AVERAGE (reading A18).  A pool that is 85% full of the initial contexts only is too small for
        the run the config asks for: the running requests age by a few hundred tokens each and their pages alone exceed
        it (96% mean occupancy, preemptions, prefill starved).  Found by bisection over host-only dry runs of the same
        scheduling code on a counting allocator (no GPU, ~0.3 s each); deterministic in the seed."""
        key = (seed, iters)
        if key in OnlineDriver._POOL_CACHE:
            return OnlineDriver._POOL_CACHE[key]

        def mean_occupancy(n_pages):
            drv = OnlineDriver(_CountingStage(n_pages), shape=None, seed=seed, device="cpu")
            for _ in range(iters):
                drv._advance(drv.plan())
            return float(np.mean(drv.stats["occupancy"]))

        lo = OnlineDriver.initial_pages(seed)
        hi = 2 * lo
        while mean_occupancy(hi) > OCCUPANCY:
            hi *= 2
        for _ in range(12):                      # occupancy falls as the pool grows
            mid = (lo + hi) // 2
            if mean_occupancy(mid) > OCCUPANCY:
                lo = mid
            else:
                hi = mid
            if hi - lo <= 8:
                break
        OnlineDriver._POOL_CACHE[key] = hi
        return hi

    def _alloc(self, req: Req, n_tokens: int) -> bool:
        need = (n_tokens + PAGE - 1) // PAGE - len(req.pages)
        if need > 0:
            if need > self.stage.num_free():
                return False
            req.pages += self.stage.kv_alloc(need)
        return True

    def _free(self, req: Req):
        if req.pages:
            self.stage.kv_free(req.pages)
            req.pages = []

    def _fresh_decode(self) -> Req:
        """A decode request whose context is taken as already cached (its pages hold whatever the pool held: the
        synthetic 'random KV pre-fill' of reading A21)."""
        ctx, rem = self._draw_decode(self.rng)
        r = Req(ctx=ctx, remaining=rem)
        while not self._alloc(r, ctx + 1):      # pool too full for this draw: halve it (keeps the run going)
            if ctx == 0:
                raise RuntimeError("page pool exhausted: not one free page for a new request")
            ctx = ctx // 2 if ctx > 16 else 0
            r.ctx = ctx
        return r

    def _fresh_prefill(self) -> Req:
        return Req(prompt=int(synth.lognormal_lengths(self.rng, 1, 600, 16, 2048)[0]))

    def occupancy(self) -> float:
        return 1.0 - self.stage.num_free() / self.n_pages

    # ---- one iteration: build the batch, call the stage, advance the state ----
    def plan(self):
        """Rows of this iteration: (request, q_len) for the 96 decode slots then the active prefill slots."""
        # Decode rows first: a running request gets the page its next token needs.  When the pool cannot give it, pages are
        # taken back in the order a continuous-batching scheduler preempts: prefilled requests still waiting in the FIFO
        # (newest first), then prompts in the middle of their prefill (they start over: recomputation), and last the
        # running request that holds the most pages (evicted; its slot takes a fresh, shorter request) — the decode set
        # alone outgrows a pool sized at 85% of the INITIAL contexts once every request has aged a few hundred tokens.
        for i in range(N_DECODE):
            if self.decode[i].remaining < 0:                   # evicted in this pass: refilled below
                continue
            while not self._alloc(self.decode[i], self.decode[i].ctx + 1):
                if self.fifo:
                    self._free(self.fifo.pop())
                    self.stats["dropped"] += 1
                    continue
                victim = max((p for p in self.prefill if p.pages), key=lambda p: len(p.pages), default=None)
                if victim is not None:
                    self._free(victim)
                    victim.ctx = 0
                    self.stats["preempted"] += 1
                    continue
                j = max((k for k in range(N_DECODE) if k != i and len(self.decode[k].pages) > 1),
                        key=lambda k: len(self.decode[k].pages), default=None)
                assert j is not None, "page pool smaller than one page per decode row"
                self._free(self.decode[j])
                self.stats["evicted"] += 1
                self.decode[j] = Req(remaining=-1)             # placeholder
        for k in range(N_DECODE):                              # evicted slots take a fresh request that fits
            if self.decode[k].remaining < 0:
                self.decode[k] = self._fresh_decode()
        rows = [(r, 1) for r in self.decode]
        # Prefill chunks only out of what is left beyond one page per decode row (the next iteration's worst case)
        for r in self.prefill:
            q = min(CHUNK, r.prompt - r.ctx)
            need = (r.ctx + q + PAGE - 1) // PAGE - len(r.pages)
            if q > 0 and self.stage.num_free() - need >= N_DECODE and self._alloc(r, r.ctx + q):
                rows.append((r, q))
        return rows

    def step(self, hidden_bank: torch.Tensor, out: torch.Tensor) -> Iteration:
        """hidden_bank: bf16 [>= T, H] device rows to feed (synthetic stage input); out: bf16 [>= T, H]."""
        if self.h_bt is None:
            self._staging()
        rows = self.plan()
        n = len(rows)
        q = np.array([ql for _, ql in rows], dtype=np.int32)
        cu = np.concatenate([[0], np.cumsum(q)]).astype(np.int32)
        T = int(cu[-1])
        bt = self.h_bt.numpy()
        for i, (r, _) in enumerate(rows):
            bt[i, :len(r.pages)] = r.pages
        self.h_cu.numpy()[:n + 1] = cu
        self.h_ctx.numpy()[:n] = [r.ctx for r, _ in rows]
        with torch.cuda.stream(self.stage.stream):
            self.d_bt.copy_(self.h_bt, non_blocking=True)
            self.d_cu.copy_(self.h_cu, non_blocking=True)
            self.d_ctx.copy_(self.h_ctx, non_blocking=True)
        self.stage.mixed(N_DECODE if self.use_mixed else 0, n, self.d_cu, self.d_ctx, self.d_bt, T,
                         hidden=hidden_bank[:T], out_hidden=out[:T])
        it = Iteration(cu.copy(), np.array([r.ctx for r, _ in rows], dtype=np.int32), bt[:n].copy(), n, T)
        self.stage.synchronize()   # the host staging buffers are rewritten next iteration
        self._advance(rows)
        return it

    def _advance(self, rows):
        st = self.stats
        for i, (r, ql) in enumerate(rows):
            r.ctx += ql
            if i < N_DECODE:
                st["decode_tokens"] += 1
                r.remaining -= 1
                if r.remaining <= 0:
                    self._free(r)
                    st["finished"] += 1
                    if self.fifo:
                        nxt = self.fifo.popleft()
                        nxt.remaining = int(synth.lognormal_lengths(self.rng, 1, 250, 1, 2048)[0])
                        self.decode[i] = nxt
                    else:
                        self.decode[i] = self._fresh_decode()
            else:
                st["prefill_tokens"] += ql
        for j, r in enumerate(self.prefill):
            if r.prompt > 0 and r.ctx >= r.prompt:
                self.fifo.append(r)
                self.prefill[j] = self._fresh_prefill()
        while self.fifo and self.occupancy() > OCCUPANCY:
            self._free(self.fifo.pop())
            st["dropped"] += 1
        st["occupancy"].append(self.occupancy())
