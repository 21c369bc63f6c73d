"""tensor parallelism inside a stage.  One GPU is all there is here, so the
D_TP ranks are D_TP shard stages of ONE process, each driven by its own host thread on its own stream; the all-reduce
they register is an in-process stand-in for NCCL that orders the streams with events and sums the partials with
torch ops (no kernel ever waits on another kernel).  What is checked is everything except the wire: the sharding, the
partial-sum path of the O / down projections, the two all-reduce points per layer, the per-rank KV pools."""
import threading

import numpy as np
import pytest
import torch

from oracle import Oracle
from paper_2606_18600_b200 import binding, synth, tp
from tests import helpers as hp

pytestmark = pytest.mark.gpu
F32 = Oracle("f32")
DEV = "cuda:0"


class InProcessAllReduce:
    def __init__(self, size):
        self.size, self.bar = size, threading.Barrier(size)
        self.buf, self.ev, self.ev2 = [None] * size, [None] * size, [None] * size
        self.calls = 0

    def fn(self, rank):
        def f(partial, stream_ptr):
            st = torch.cuda.ExternalStream(stream_ptr)
            e = torch.cuda.Event()
            e.record(st)
            self.buf[rank], self.ev[rank] = partial, e
            self.bar.wait()
            with torch.cuda.stream(st):
                for j in range(self.size):
                    st.wait_event(self.ev[j])
                tmp = self.buf[0].clone()
                for j in range(1, self.size):       # fixed order: every rank gets the same bits
                    tmp += self.buf[j]
            e2 = torch.cuda.Event()
            e2.record(st)
            self.ev2[rank] = e2
            self.bar.wait()
            with torch.cuda.stream(st):
                for j in range(self.size):
                    st.wait_event(self.ev2[j])      # nobody overwrites a partial another rank still reads
                partial.copy_(tmp)
            if rank == 0:
                self.calls += 1
            self.bar.wait()
        return f


def _dev_bf16(bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16).copy()).view(torch.bfloat16).to(DEV)


def _i32(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(DEV)


def _bits(t):
    return t.cpu().view(torch.int16).numpy().view(np.uint16)


@pytest.mark.parametrize("shape,size", [(synth.TINY_QWEN, 2), (synth.TINY128, 1)])
def test_tp_shards_prefill_then_decode_vs_oracle(shape, size):
    if shape.n_kv % size or shape.ffn % (8 * size):
        pytest.skip("shape not divisible")
    L = shape.n_layers
    lens = np.array([37, 16, 129, 70], dtype=np.int32)
    rng = np.random.default_rng(11)
    pb = synth.paged_batch(rng, lens, extra_tokens=4, pool_factor=1.5)
    tw, wb = hp.weights_bits(shape, 11)
    T = int(lens.sum())
    x = synth.bits(synth.hidden_rows(T + len(lens), shape.hidden, 11))
    sshape = tp.shard_shape(shape, size)
    dims = binding.make_dims(sshape, max_tokens=T + 8, max_seqs=8, max_blocks=pb.max_blocks, n_layers_total=L)
    stages = []
    for r in range(size):
        dw = [{k: (None if v is None else v.to(DEV)) for k, v in tp.shard_layer_weights(w, r, size, shape).items()} for w in tw]
        stages.append(binding.Stage(dims, 0, L, dw, None, n_pages=pb.n_pages_pool, device=DEV))
    ar = InProcessAllReduce(size)
    for r, st in enumerate(stages):
        st.pool_view().view(torch.int16).fill_(0x7FC1)
        st.set_allreduce(ar.fn(r))
    try:
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        outs = [torch.empty((T, shape.hidden), dtype=torch.bfloat16, device=DEV) for _ in range(size)]
        outs_d = [torch.empty((len(lens), shape.hidden), dtype=torch.bfloat16, device=DEV) for _ in range(size)]
        a = (_i32(cu), _i32(np.zeros_like(lens)), _i32(pb.block_tables), _dev_bf16(x[:T]), _i32(lens), _dev_bf16(x[T:]))
        torch.cuda.synchronize()
        errs = []

        def run(r):
            try:
                st = stages[r]
                st.prefill(len(lens), a[0], a[1], a[2], T, hidden=a[3], out_hidden=outs[r])
                st.decode(len(lens), a[2], a[4], hidden=a[5], out_hidden=outs_d[r])
                st.synchronize()
            except Exception as e:  # noqa: BLE001
                errs.append(e)
                ar.bar.abort()

        th = [threading.Thread(target=run, args=(r,)) for r in range(size)]
        for t in th:
            t.start()
        for t in th:
            t.join(120)
        assert not errs, errs
        assert ar.calls == 2 * L * 2                      # two all-reduces per layer, in each of the two calls
        pool = hp.new_pool(shape, pb.n_pages_pool, L)
        want, _, _ = hp.run_oracle_prefill(F32, shape, wb, pool, lens, pb.block_tables, x[:T])
        want_d, _ = hp.run_oracle_decode(F32, shape, wb, pool, lens, pb.block_tables, x[T:])
        for r in range(size):
            got = synth.bf16_bits_to_f32(_bits(outs[r]))
            got_d = synth.bf16_bits_to_f32(_bits(outs_d[r]))
            assert hp.rel_err_rows(got, want) < 2e-2 and hp.rel_err_rows(got_d, want_d) < 2e-2
            assert torch.equal(outs[r], outs[0]) and torch.equal(outs_d[r], outs_d[0])   # ranks agree bit for bit
        # per-rank KV pools: rank r holds kv heads [r * n_kv/size, (r+1) * n_kv/size) of the oracle's pool
        hk = shape.n_kv // size
        pool1 = hp.new_pool(shape, pb.n_pages_pool, L)
        hp.run_oracle_prefill(F32, shape, wb, pool1, lens, pb.block_tables, x[:T], rounding=1)
        hp.run_oracle_decode(F32, shape, wb, pool1, lens, pb.block_tables, x[T:], rounding=1)
        for r, st in enumerate(stages):
            pg = _bits(st.pool_view())
            ref = pool1[:, :, :, r * hk:(r + 1) * hk]
            written = ref != 0x7FC1
            assert np.array_equal(pg != 0x7FC1, written)                                # indexing: same slots
            fa, fb = synth.bf16_bits_to_f32(pg[0][written[0]]), synth.bf16_bits_to_f32(ref[0][written[0]])
            assert (np.abs(fa - fb) <= 4e-3 * np.abs(fb).max()).all()                   # layer 0 values
    finally:
        for st in stages:
            st.destroy()
