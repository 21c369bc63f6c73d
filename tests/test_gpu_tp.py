"""tensor parallelism inside a stage.  One GPU is all there is here, so the
D_TP ranks are D_TP shard stages of ONE process, each driven by its own host thread on its own stream; the all-reduce
they register is an in-process stand-in for NCCL that orders the streams with events and sums the partials with
torch ops (no kernel ever waits on another kernel).  What is checked is everything except the wire: the sharding, the
partial-sum path of the O / down projections, the two all-reduce points per layer, the per-rank KV pools."""
import ctypes as C
import multiprocessing as mp
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


@pytest.mark.parametrize("shape,size", [(synth.TINY_QWEN, 2), (synth.TINY128, 1), (synth.TINY, 2)])
def test_tp_fused_allreduce_decode_vs_oracle(shape, size):
    """ss_stage_set_tp_fused (the all-reduce fused into the O / down projections): every rank's GEMM
    epilogue stores its stream-K pieces into every rank's exchange buffer, the streams wait on arrival counters
    (cuStreamWaitValue32 — no kernel waits on another kernel, so the D_TP ranks can share this one GPU as D_TP stages
    of one process on D_TP streams), the residual + RMSNorm kernel adds all ranks' pieces in (rank, CTA) order.  The
    decode steps stay CUDA graphs.  Checked: outputs vs the oracle, ranks bit-identical, per-rank KV pools, graphs used;
    prefill (more than 128 tokens) still goes through the registered all-reduce callback."""
    if shape.n_kv % size or shape.ffn % (8 * size):
        pytest.skip("shape not divisible")
    L = shape.n_layers
    lens = np.array([37, 16, 129, 70], dtype=np.int32)
    n = len(lens)
    rng = np.random.default_rng(12)
    pb = synth.paged_batch(rng, lens, extra_tokens=6, pool_factor=1.5)
    tw, wb = hp.weights_bits(shape, 12)
    T = int(lens.sum())
    steps = 3
    x = synth.bits(synth.hidden_rows(T + steps * n, shape.hidden, 12))
    sshape = tp.shard_shape(shape, size)
    dims = binding.make_dims(sshape, max_tokens=T + 8, max_seqs=8, max_blocks=pb.max_blocks, n_layers_total=L)
    lib = binding.load_library()
    nbytes = lib.ss_tp_xchg_bytes(size)
    assert nbytes > 0 and lib.ss_tp_xchg_bytes(0) == 0 and lib.ss_tp_xchg_bytes(9) == 0
    xchg = [torch.empty(nbytes, dtype=torch.uint8, device=DEV) for _ in range(size)]
    stages = []
    for r in range(size):
        dw = [{k: (None if v is None else v.to(DEV)) for k, v in tp.shard_layer_weights(w, r, size, shape).items()} for w in tw]
        stages.append(binding.Stage(dims, 0, L, dw, None, n_pages=pb.n_pages_pool, device=DEV))
    ar = InProcessAllReduce(size)
    for r, st in enumerate(stages):
        st.pool_view().view(torch.int16).fill_(0x7FC1)
        st.set_allreduce(ar.fn(r))
        st.set_tp_fused(r, size, [b.data_ptr() for b in xchg])
    try:
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        outs = [torch.empty((T, shape.hidden), dtype=torch.bfloat16, device=DEV) for _ in range(size)]
        a = (_i32(cu), _i32(np.zeros_like(lens)), _i32(pb.block_tables), _dev_bf16(x[:T]))
        torch.cuda.synchronize()
        errs = []

        def run(r):   # prefill: 252 tokens > 128 -> the callback path, one host thread per rank as above
            try:
                stages[r].prefill(n, a[0], a[1], a[2], T, hidden=a[3], out_hidden=outs[r])
                stages[r].synchronize()
            except Exception as e:  # noqa: BLE001
                errs.append(e)
                ar.bar.abort()

        th = [threading.Thread(target=run, args=(r,)) for r in range(size)]
        for t in th:
            t.start()
        for t in th:
            t.join(120)
        assert not errs, errs
        calls_after_prefill = ar.calls
        assert calls_after_prefill == 2 * L
        # decode steps: fused path.  ONE host thread enqueues rank 0's step, then rank 1's: nothing blocks on the host,
        # the streams sort themselves out through the arrival counters
        pool = hp.new_pool(shape, pb.n_pages_pool, L)
        hp.run_oracle_prefill(F32, shape, wb, pool, lens, pb.block_tables, x[:T])
        bt = _i32(pb.block_tables)
        for k in range(steps):
            xs = x[T + k * n: T + (k + 1) * n]
            od = [torch.empty((n, shape.hidden), dtype=torch.bfloat16, device=DEV) for _ in range(size)]
            ctx, xd = _i32(lens + k), _dev_bf16(xs)
            torch.cuda.synchronize()
            for r in range(size):
                stages[r].decode(n, bt, ctx, hidden=xd, out_hidden=od[r])
            for r in range(size):
                stages[r].synchronize()
            want_d, _ = hp.run_oracle_decode(F32, shape, wb, pool, lens + k, pb.block_tables, xs)
            for r in range(size):
                got_d = synth.bf16_bits_to_f32(_bits(od[r]))
                err = hp.rel_err_rows(got_d, want_d)
                assert err < 2e-2, (k, r, err)
                assert torch.equal(od[r], od[0])            # ranks agree bit for bit
        assert ar.calls == calls_after_prefill              # the decode steps never used the callback
        for st in stages:
            assert st.graph_count() == 1                     # ... and ran as ONE captured graph, replayed
        hk = shape.n_kv // size
        pool1 = hp.new_pool(shape, pb.n_pages_pool, L)
        hp.run_oracle_prefill(F32, shape, wb, pool1, lens, pb.block_tables, x[:T], rounding=1)
        for k in range(steps):
            hp.run_oracle_decode(F32, shape, wb, pool1, lens + k, pb.block_tables, x[T + k * n: T + (k + 1) * n], rounding=1)
        for r, st in enumerate(stages):
            pg = _bits(st.pool_view())
            ref = pool1[:, :, :, r * hk:(r + 1) * hk]
            assert np.array_equal(pg != 0x7FC1, ref != 0x7FC1)                          # indexing: same slots
    finally:
        for st in stages:
            st.destroy()


# ---- the same fused all-reduce across two PROCESSES: exchange buffers are whole allocations of ss_store_alloc, handed
# over as CUDA IPC handles (ss_store_export / ss_store_attach), which is how two ranks on two GPUs of a node would map
# each other's memory.  The cross-rank waits are stream waits (cuStreamWaitValue32), never spinning kernels, so the two
# ranks can share the one GPU of this box.  Decode steps only (no callback needed): both ranks start from the same
# seeded random pool, each holding its kv heads. ----
IPC_SHAPE, IPC_SIZE, IPC_SEED, IPC_STEPS = synth.TINY_QWEN, 2, 21, 3


def _ipc_problem():
    shape = IPC_SHAPE
    ctx = np.array([40, 16, 127, 75, 3], dtype=np.int32)
    pb = synth.paged_batch(np.random.default_rng(IPC_SEED), ctx, extra_tokens=IPC_STEPS + 2, pool_factor=1.5)
    pool = hp.new_pool(shape, pb.n_pages_pool, shape.n_layers, fill="random", seed=IPC_SEED)
    x = synth.bits(synth.hidden_rows(IPC_STEPS * len(ctx), shape.hidden, IPC_SEED))
    return ctx, pb, pool, x


def _ipc_rank(rank, conn):
    """One tensor-parallel rank (runs in the pytest process for rank 0, in a spawned process for rank 1)."""
    shape, size = IPC_SHAPE, IPC_SIZE
    lib = binding.load_library()
    torch.cuda.init()
    ctx, pb, pool, x = _ipc_problem()
    n, L = len(ctx), shape.n_layers
    nbytes = lib.ss_tp_xchg_bytes(size)
    mine = C.c_void_p()
    assert lib.ss_store_alloc(C.byref(mine), nbytes) == 0
    handle = (C.c_ubyte * 64)()
    assert lib.ss_store_export(mine, handle) == 0
    conn.send(bytes(handle))
    peer_handle = (C.c_ubyte * 64).from_buffer_copy(conn.recv())
    peer = C.c_void_p()
    assert lib.ss_store_attach(peer_handle, C.byref(peer)) == 0, lib.ss_last_cuda_error()
    ptrs = [None, None]
    ptrs[rank], ptrs[1 - rank] = mine.value, peer.value
    tw, _ = hp.weights_bits(shape, IPC_SEED)
    sshape = tp.shard_shape(shape, size)
    dims = binding.make_dims(sshape, max_tokens=64, max_seqs=8, max_blocks=pb.max_blocks, n_layers_total=L)
    dw = [{k: (None if v is None else v.to(DEV)) for k, v in tp.shard_layer_weights(w, rank, size, shape).items()} for w in tw]
    hk = shape.n_kv // size
    shard_pool = np.ascontiguousarray(pool[:, :, :, rank * hk:(rank + 1) * hk])
    pool_dev = torch.from_numpy(shard_pool.view(np.int16)).view(torch.bfloat16).to(DEV).contiguous()
    st = binding.Stage(dims, 0, L, dw, None, kv_pool=pool_dev.view(-1), device=DEV)
    st.set_tp_fused(rank, size, ptrs)
    conn.send("ready")
    assert conn.recv() == "go"           # both ranks have zeroed their counters
    outs = []
    bt = _i32(pb.block_tables)
    for k in range(IPC_STEPS):
        od = torch.empty((n, shape.hidden), dtype=torch.bfloat16, device=DEV)
        st.decode(n, bt, _i32(ctx + k), hidden=_dev_bf16(x[k * n:(k + 1) * n]), out_hidden=od)
        st.synchronize()
        outs.append(_bits(od).copy())
    graphs = st.graph_count()
    st.destroy()
    assert lib.ss_store_detach(peer) == 0
    conn.send("done")
    assert conn.recv() == "bye"          # the peer has detached: the arena may go
    assert lib.ss_store_free(mine) == 0
    return outs, graphs


def _ipc_child(conn):
    try:
        outs, graphs = _ipc_rank(1, conn)
        conn.send(("ok", outs, graphs))
    except Exception as e:  # noqa: BLE001 - surface the failure in the parent instead of a hang
        conn.send(("error", repr(e), 0))


class _Relay:
    """Parent-side end of rank 0's conversation: forwards handle / ready / done between rank 0 (in-process) and the child."""

    def __init__(self, child_conn):
        self.c, self.stage = child_conn, 0

    def send(self, msg):
        if self.stage == 0:
            self.c.send(msg)             # rank 0's handle -> child
        self.stage += 1

    def recv(self):
        if self.stage == 1:              # the child's handle
            assert self.c.poll(180), "rank 1 did not answer"
            return self.c.recv()
        if self.stage == 2:              # rank 0 is ready: wait for the child's "ready", release both
            assert self.c.poll(180) and self.c.recv() == "ready"
            self.c.send("go")
            return "go"
        assert self.c.poll(180) and self.c.recv() == "done"
        self.c.send("bye")
        return "bye"


def test_tp_fused_allreduce_across_two_processes_over_cuda_ipc():
    ctxm = mp.get_context("spawn")
    parent, child = ctxm.Pipe()
    proc = ctxm.Process(target=_ipc_child, args=(child,), daemon=True)
    proc.start()
    try:
        outs0, graphs0 = _ipc_rank(0, _Relay(parent))
        assert parent.poll(180), "rank 1 did not finish"
        kind, outs1, graphs1 = parent.recv()
        assert kind == "ok", outs1
    finally:
        proc.join(60)
    ctx, pb, pool, x = _ipc_problem()
    _, wb = hp.weights_bits(IPC_SHAPE, IPC_SEED)
    n = len(ctx)
    for k in range(IPC_STEPS):
        want, _ = hp.run_oracle_decode(F32, IPC_SHAPE, wb, pool, ctx + k, pb.block_tables, x[k * n:(k + 1) * n])
        assert np.array_equal(outs0[k], outs1[k]), f"step {k}: the two ranks' outputs differ"
        err = hp.rel_err_rows(synth.bf16_bits_to_f32(outs0[k]), want)
        print(f"two-process fused TP decode step {k}: rel err vs oracle {err:.3e}")
        assert err < 2e-2
    assert graphs0 == 1 and graphs1 == 1
