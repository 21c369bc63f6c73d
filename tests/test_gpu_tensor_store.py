"""Shared Tensor Store (Figure 7): weights and KV space owned by a separate process, attached
zero-copy through CUDA IPC by engine processes that coexist during "concurrent initialization".  -m gpu.

What is checked: (i) an engine running on attached tensors matches the oracle like one that owns its tensors;
(ii) a SECOND engine process attached to the same store while the first is alive costs no second copy of the arena
(device free memory barely moves) and sees the KV the first engine wrote — its decode step is bit-identical to the
first engine's; (iii) the first engine keeps working after the second has detached (the store outlives both)."""
import multiprocessing as mp

import numpy as np
import pytest
import torch

from paper_2606_18600_b200 import synth

pytestmark = pytest.mark.gpu

SHAPE = synth.TINY
SEED = 5
BALLAST_MB = 384          # makes a duplicated arena visible in cudaMemGetInfo
MAX_TOKENS, MAX_SEQS = 640, 16


def _store_main(conn, n_pages, max_blocks):
    """The store process: lays out the stage's weights + KV pool (+ ballast), publishes the manifest, stays alive."""
    from paper_2606_18600_b200 import tensor_store as ts
    try:
        L = SHAPE.n_layers
        layers = [synth.layer_weights(SHAPE, l, SEED, 0.02) for l in range(L)]
        kv_elems = L * 2 * n_pages * SHAPE.n_kv * 16 * SHAPE.d
        ent = ts.stage_entries(layers, None, kv_elems)
        ent["ballast"] = ("uint8", (BALLAST_MB << 20,))
        st = ts.TensorStore(ent)
        for i, w in enumerate(layers):
            for n, t in w.items():
                if t is not None:
                    st.put(f"layers.{i}.{n}", t)
        sentinel = torch.full((kv_elems,), 0x7FC1, dtype=torch.int16).view(torch.bfloat16)
        st.put("kv_pool", sentinel)
        conn.send(("manifest", st.manifest()))
        conn.recv()          # "stop"
        st.close()
        conn.send(("closed", None))
    except Exception as e:  # surface the failure in the parent instead of a hang
        conn.send(("error", repr(e)))


def _make_engine(manifest, max_blocks):
    from paper_2606_18600_b200 import binding, tensor_store as ts
    from tests import gpu_helpers as gh
    att = ts.attach(manifest)
    layers, edge, kv = ts.stage_tensors(att, SHAPE.n_layers)
    dims = binding.make_dims(SHAPE, MAX_TOKENS, MAX_SEQS, max_blocks, n_layers_total=SHAPE.n_layers)
    P = object.__new__(gh.Problem)          # the Problem helpers (prefill / decode marshalling) over borrowed tensors
    P.shape, P.L, P.dims = SHAPE, SHAPE.n_layers, dims
    P.stage = binding.Stage(dims, 0, SHAPE.n_layers, layers, edge, kv_pool=kv, device=gh.DEV)
    return att, P


def _engine_b_main(conn, manifest, max_blocks, ctx, bt, xs):
    """A second engine process, started while the first one is serving."""
    try:
        torch.cuda.init()
        torch.empty(1 << 20, device="cuda:0")
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info(0)
        from paper_2606_18600_b200 import tensor_store as ts
        att = ts.attach(manifest)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info(0)
        att.close()
        att, P = _make_engine(manifest, max_blocks)
        out = P.decode(ctx, bt, xs)
        pool = P.pool_bits().copy()
        P.close()
        att.close()
        conn.send(("ok", (out, pool, int(free0 - free1))))
    except Exception as e:
        conn.send(("error", repr(e)))


def test_two_engines_attach_to_one_store_and_agree():
    from oracle import Oracle
    from tests import helpers as hp
    ctxm = mp.get_context("spawn")
    rng = np.random.default_rng(SEED)
    lens = synth.cfg1_contexts(SEED).astype(np.int32)
    pb = synth.paged_batch(rng, lens, extra_tokens=4, pool_factor=2.0)
    bt, T = pb.block_tables, int(lens.sum())
    x = synth.bits(synth.hidden_rows(T + 16, SHAPE.hidden, SEED))
    _, wb = hp.weights_bits(SHAPE, SEED, 0.02)

    pa, ca = ctxm.Pipe()
    store = ctxm.Process(target=_store_main, args=(ca, pb.n_pages_pool, pb.max_blocks), daemon=True)
    store.start()
    assert pa.poll(180), "store process did not answer"
    kind, manifest = pa.recv()
    assert kind == "manifest", manifest
    att = P = None
    try:
        # ---- engine A (this process) on attached tensors vs the oracle
        att, P = _make_engine(manifest, pb.max_blocks)
        assert P.stage.num_pages() == pb.n_pages_pool
        w0 = synth.layer_weights(SHAPE, 1, SEED, 0.02)["w_down"]
        assert torch.equal(att.tensors["layers.1.w_down"].cpu(), w0), "attached weight bytes differ from the store's"
        F32 = Oracle("f32")
        pool0 = hp.new_pool(SHAPE, pb.n_pages_pool, SHAPE.n_layers)
        want, _, _ = hp.run_oracle_prefill(F32, SHAPE, wb, pool0, lens, bt, x[:T])
        got = P.prefill(lens, bt, x[:T])
        assert hp.rel_err_rows(got, want) < 2e-2
        xs = x[T:T + len(lens)]
        want_d, _ = hp.run_oracle_decode(F32, SHAPE, wb, pool0, lens, bt, xs)
        pool_before = P.pool_bits().copy()

        # ---- engine B: a second process, while A is alive (Figure 7: old and new engine coexist on the node)
        pb_, cb = ctxm.Pipe()
        eng = ctxm.Process(target=_engine_b_main, args=(cb, manifest, pb.max_blocks, lens, bt, xs), daemon=True)
        eng.start()
        assert pb_.poll(300), "engine B did not answer"
        kind, res = pb_.recv()
        assert kind == "ok", res
        out_b, pool_b, attach_cost = res
        eng.join(60)
        arena = manifest["bytes"]
        assert arena > BALLAST_MB << 20
        assert attach_cost < arena // 4, f"attaching cost {attach_cost} bytes of device memory for a {arena}-byte arena"
        assert hp.rel_err_rows(out_b, want_d) < 2e-2
        # B appended this step's K/V into the SHARED pool: A sees exactly B's bytes, and only the new slots changed
        pool_after_b = P.pool_bits()
        assert np.array_equal(pool_after_b, pool_b)
        changed = pool_after_b != pool_before
        assert changed.any() and np.count_nonzero(changed.any(axis=(0, 1, 3, 5))) == len(lens)

        # ---- A runs the same step over the same cache: bit-identical hidden rows, pool unchanged (same K/V rewritten)
        out_a = P.decode(lens, bt, xs)
        assert np.array_equal(out_a, out_b)
        assert np.array_equal(P.pool_bits(), pool_b)
    finally:
        if P is not None:
            P.close()
        if att is not None:
            att.close()
        pa.send("stop")
        if pa.poll(60):
            assert pa.recv()[0] == "closed"
        store.join(60)


def test_export_of_a_foreign_pointer_and_reattach_in_the_owner_fail_loudly():
    """cudaIpcOpenMemHandle refuses a handle in the process that exported it; the error surfaces as SS_ERR_CUDA."""
    from paper_2606_18600_b200 import binding, tensor_store as ts
    st = ts.TensorStore({"a": ("float32", (1024,))})
    try:
        m = st.manifest()
        assert len(bytes.fromhex(m["handle"])) == 64 and m["tensors"]["a"]["offset"] % ts.ALIGN == 0
        with pytest.raises(binding.ShuntStageError) as ei:
            ts.attach(m)
        assert ei.value.code == -6
        torch.cuda.synchronize()
    finally:
        # the failed open left a sticky-free error state at most; the arena must still free cleanly
        st.close()
