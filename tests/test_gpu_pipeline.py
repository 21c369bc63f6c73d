"""SURVEY 8(f) NEXT-2 (the composition part): a model cut into stages of UNEVEN layer counts (the paper's asymmetric
partitioning, Fig. 2) — each stage an ss_stage over its own layer range [l0, l1) with its own KV
pool — chained through the bf16 [T, H] tensor that crosses a stage boundary.  Stage 0 takes token ids,
the last stage produces logits / argmax.  Checked against the oracle run stage by stage with the same bf16 hand-off."""
import numpy as np
import pytest
import torch

from oracle import Oracle
from paper_2606_18600_b200 import binding, synth
from tests import helpers as hp

pytestmark = pytest.mark.gpu
F32 = Oracle("f32")
DEV = "cuda:0"


def _bits(t):
    return t.cpu().view(torch.int16).numpy().view(np.uint16)


def _i32(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(DEV)


def test_uneven_three_stage_pipeline_vs_oracle():
    base = synth.TINY_QWEN
    L = 6
    shape = synth.ModelShape(base.name, base.hidden, base.n_q, base.n_kv, base.d, base.ffn, L, base.eps, base.theta,
                             base.qk_norm, base.vocab)
    cuts = [(0, 1), (1, 4), (4, 6)]                      # 1 + 3 + 2 layers
    lens = np.array([21, 64, 130, 5], dtype=np.int32)
    rng = np.random.default_rng(21)
    pb = synth.paged_batch(rng, lens, extra_tokens=4, pool_factor=1.5)
    tw, wb = hp.weights_bits(shape, 21)
    edge = synth.edge_weights(shape, 21)
    eb = {k: synth.bits(v) for k, v in edge.items()}
    edge_dev = {k: v.to(DEV) for k, v in edge.items()}
    T = int(lens.sum())
    ids = rng.integers(0, shape.vocab, T + len(lens)).astype(np.int32)
    dims = binding.make_dims(shape, max_tokens=T + 8, max_seqs=8, max_blocks=pb.max_blocks, n_layers_total=L)
    stages = []
    for (l0, l1) in cuts:
        dw = [{k: (None if v is None else v.to(DEV)) for k, v in tw[l].items()} for l in range(l0, l1)]
        e = None
        if l0 == 0 or l1 == L:
            e = {"embed": edge_dev["embed"] if l0 == 0 else None,
                 "final_norm": edge_dev["final_norm"] if l1 == L else None,
                 "lm_head": edge_dev["lm_head"] if l1 == L else None}
        stages.append(binding.Stage(dims, l0, l1, dw, e, n_pages=pb.n_pages_pool, device=DEV))
    try:
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        bt_d, cu_d, z_d, lens_d = _i32(pb.block_tables), _i32(cu), _i32(np.zeros_like(lens)), _i32(lens)
        n = len(lens)

        def gpu_pass(decode, ids_np, rows):
            h = [torch.empty((rows, shape.hidden), dtype=torch.bfloat16, device=DEV) for _ in cuts]
            lg = torch.empty((n, shape.vocab), dtype=torch.float32, device=DEV)
            am = torch.empty((n,), dtype=torch.int32, device=DEV)
            ids_d = _i32(ids_np)
            torch.cuda.synchronize()
            for i, st in enumerate(stages):
                kw = dict(token_ids=ids_d) if i == 0 else dict(hidden=h[i - 1])
                if i == len(stages) - 1:
                    kw.update(out_logits=lg, out_argmax=am)
                if decode:
                    st.decode(n, bt_d, lens_d, out_hidden=h[i], **kw)
                else:
                    st.prefill(n, cu_d, z_d, bt_d, rows, out_hidden=h[i], **kw)
                st.synchronize()                           # stage boundary: the next stage reads h[i]
            return h, lg.cpu().numpy(), am.cpu().numpy()

        def oracle_pass(pools, cu_q, ctx_before, ids_np):
            x_bits, y = None, None
            for i, (l0, l1) in enumerate(cuts):
                kw = dict(token_ids=ids_np, embed=eb["embed"]) if i == 0 else dict(x_in_bf16=x_bits)
                y, _ = F32.stage(hp.odims(shape), wb[l0:l1], pools[i], cu_q, ctx_before, pb.block_tables, **kw)
                x_bits = synth.bits(torch.from_numpy(np.ascontiguousarray(y, dtype=np.float32)).to(torch.bfloat16)).copy()
            return y

        pools = [hp.new_pool(shape, pb.n_pages_pool, l1 - l0) for (l0, l1) in cuts]
        want = oracle_pass(pools, cu, np.zeros_like(lens), ids[:T])
        h, lg, am = gpu_pass(False, ids[:T], T)
        got = synth.bf16_bits_to_f32(_bits(h[-1]))
        assert hp.rel_err_rows(got, want) < 2e-2
        wl, wa, wm = F32.logits(hp.odims(shape), want[cu[1:] - 1], eb["final_norm"], eb["lm_head"])
        assert np.array_equal(am, np.argmax(lg, axis=1).astype(np.int32))
        safe = wm > 8 * np.abs(lg - wl).max()
        assert np.array_equal(am[safe], wa[safe]) and hp.rel_err_rows(lg, wl) < 2e-2
        # decode step through the pipeline
        want_d = oracle_pass(pools, np.arange(n + 1, dtype=np.int32), lens, ids[T:])
        hd, lg2, am2 = gpu_pass(True, ids[T:], n)
        assert hp.rel_err_rows(synth.bf16_bits_to_f32(_bits(hd[-1])), want_d) < 2e-2
        assert np.array_equal(am2, np.argmax(lg2, axis=1).astype(np.int32))
        # every stage's pool is sized for exactly its own layers
        for i, st in enumerate(stages):
            assert st.pool_view().shape[0] == cuts[i][1] - cuts[i][0]
    finally:
        for st in stages:
            st.destroy()


# ---- two processes, one stage each, micro-batched (paper_2606_18600_b200/pipeline.py) --------------------------------
# The box has one GPU: both ranks open cuda:0 and talk through gloo with host staging (wire="host"); the ranks never
# wait on each other inside a kernel, only in the host-side exchange.  What must hold: the pipelined run generates
# exactly the tokens of the same two stages called one after the other in ONE process (same kernels, same shapes).
_CUTS2 = [(0, 2), (2, 6)]
_LENS2 = [np.array([21, 64, 5], dtype=np.int32), np.array([130, 17], dtype=np.int32)]
_ITERS2 = 4


def _pipe_problem():
    base = synth.TINY_QWEN
    shape = synth.ModelShape(base.name, base.hidden, base.n_q, base.n_kv, base.d, base.ffn, 6, base.eps, base.theta,
                             base.qk_norm, base.vocab)
    rng = np.random.default_rng(33)
    all_lens = np.concatenate(_LENS2)
    pb = synth.paged_batch(rng, all_lens, extra_tokens=_ITERS2 + 1, pool_factor=1.5)
    batches, r0 = [], 0
    for lens in _LENS2:
        batches.append(dict(lens=lens, block_tables=pb.block_tables[r0:r0 + len(lens)],
                            prompt=rng.integers(0, shape.vocab, int(lens.sum())).astype(np.int32)))
        r0 += len(lens)
    return shape, pb, batches


def _build_stage(shape, pb, l0, l1):
    tw, _ = hp.weights_bits(shape, 33)
    edge = {k: v.to(DEV) for k, v in synth.edge_weights(shape, 33).items()}
    L = shape.n_layers
    T = int(max(l.sum() for l in _LENS2))
    dims = binding.make_dims(shape, max_tokens=T + 8, max_seqs=8, max_blocks=pb.max_blocks, n_layers_total=L)
    dw = [{k: (None if v is None else v.to(DEV)) for k, v in tw[l].items()} for l in range(l0, l1)]
    e = {"embed": edge["embed"] if l0 == 0 else None, "final_norm": edge["final_norm"] if l1 == L else None,
         "lm_head": edge["lm_head"] if l1 == L else None}
    return binding.Stage(dims, l0, l1, dw, e, n_pages=pb.n_pages_pool, device=DEV)


def _pipe_rank(rank, world, port, q):
    import os
    import torch.distributed as dist
    from paper_2606_18600_b200 import pipeline
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    shape, pb, batches = _pipe_problem()
    st = _build_stage(shape, pb, *_CUTS2[rank])
    try:
        pl = pipeline.StagePipeline(st, rank, world, batches, _ITERS2, shape.hidden, DEV, wire="host")
        gen = pl.run()
        launches = st.launch_count()
    finally:
        st.destroy()
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, {k: v.tolist() for k, v in gen.items()}, launches))


def test_two_process_microbatched_pipeline_equals_in_process_chain():
    import os
    import torch.multiprocessing as mp
    shape, pb, batches = _pipe_problem()
    # in-process chain: stage 0 then stage 1, micro-batch after micro-batch, greedy feedback
    stages = [_build_stage(shape, pb, *c) for c in _CUTS2]
    want = {}
    try:
        for j, b in enumerate(batches):
            lens = b["lens"]
            n, T = len(lens), int(lens.sum())
            cu = _i32(np.concatenate([[0], np.cumsum(lens)]))
            bt, zero = _i32(b["block_tables"]), _i32(np.zeros_like(lens))
            tok = _i32(b["prompt"])
            for t in range(_ITERS2):
                rows = T if t == 0 else n
                h = torch.empty((rows, shape.hidden), dtype=torch.bfloat16, device=DEV)
                am = torch.empty((n,), dtype=torch.int32, device=DEV)
                torch.cuda.synchronize()
                if t == 0:
                    stages[0].prefill(n, cu, zero, bt, T, token_ids=tok, out_hidden=h)
                    stages[0].synchronize()
                    stages[1].prefill(n, cu, zero, bt, T, hidden=h, out_argmax=am)
                else:
                    ctx = _i32(lens + t - 1)
                    torch.cuda.synchronize()
                    stages[0].decode(n, bt, ctx, token_ids=tok, out_hidden=h)
                    stages[0].synchronize()
                    stages[1].decode(n, bt, ctx, hidden=h, out_argmax=am)
                stages[1].synchronize()
                want[(t, j)] = am.cpu().tolist()
                tok = am
    finally:
        for st in stages:
            st.destroy()
    ctx_mp = mp.get_context("spawn")
    q = ctx_mp.Queue()
    port = 35000 + os.getpid() % 2000
    ps = [ctx_mp.Process(target=_pipe_rank, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = {}
    for _ in ps:
        r, gen, launches = q.get(timeout=300)
        res[r] = (gen, launches)
    for p in ps:
        p.join(120)
        assert p.exitcode == 0
    assert {tuple(k): v for k, v in res[1][0].items()} == want
    assert res[0][0] == {} and res[0][1] > 0 and res[1][1] > 0           # both ranks launched their own kernels
    assert len(want) == _ITERS2 * len(batches) and len({tuple(v) for v in want.values()}) > 1
