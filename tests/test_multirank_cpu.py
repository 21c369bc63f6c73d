"""The N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only, no data-path collective (DESIGN.md
section 8; the paper's replicas are independent pipelines).  What is multi-rank is the timing
rule (max over ranks, whole-job value) and the launch contract (rank 0 alone prints one JSON line)."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [10.0, 12.5][rank]          # rank 1 is the slow replica
    e2e = [11.0, 10.5][rank]
    got = bench.max_over_ranks([ms, e2e], "cpu")
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, got))


def test_max_over_ranks_and_whole_job_value_gloo_world2():
    sys.path.insert(0, ROOT)
    import bench
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29000 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    assert res[0] == [12.5, 11.0] and res[1] == [12.5, 11.0]
    # 64 tokens x 20 steps per rank, 2 ranks, slowest rank 12.5 ms in total
    assert bench.whole_job_value(64 * 20, 2, 12.5) == 2 * 64 * 20 / 12.5e-3


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    """`bench.py --impl reference` launched the way the driver launches N > 1: rank 0 alone runs the oracle and
    prints; the other rank exits 0 without work."""
    port = 31000 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl",
           "reference", "--workload", "tiny", "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["unit"] == "tokens/s"


def _tp_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2606_18600_b200 import synth, tp
    dist.init_process_group("gloo", rank=rank, world_size=world)
    shape = synth.TINY_QWEN
    w = {k: (None if v is None else v.float()) for k, v in synth.layer_weights(shape, 0, 3).items()}
    ws = tp.shard_layer_weights(w, rank, world, shape)
    g = torch.Generator().manual_seed(5)
    T = 9
    h = torch.randn((T, shape.hidden), generator=g)
    o_full = torch.randn((T, shape.hq), generator=g)          # attention output, all heads
    # rank's slice of the heads -> partial of the O projection -> all-reduce (first all-reduce of the layer)
    hq = shape.hq // world
    part_o = o_full[:, rank * hq:(rank + 1) * hq] @ ws["wo"].T
    dist.all_reduce(part_o)
    # FFN: rank's FFN columns -> partial of the down projection -> all-reduce (second one)
    a = torch.nn.functional.silu(h @ ws["w_gate"].T) * (h @ ws["w_up"].T)
    part_d = a @ ws["w_down"].T
    dist.all_reduce(part_d)
    # the rank's q/k/v rows are whole heads of the full projections
    q_r = h @ ws["wq"].T
    k_r = h @ ws["wk"].T
    want_o = o_full @ w["wo"].T
    want_d = (torch.nn.functional.silu(h @ w["w_gate"].T) * (h @ w["w_up"].T)) @ w["w_down"].T
    q_full, k_full = h @ w["wq"].T, h @ w["wk"].T
    hkv = shape.hkv // world
    ok = (torch.allclose(part_o, want_o, rtol=1e-5, atol=1e-5) and torch.allclose(part_d, want_d, rtol=1e-5, atol=1e-5)
          and torch.equal(q_r, q_full[:, rank * hq:(rank + 1) * hq]) and torch.equal(k_r, k_full[:, rank * hkv:(rank + 1) * hkv]))
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, bool(ok)))


def test_tensor_parallel_sharding_algebra_gloo_world2():
    """NEXT-1 on CPU: with the layer cut by tp.shard_layer_weights, the ranks' partials of the O and down projections
    all-reduce (gloo, world_size 2) to the unsharded projections, and each rank's q/k rows are whole heads."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33000 + os.getpid() % 2000
    ps = [ctx.Process(target=_tp_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    assert res == {0: True, 1: True}


# ---- NEXT-2: the micro-batched pipeline driver (paper_2606_18600_b200/pipeline.py) on gloo, host logic only ----
_PIPE_H, _PIPE_N, _PIPE_T = 6, [3, 5, 2, 4], [7, 9, 4, 6]     # hidden size, sequences and prompt tokens per micro-batch


def _toy_stage(r, P):
    """a stand-in for a stage's arithmetic (exact in fp32): embeds on stage 0, emits tokens on the last stage"""
    def compute(t, j, inp, out):
        x = inp
        if r == 0:
            x = (inp.to(torch.float32) % 13).unsqueeze(1) + 0.5 * torch.arange(_PIPE_H, dtype=torch.float32) + t
        x = x * (r + 2) + j + 1
        if r == P - 1:
            x = (x[:out.numel()].sum(1).to(torch.int64) % 101).to(torch.int32)
        out.copy_(x)
    return compute


def _toy_prompt(j):
    return (torch.arange(_PIPE_T[j], dtype=torch.int32) * 3 + j) % 29


def _pipe_worker(rank, world, port, M, n_iters, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2606_18600_b200 import pipeline
    dist.init_process_group("gloo", rank=rank, world_size=world)
    drv = pipeline.PipelineRank(rank, world, M, n_iters, _PIPE_H, rows=lambda t, j: _PIPE_T[j] if t == 0 else _PIPE_N[j],
                                n_tok=lambda j: _PIPE_N[j], compute=_toy_stage(rank, world), first_tokens=_toy_prompt,
                                hidden_dtype=torch.float32, wire="host")
    gen = drv.run()
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, {k: v.tolist() for k, v in gen.items()}, drv.ticks))


def _pipe_sequential(P, M, n_iters):
    want = {}
    for j in range(M):
        tok = _toy_prompt(j)
        for t in range(n_iters):
            x = tok
            for r in range(P):
                rows = _PIPE_T[j] if t == 0 else _PIPE_N[j]
                o = torch.empty((_PIPE_N[j],), dtype=torch.int32) if r == P - 1 else torch.empty((rows, _PIPE_H))
                _toy_stage(r, P)(t, j, x, o)
                x = o
            want[(t, j)] = x.tolist()
            tok = x
    return want


def test_pipeline_schedule_closed_forms():
    sys.path.insert(0, ROOT)
    from paper_2606_18600_b200 import pipeline
    # full pipeline (M >= P): one item per tick, n_items + P - 1 ticks (fill + drain), the max-of-stages regime of Eq. 5
    for P, M, n in [(1, 1, 5), (2, 2, 3), (3, 4, 6), (4, 4, 2), (4, 9, 3)]:
        assert pipeline.item_starts(P, M, n) == list(range(M * n)) and pipeline.n_ticks(P, M, n) == M * n + P - 1
    # M < P: every iteration of a micro-batch waits for its own tokens: P ticks per iteration, P - M of them bubbles
    for P, M, n in [(3, 1, 4), (4, 2, 3), (5, 3, 2)]:
        s = pipeline.item_starts(P, M, n)
        assert all(s[t * M + j] == t * P + j for t in range(n) for j in range(M))
        assert pipeline.n_ticks(P, M, n) == (n - 1) * P + M - 1 + P
    # causality for arbitrary (P, M): stage 0 never runs (t, j) before the last stage finished (t - 1, j)
    for P in range(1, 6):
        for M in range(1, 7):
            s = pipeline.item_starts(P, M, 4)
            assert all(s[k] >= s[k - M] + P for k in range(M, len(s))) and all(b > a for a, b in zip(s, s[1:]))


def _run_pipe(world, M, n_iters):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33000 + (os.getpid() * 7 + world * 13 + M) % 2000
    ps = [ctx.Process(target=_pipe_worker, args=(r, world, port, M, n_iters, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = {}
    for _ in ps:
        r, gen, ticks = q.get(timeout=180)
        res[r] = (gen, ticks)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    return res


def test_pipeline_driver_gloo_world3_full_and_bubbled():
    sys.path.insert(0, ROOT)
    from paper_2606_18600_b200 import pipeline
    for M in (4, 2):                                         # M >= P: full pipeline; M < P: bubbles
        res = _run_pipe(3, M, 4)
        want = _pipe_sequential(3, M, 4)
        assert {tuple(k): v for k, v in res[2][0].items()} == want       # the last stage saw every (t, j), right values
        assert res[0][0] == {} and res[1][0] == {}
        assert all(res[r][1] == pipeline.n_ticks(3, M, 4) for r in range(3))
