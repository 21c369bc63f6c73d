#!/usr/bin/env python
"""bench.py — stage decode tokens/s (+ % of HBM roofline) and migration-recompute prefill tokens/s of one
ShuntServe pipeline stage on B200, on synthetic workloads shaped like the paper's (BASELINE.json configs).

Default (the driver's contract): `python bench.py --gpus 1 --steps K --warmup W` times K decode steps of the
Llama-3.1-70B-shaped 20-layer stage (configs[1], "cfg2") and prints ONE JSON line.  A "step" is one pass of the
whole hot path (steps S0-S11 of DESIGN.md) over one batch of 64 sequences.  N > 1 (torchrun): independent
replicas, one per GPU, no data-path collective ("scaling": "weak").
`--impl reference` times the CPU oracle (as it stands) on a bounded sample of the same workload.
`--workload cfg3|cfg4|tiny` selects the other workloads for local measurement.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg2", "cfg3", "cfg4", "cfg5", "migrate", "pipeline", "estimator", "gemm", "tp_emul", "tiny"])
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--layers", type=int, default=0, help="override the stage depth (debug only; marks the line)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--batch-invariant", action="store_true",
                    help="run the stage in ss_stage_set_batch_invariant mode (measures what exact migration costs)")
    ap.add_argument("--tp", action="store_true",
                    help="cfg2/cfg3 decode as ONE stage sharded over the N ranks (tensor parallelism, fused all-reduce over "
                         "peer memory, DESIGN.md 8d) instead of N replicas; scaling = strong")
    ap.add_argument("--no-sub", action="store_true",
                    help="default workload only: skip the cfg-4 prefill and cfg-3 decode sub-records")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"],
                "bf16_tflops_sustained": d.get("bf16_tflops_sustained", d["bf16_tflops"]), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


def max_over_ranks(values, device):
    """Replicas only: no data-path collective; the one exchange is this MAX all-reduce of the
    ranks' device-timed milliseconds, so that the job's time is the slowest replica's."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_value(units_per_rank, world, ms_max):
    """units all ranks processed / max-over-ranks time (weak scaling: per-GPU work is fixed)."""
    return units_per_rank * world / (ms_max * 1e-3)


def source_hash():
    """sha1 over the CUDA sources of the library being timed (what 'the build' means for the ncu captures)."""
    import hashlib
    h = hashlib.sha1()
    d = os.path.join(ROOT, "paper_2606_18600_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh", ".h")):
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:12]


def ncu_traffic(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel (gate/up + SwiGLU GEMM) in
    this workload, from the committed `ncu --set full` capture (profiles/r02_traffic.json: a profiler cannot run inside
    the timed program).  Returns (bytes or None, label): the label names the build (source hash) the capture was taken
    from and says whether it is the build being timed."""
    p = os.path.join(ROOT, "profiles", "r02_traffic.json")
    try:
        e = json.load(open(p)).get(workload)
    except (OSError, ValueError):
        return None, "no capture committed"
    if not e:
        return None, "no capture committed for this workload"
    same = e.get("source_hash") == source_hash()
    return (e["dram_bytes_read"] + e["dram_bytes_write"],
            f"ncu --set full capture of build {e.get('source_hash')} ({e.get('profile')}); "
            + ("same sources as the library timed here" if same else "NOT the build timed here: context only"))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.gpu)], stdout=subprocess.PIPE, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for l in self.proc.stdout:
            self.lines.append(l.strip())

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------------------
# workloads
# ---------------------------------------------------------------------------------------------------------------
def workload_spec(name, layers_override=0):
    from paper_2606_18600_b200 import synth
    if name == "cfg2":
        shape, ctx, kind = synth.LLAMA70B, synth.cfg2_contexts, "decode"
    elif name == "cfg3":
        shape, ctx, kind = synth.QWEN32B, synth.cfg3_contexts, "decode"
    elif name == "cfg4":
        shape, ctx, kind = synth.LLAMA70B, synth.cfg4_lengths, "prefill"
    elif name == "cfg5":
        shape, ctx, kind = synth.QWEN32B, None, "online"
    elif name == "migrate":
        shape, ctx, kind = synth.LLAMA70B, None, "migrate"
    elif name == "pipeline":
        shape, ctx, kind = synth.LLAMA70B, synth.cfg2_contexts, "pipeline"
    elif name == "estimator":
        shape, ctx, kind = synth.LLAMA70B, None, "estimator"
    elif name == "gemm":
        shape, ctx, kind = synth.LLAMA70B, synth.cfg4_lengths, "gemm"
    elif name == "tp_emul":
        shape, ctx, kind = synth.LLAMA70B, synth.cfg2_contexts, "tp_emul"
    else:
        shape, ctx, kind = synth.TINY, synth.cfg1_contexts, "decode"
    L = layers_override or shape.n_layers
    if L != shape.n_layers:
        shape = synth.ModelShape(shape.name, shape.hidden, shape.n_q, shape.n_kv, shape.d, shape.ffn, L, shape.eps,
                                 shape.theta, shape.qk_norm, shape.vocab)
    return shape, ctx, kind


def decode_bytes_per_step(shape, ctx_now):
    """Algorithmic HBM bytes of one decode step: weights once, every cached K/V
    byte once (ctx+1 tokens incl. the new one), the new K/V written, stage input and output."""
    B = len(ctx_now)
    kv_tok = 2 * shape.hkv * 2
    per_layer = 2 * shape.layer_params() + int((ctx_now + 1).sum()) * kv_tok + B * kv_tok
    return shape.n_layers * per_layer + 2 * B * shape.hidden * 2


def prefill_flops(shape, lens):
    T = int(lens.sum())
    pairs = int((lens.astype(np.int64) * (lens.astype(np.int64) + 1) // 2).sum())
    return shape.n_layers * (2 * shape.layer_params() * T + 4 * shape.hq * pairs)


def gpu_weights(shape, dev, seed):
    """Random-init bf16 weights of the stage, generated on the device (synthetic; A21 value distributions)."""
    import torch
    g = torch.Generator(device=dev)
    g.manual_seed(seed * 1_000_003 + 17)
    H, Hq, Hkv, F, d = shape.hidden, shape.hq, shape.hkv, shape.ffn, shape.d

    def mat(r, c):
        return (torch.randn((r, c), generator=g, device=dev, dtype=torch.float32) * 0.02).to(torch.bfloat16)

    def gain(n):
        return (1 + 0.02 * torch.randn((n,), generator=g, device=dev, dtype=torch.float32)).to(torch.bfloat16)

    layers = []
    for _ in range(shape.n_layers):
        layers.append({"ln1": gain(H), "wq": mat(Hq, H), "wk": mat(Hkv, H), "wv": mat(Hkv, H),
                       "q_norm": gain(d) if shape.qk_norm else None, "k_norm": gain(d) if shape.qk_norm else None,
                       "wo": mat(H, Hq), "ln2": gain(H), "w_gate": mat(F, H), "w_up": mat(F, H), "w_down": mat(H, F)})
    return layers


def cuda_time_ms(stream, fn, n):
    """n calls of fn() on `stream`, timed with CUDA events recorded on that stream (ms total)."""
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream.synchronize()
    e0.record(stream)
    for i in range(n):
        fn(i)
    e1.record(stream)
    stream.synchronize()
    return e0.elapsed_time(e1)


def run_decode(args, shape, ctx_fn, rank, world, layers=None, K=None, W=None, dominant=True):
    import torch
    from paper_2606_18600_b200 import binding, synth
    dev = torch.device(f"cuda:{int(os.environ.get('LOCAL_RANK', 0))}")
    torch.cuda.set_device(dev)
    K, W = (args.steps if K is None else K), (args.warmup if W is None else W)
    rng = np.random.default_rng(args.seed)
    ctx0 = ctx_fn(args.seed).astype(np.int32)
    B = len(ctx0)
    total_steps = 2 * (K + W) + 8                        # device-timed pass + e2e pass
    pb = synth.paged_batch(rng, ctx0, extra_tokens=total_steps + 1)
    full_shape = shape
    if args.tp:
        from paper_2606_18600_b200 import tp as tpmod
        shape = tpmod.shard_shape(shape, world)          # this rank's shard (random-init: drawn at the shard's shape)
        layers = None
    if layers is None:
        layers = gpu_weights(shape, dev, args.seed + (1000 * rank if args.tp else 0))
    dims = binding.make_dims(shape, max_tokens=B, max_seqs=B, max_blocks=pb.max_blocks,
                             max_pos=int(ctx0.max()) + total_steps + 64)
    st = binding.Stage(dims, 0, shape.n_layers, layers, None, n_pages=pb.n_pages_pool, device=dev)
    st.set_batch_invariant(args.batch_invariant)
    tp_state = tp_fused_setup(st, rank, world) if args.tp else None
    g = torch.Generator(device=dev)
    g.manual_seed(args.seed + 99)
    _fill_randn(st.kv_pool.view(-1), g)                  # random KV pre-fill N(0,1) (A21)
    bank = [torch.randn((B, shape.hidden), generator=g, device=dev, dtype=torch.float32).to(torch.bfloat16)
            for _ in range(8)]                            # inputs cycled from a bank of 8
    bt = torch.from_numpy(pb.block_tables).to(dev)
    ctx_steps = torch.from_numpy(ctx0[None, :] + np.arange(total_steps, dtype=np.int32)[:, None]).to(dev).contiguous()
    out = torch.empty((B, shape.hidden), dtype=torch.bfloat16, device=dev)
    torch.cuda.synchronize(dev)

    step_no = [0]

    def one(i):
        s = step_no[0]
        st.decode(B, bt, ctx_steps[s], hidden=bank[s % 8], out_hidden=out)
        step_no[0] += 1

    for i in range(W):
        one(i)
    st.synchronize()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    torch.cuda.synchronize(dev)
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    n0 = st.launch_count()
    first_step = step_no[0]
    ms = cuda_time_ms(st.stream, one, K)
    launches = st.launch_count() - n0
    clocks = sampler.stop()
    # algorithmic bytes averaged over the timed steps (contexts grow by one token per step)
    byts = np.mean([decode_bytes_per_step(full_shape, ctx0 + first_step + i) for i in range(K)])

    # ---- e2e: the same step through the C-ABI with HOST buffers (pinned), H2D of inputs + D2H of the result inside
    e2e = None
    if not args.no_e2e:
        h_in = [b.cpu().pin_memory() for b in bank]
        h_bt = torch.from_numpy(pb.block_tables).pin_memory()
        h_ctx = (torch.from_numpy(ctx0[None, :] + np.arange(total_steps, dtype=np.int32)[:, None])).pin_memory()
        h_out = torch.empty((B, shape.hidden), dtype=torch.bfloat16).pin_memory()
        d_in = torch.empty_like(bank[0]); d_bt = torch.empty_like(bt); d_ctx = torch.empty_like(ctx_steps[0])

        def one_e2e(i):
            s = step_no[0]
            with torch.cuda.stream(st.stream):
                d_in.copy_(h_in[s % 8], non_blocking=True)
                d_bt.copy_(h_bt, non_blocking=True)
                d_ctx.copy_(h_ctx[s], non_blocking=True)
                st.decode(B, d_bt, d_ctx, hidden=d_in, out_hidden=out)
                h_out.copy_(out, non_blocking=True)
            st.stream.synchronize()                      # the caller reads the result of every step
            step_no[0] += 1

        for i in range(min(W, 3)):
            one_e2e(i)
        t0 = time.perf_counter()
        for i in range(K):
            one_e2e(i)
        dt = time.perf_counter() - t0
        e2e = {"ms_per_step": dt * 1e3 / K, "h2d": h_in[0].numel() * 2 + h_bt.numel() * 4 + B * 4,
               "d2h": h_out.numel() * 2}

    dom = dominant_gemm(st, shape, layers, B, dev) if dominant else None
    st.synchronize()
    o32 = out.float()
    if not bool(torch.isfinite(o32).all()):
        raise SystemExit("bench.py: the last decode step produced non-finite hidden states")
    res = {"ms": ms, "tokens": B * K, "bytes_per_step": float(byts), "launches": int(launches), "clocks": clocks,
           "e2e": e2e, "dominant": dom, "B": B, "ctx_sum": int(ctx0.sum()), "pages": int(pb.n_pages_pool),
           "checksum": float(o32.abs().mean()), "K": K, "W": W, "graphs": st.graph_count()}
    st.destroy()
    if tp_state is not None:
        tp_fused_teardown(tp_state, world)
    return res


def tp_fused_setup(st, rank, world):
    """Exchange buffers of the fused tensor-parallel all-reduce: one whole allocation per rank (ss_store_alloc), its
    CUDA IPC handle all-gathered over torch.distributed, the peers' buffers attached (ss_store_attach)."""
    import ctypes as C
    import torch.distributed as dist
    from paper_2606_18600_b200 import binding
    lib = binding.load_library()
    nbytes = lib.ss_tp_xchg_bytes(world)
    mine = C.c_void_p()
    if lib.ss_store_alloc(C.byref(mine), nbytes) != 0:
        raise SystemExit("ss_store_alloc failed: " + lib.ss_last_cuda_error().decode())
    handle = (C.c_ubyte * 64)()
    lib.ss_store_export(mine, handle)
    handles = [None] * world
    if world > 1:
        dist.all_gather_object(handles, bytes(handle))
    ptrs, attached = [None] * world, []
    for r in range(world):
        if r == rank:
            ptrs[r] = mine.value
        else:
            p = C.c_void_p()
            if lib.ss_store_attach((C.c_ubyte * 64).from_buffer_copy(handles[r]), C.byref(p)) != 0:
                raise SystemExit("ss_store_attach failed: " + lib.ss_last_cuda_error().decode())
            ptrs[r] = p.value
            attached.append(p)
    st.set_tp_fused(rank, world, ptrs)
    if world > 1:
        dist.barrier()                      # every rank's counters are zero before anybody's first step
    return lib, mine, attached


def tp_fused_teardown(state, world):
    lib, mine, attached = state
    for p in attached:
        lib.ss_store_detach(p)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()                      # every peer has detached
    lib.ss_store_free(mine)


def _fill_randn(pool, g):
    """N(0,1) bf16 fill of a pool too large for one temporary."""
    import torch
    n = pool.numel()
    step = 1 << 28
    for o in range(0, n, step):
        m = min(step, n - o)
        pool[o:o + m] = torch.randn((m,), generator=g, device=pool.device, dtype=torch.float32).to(torch.bfloat16)
    return pool


def dominant_gemm(st, shape, layers, T, dev):
    """The dominant kernel of the decode step is the fused gate/up + SwiGLU GEMM (45% of the step's bytes).  Time it
    alone with CUDA events on its stream, over the stage's own weights layer after layer (so nothing is L2-resident:
    each launch streams 2*H*F*2 bytes >> L2).  Launches are plain stream-ordered (no programmatic dependent launch:
    with PDL consecutive launches overlap head and tail and the per-launch time drops to 140.9 us = 102% of the
    measured copy peak, which is a throughput of overlapped launches, not one kernel's duration)."""
    import torch
    from paper_2606_18600_b200 import binding
    g = torch.Generator(device=dev)
    g.manual_seed(5)
    x = torch.randn((T, shape.hidden), generator=g, device=dev, dtype=torch.float32).to(torch.bfloat16)
    torch.cuda.synchronize(dev)
    L = len(layers)

    def one(i):
        w = layers[i % L]
        binding.op_gemm_swiglu_bf16(x, w["w_gate"], w["w_up"], stream=st.stream)

    for i in range(min(L, 4)):
        one(i)
    n = max(L, 20)
    ms = cuda_time_ms(st.stream, one, n)
    alg = 2 * shape.hidden * shape.ffn * 2 + T * shape.hidden * 2 + T * shape.ffn * 2
    return {"kernel": "gemm_kernel<DUAL> (gate/up + SwiGLU)", "us": ms * 1e3 / n, "bytes": alg,
            "flops": 4 * T * shape.hidden * shape.ffn}


def run_prefill(args, shape, len_fn, rank, world, layers=None, K=None, W=None):
    """cfg4: migration recompute — one ss_stage_prefill over all migrated requests, packed varlen, ctx_before = 0."""
    import torch
    from paper_2606_18600_b200 import binding, synth
    dev = torch.device(f"cuda:{int(os.environ.get('LOCAL_RANK', 0))}")
    torch.cuda.set_device(dev)
    K, W = (args.steps if K is None else K), (args.warmup if W is None else W)
    rng = np.random.default_rng(args.seed)
    lens = len_fn(args.seed).astype(np.int32)
    n = len(lens)
    T = int(lens.sum())
    pb = synth.paged_batch(rng, lens, extra_tokens=1)
    if layers is None:
        layers = gpu_weights(shape, dev, args.seed)
    dims = binding.make_dims(shape, max_tokens=T, max_seqs=n, max_blocks=pb.max_blocks, max_pos=int(lens.max()) + 64)
    st = binding.Stage(dims, 0, shape.n_layers, layers, None, n_pages=pb.n_pages_pool, device=dev)
    st.set_batch_invariant(args.batch_invariant)
    g = torch.Generator(device=dev)
    g.manual_seed(args.seed + 99)
    x = torch.randn((T, shape.hidden), generator=g, device=dev, dtype=torch.float32).to(torch.bfloat16)
    bt = torch.from_numpy(pb.block_tables).to(dev)
    cu = torch.from_numpy(np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)).to(dev)
    ctxb = torch.zeros(n, dtype=torch.int32, device=dev)
    out = torch.empty((T, shape.hidden), dtype=torch.bfloat16, device=dev)
    torch.cuda.synchronize(dev)

    def one(i):
        st.prefill(n, cu, ctxb, bt, T, hidden=x, out_hidden=out)

    for i in range(W):
        one(i)
    st.synchronize()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    n0 = st.launch_count()
    ms = cuda_time_ms(st.stream, one, K)
    launches = st.launch_count() - n0
    clocks = sampler.stop()
    e2e = None
    if not args.no_e2e:
        h_x = x.cpu().pin_memory()
        h_out = torch.empty((T, shape.hidden), dtype=torch.bfloat16).pin_memory()
        h_bt, h_cu = pb.block_tables, cu.cpu().pin_memory()
        h_btp = torch.from_numpy(h_bt).pin_memory()

        def one_e2e(i):
            with torch.cuda.stream(st.stream):
                x.copy_(h_x, non_blocking=True)
                bt.copy_(h_btp, non_blocking=True)
                cu.copy_(h_cu, non_blocking=True)
                st.prefill(n, cu, ctxb, bt, T, hidden=x, out_hidden=out)
                h_out.copy_(out, non_blocking=True)
            st.stream.synchronize()

        one_e2e(0)
        t0 = time.perf_counter()
        for i in range(K):
            one_e2e(i)
        dt = time.perf_counter() - t0
        e2e = {"ms_per_step": dt * 1e3 / K, "h2d": h_x.numel() * 2 + h_btp.numel() * 4 + h_cu.numel() * 4,
               "d2h": h_out.numel() * 2}
    st.synchronize()
    if not bool(torch.isfinite(out[-4096:].float()).all()):
        raise SystemExit("bench.py: the prefill produced non-finite hidden states")
    res = {"ms": ms, "tokens": T * K, "flops_per_step": float(prefill_flops(shape, lens)), "launches": int(launches),
           "clocks": clocks, "e2e": e2e, "T": T, "n_seqs": n, "pages": int(pb.n_pages_pool), "K": K, "W": W,
           "checksum": float(out[-4096:].float().abs().mean())}
    st.destroy()
    return res


def run_migrate(args, shape):
    """SURVEY 8(f) NEXT-4 / the paper's Fig. 5 question: migrate one request of context L
    by RECOMPUTATION (one ss_stage_prefill of its L tokens) or by KV TRANSFER (ss_kv_export gather -> GPU-to-GPU copy
    -> ss_kv_import scatter).  One GPU here: gather and scatter are measured, the link is modelled at NVLink 5's
    900 GB/s per direction (stated in the output)."""
    import torch
    from paper_2606_18600_b200 import binding
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    lengths = [1024, 4096, 16384, 65536]
    Lmax = lengths[-1]
    n_pages = Lmax // 16 + 8
    layers = gpu_weights(shape, dev, args.seed)
    dims = binding.make_dims(shape, max_tokens=Lmax, max_seqs=1, max_blocks=n_pages, max_pos=Lmax + 64)
    st = binding.Stage(dims, 0, shape.n_layers, layers, None, n_pages=n_pages, device=dev)
    g = torch.Generator(device=dev)
    g.manual_seed(args.seed + 7)
    x = torch.randn((Lmax, shape.hidden), generator=g, device=dev, dtype=torch.float32).to(torch.bfloat16)
    out = torch.empty_like(x)
    perm = torch.randperm(n_pages, generator=g, device=dev).to(torch.int32)
    bt = perm.view(1, -1).contiguous()
    ctxb = torch.zeros(1, dtype=torch.int32, device=dev)
    page_bytes = shape.n_layers * 2 * shape.hkv * 16 * 2
    rows = []
    for L in lengths:
        cu = torch.tensor([0, L], dtype=torch.int32, device=dev)
        n = (L + 15) // 16
        ids = perm[:n].contiguous()
        buf = torch.empty(n * page_bytes // 2, dtype=torch.bfloat16, device=dev)
        st.prefill(1, cu, ctxb, bt, L, hidden=x[:L], out_hidden=out[:L])       # warm-up (also fills the pages)
        rec = cuda_time_ms(st.stream, lambda i: st.prefill(1, cu, ctxb, bt, L, hidden=x[:L], out_hidden=out[:L]), 1)
        st.kv_export(ids, buf); st.kv_import(ids, buf)
        reps = 5
        ex = cuda_time_ms(st.stream, lambda i: st.kv_export(ids, buf), reps) / reps
        im = cuda_time_ms(st.stream, lambda i: st.kv_import(ids, buf), reps) / reps
        nbytes = n * page_bytes
        link = nbytes / 900e9 * 1e3
        rows.append({"context": L, "kv_bytes": nbytes, "recompute_ms": rec, "export_ms": ex, "import_ms": im,
                     "export_GBs": 2 * nbytes / (ex * 1e-3) / 1e9, "link_ms_modelled_900GBs": link,
                     "transfer_ms": ex + link + im, "recompute_over_transfer": rec / (ex + link + im)})
    st.destroy()
    return rows


def run_pipeline(args, shape, ctx_fn):
    """SURVEY 8(f) NEXT-2 / Eq. 5: an 80-layer 70B-shaped model cut into 4 stages, evenly (20 x 4) and
    unevenly (12 + 28 + 20 + 20, the paper's asymmetric partitioning).  The box has ONE B200, so each
    stage is measured alone, exactly as its own GPU would run it (cfg-2 micro-batch, B = 64; the last stage with the
    final norm + lm_head + argmax tail); the hop between stages is MODELLED (one [B, H] bf16 message over NVLink 5,
    900 GB/s + 10 us).  With M >= P micro-batches in flight (paper_2606_18600_b200/pipeline.py) every tick delivers one
    micro-batch iteration, so throughput = B / (max_i L^i + hop): the slowest stage sets it."""
    import torch
    from paper_2606_18600_b200 import binding, estimator, synth
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    K, W = args.steps, args.warmup
    pk = peaks()
    rng = np.random.default_rng(args.seed)
    ctx0 = ctx_fn(args.seed).astype(np.int32)
    B = len(ctx0)
    steps = 2 * (K + W) + 4
    pb = synth.paged_batch(rng, ctx0, extra_tokens=steps + 1)
    splits = {"even": [20, 20, 20, 20], "uneven": [12, 28, 20, 20]}
    depths = sorted({l for v in splits.values() for l in v})
    layers = gpu_weights(synth.ModelShape(shape.name, shape.hidden, shape.n_q, shape.n_kv, shape.d, shape.ffn,
                                          max(depths), shape.eps, shape.theta, shape.qk_norm, shape.vocab), dev, args.seed)
    g = torch.Generator(device=dev)
    g.manual_seed(args.seed + 99)
    edge = {"embed": None, "final_norm": torch.ones(shape.hidden, device=dev, dtype=torch.bfloat16),
            "lm_head": (torch.randn((shape.vocab, shape.hidden), generator=g, device=dev) * 0.02).to(torch.bfloat16)}
    bank = [torch.randn((B, shape.hidden), generator=g, device=dev, dtype=torch.float32).to(torch.bfloat16)
            for _ in range(8)]
    bt = torch.from_numpy(pb.block_tables).to(dev)
    ctx_steps = torch.from_numpy(ctx0[None, :] + np.arange(steps, dtype=np.int32)[:, None]).to(dev).contiguous()
    out = torch.empty((B, shape.hidden), dtype=torch.bfloat16, device=dev)
    am = torch.empty((B,), dtype=torch.int32, device=dev)
    measured, launches = {}, 0
    sampler = ClockSampler(0)
    sampler.start()
    for l in depths:
        for tail in (False, True):
            if tail and l != splits["even"][-1] and l != splits["uneven"][-1]:
                continue
            dims = binding.make_dims(shape, max_tokens=B, max_seqs=B, max_blocks=pb.max_blocks,
                                     max_pos=int(ctx0.max()) + steps + 64, n_layers_total=80)
            st = binding.Stage(dims, 80 - l if tail else 0, 80 if tail else l, layers[:l], edge if tail else None,
                               n_pages=pb.n_pages_pool, device=dev)
            _fill_randn(st.kv_pool.view(-1), g)
            torch.cuda.synchronize(dev)
            no = [0]

            def one(i):
                kw = dict(out_argmax=am) if tail else dict(out_hidden=out)
                st.decode(B, bt, ctx_steps[no[0]], hidden=bank[no[0] % 8], **kw)
                no[0] += 1

            for i in range(W):
                one(i)
            n0 = st.launch_count()
            measured[(l, tail)] = cuda_time_ms(st.stream, one, K) / K
            launches += st.launch_count() - n0
            st.destroy()
    clocks = sampler.stop()
    hop_ms = (B * shape.hidden * 2 / 900e9 + 10e-6) * 1e3
    rows = []
    for name, cut in splits.items():
        Li = [measured[(l, i == len(cut) - 1)] for i, l in enumerate(cut)]
        est = [estimator.decode_step_ms(synth.ModelShape(shape.name, shape.hidden, shape.n_q, shape.n_kv, shape.d,
                                                         shape.ffn, l, shape.eps, shape.theta, shape.qk_norm, shape.vocab),
                                        ctx0, pk["bf16_tflops"] * 1e12, pk["hbm_gbs"] * 1e9) for l in cut]
        rows.append({"split": name, "layers": cut, "stage_ms_measured": Li, "stage_ms_estimator_no_tail": est,
                     "max_stage_ms": max(Li), "sum_stage_ms": sum(Li), "hop_ms_modelled": hop_ms,
                     "tokens_per_s": B / ((max(Li) + hop_ms) * 1e-3),
                     "token_latency_ms": sum(Li) + (len(cut) - 1) * hop_ms})
    return rows, B, launches, clocks


def run_estimator(args, shape):
    """SURVEY 8(f) NEXT-3, the Fig. 8 question asked of this B200: how well does the paper's static
    estimator (Eq. 1 + Table 2, computed by libshuntplace's sp_stage_latency) predict a stage's measured latency?  The
    paper's protocol: S_in = 763, S_out = 232, static batches of 1-32, pipeline depths PP2 / PP4 / PP8 of an 80-layer
    70B-shaped model (40 / 20 / 10 layers per stage; TP1), prefill latency and the total over the 232 decode
    iterations, MAPE over the configurations.  Two predictions: with the peaks of MEASURED_PEAKS.json, and after the
    paper's "one-time hardware calibration (FLOPS, memory bandwidth)": effective FLOPS from ONE measured prefill and
    effective bandwidth from ONE measured decode run (20 layers, batch 32), applied to every other configuration."""
    import torch
    from paper_2606_18600_b200 import binding, placement, synth
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    pk = peaks()
    S_in, S_out = 763, 232
    depths, batches = [10, 20, 40], [1, 2, 4, 8, 16, 32]
    mk = lambda l: synth.ModelShape(shape.name, shape.hidden, shape.n_q, shape.n_kv, shape.d, shape.ffn, l, shape.eps,
                                    shape.theta, shape.qk_norm, shape.vocab)
    layers = gpu_weights(mk(max(depths)), dev, args.seed)
    g = torch.Generator(device=dev)
    g.manual_seed(args.seed + 5)
    Bmax = max(batches)
    x = torch.randn((Bmax * S_in, shape.hidden), generator=g, device=dev, dtype=torch.float32).to(torch.bfloat16)
    out = torch.empty_like(x)
    rows, launches = [], 0
    sampler = ClockSampler(0)
    sampler.start()
    for l in depths:
        for B in batches:
            lens = np.full(B, S_in, dtype=np.int32)
            pb = synth.paged_batch(np.random.default_rng(args.seed), lens, extra_tokens=S_out + 2)
            dims = binding.make_dims(shape, max_tokens=B * S_in, max_seqs=B, max_blocks=pb.max_blocks,
                                     max_pos=S_in + S_out + 64, n_layers_total=80)
            st = binding.Stage(dims, 0, l, layers[:l], None, n_pages=pb.n_pages_pool, device=dev)
            i32 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).to(dev)
            cu, zero, bt = i32(np.arange(B + 1) * S_in), i32(np.zeros(B)), i32(pb.block_tables)
            ctx = i32(S_in + np.arange(S_out)[:, None] + np.zeros((1, B), dtype=np.int32))
            T = B * S_in
            torch.cuda.synchronize(dev)
            n0 = st.launch_count()
            pre = lambda i: st.prefill(B, cu, zero, bt, T, hidden=x[:T], out_hidden=out[:T])
            pre(0)
            pre_ms = cuda_time_ms(st.stream, pre, 2) / 2
            dec = lambda i: st.decode(B, bt, ctx[i], hidden=x[i * B:(i + 1) * B], out_hidden=out[:B])
            for i in range(3):
                dec(i)
            dec_ms = cuda_time_ms(st.stream, dec, S_out)
            launches += st.launch_count() - n0
            st.destroy()
            rows.append({"layers": l, "B": B, "prefill_ms": pre_ms, "decode_total_ms": dec_ms})
    clocks = sampler.stop()
    m = placement.sp_model(shape.hidden, shape.hq, shape.hkv, shape.ffn, 0, 80, 2)
    o = placement.sp_opts(s_in=S_in, s_out=S_out, alpha_inter=0.0, beta_inter=1e30, beam=1, max_stages=8)

    def predict(flops, bw, l, B, phase):
        inst = placement.sp_instance(flops, bw, 180e9, 1, 0.0, 1.0, 1.0)
        return 1e3 * placement.stage_latency(m, inst, o, l, B, phase, False, False)

    peak_f, peak_b = pk["bf16_tflops"] * 1e12, pk["hbm_gbs"] * 1e9
    cal = next(r for r in rows if r["layers"] == 20 and r["B"] == 32)
    # one-time calibration: the estimator is linear in 1/FLOPS when compute-bound and in 1/BW when memory-bound
    f_eff = peak_f * predict(peak_f, 1e30, 20, 32, 0) / cal["prefill_ms"]
    b_eff = peak_b * predict(1e30, peak_b, 20, 32, 1) / cal["decode_total_ms"]
    errs = {"peaks": [], "calibrated": []}
    for r in rows:
        meas = r["prefill_ms"] + r["decode_total_ms"]
        for name, (f, b) in {"peaks": (peak_f, peak_b), "calibrated": (f_eff, b_eff)}.items():
            pred = predict(f, b, r["layers"], r["B"], 0) + predict(f, b, r["layers"], r["B"], 1)
            r[f"predicted_ms_{name}"] = pred
            r[f"err_pct_{name}"] = 100.0 * (pred - meas) / meas
            if not (name == "calibrated" and r is cal):
                errs[name].append(abs(pred - meas) / meas)
    return {"rows": rows, "mape_pct_peaks": 100 * float(np.mean(errs["peaks"])),
            "mape_pct_calibrated": 100 * float(np.mean(errs["calibrated"])),
            "max_err_pct_calibrated": 100 * float(np.max(errs["calibrated"])),
            "calibration": {"config": "20 layers, B=32", "flops_eff_TFLOPs": f_eff / 1e12, "bw_eff_GBs": b_eff / 1e9,
                            "peaks": {"bf16_tflops": pk["bf16_tflops"], "hbm_gbs": pk["hbm_gbs"]}},
            "launches": launches, "clocks": clocks}


def run_gemm_sustained(args, shape, len_fn, seconds=4.0):
    """The prefill projections alone, each launched back to back for >= `seconds` (so the chip sits at its power-capped
    clocks, like MEASURED_PEAKS.json's bf16_tflops_sustained), at cfg-4's token count and the 70B layer shapes, through
    the op-level C-ABI entry points (the same kernel the stage runs).  Reports TFLOP/s per projection and clocks."""
    import torch
    from paper_2606_18600_b200 import binding
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    T = int(len_fn(args.seed).sum())
    H, Hq, Hkv, F = shape.hidden, shape.hq, shape.hkv, shape.ffn
    g = torch.Generator(device=dev)
    g.manual_seed(args.seed + 3)
    rnd = lambda r, c, sd: (torch.randn((r, c), generator=g, device=dev, dtype=torch.float32) * sd).to(torch.bfloat16)
    stream = torch.cuda.Stream(device=dev)
    cases = [("gate/up + SwiGLU", True, F, H), ("down", False, H, F), ("QKV (as one [Hq+2Hkv, H] matrix)", False, Hq + 2 * Hkv, H),
             ("O", False, H, Hq)]
    rows = []
    for name, dual, N, K in cases:
        x = rnd(T, K, 1.0)
        w0 = rnd(N, K, 0.02)
        w1 = rnd(N, K, 0.02) if dual else None
        call = (lambda: binding.op_gemm_swiglu_bf16(x, w0, w1, stream=stream)) if dual else \
            (lambda: binding.op_gemm_bf16(x, w0, stream=stream))
        flops = (4 if dual else 2) * T * N * K
        with torch.cuda.stream(stream):
            for _ in range(3):
                call()
        stream.synchronize()
        one = cuda_time_ms(stream, lambda i: call(), 3) / 3
        n = max(3, int(seconds * 1e3 / one))
        sampler = ClockSampler(0)
        sampler.start()
        ms = cuda_time_ms(stream, lambda i: call(), n)
        clocks = sampler.stop()
        rows.append({"projection": name, "T": T, "N": N, "K": K, "launches": n, "seconds": ms * 1e-3,
                     "tflops_first_launches": flops / (one * 1e-3) / 1e12, "tflops_sustained": flops * n / (ms * 1e-3) / 1e12,
                     "clocks": clocks})
        del x, w0, w1
        torch.cuda.empty_cache()
    return rows


def run_tp_emulated(args, shape, ctx_fn, size=2):
    """What the fused tensor-parallel all-reduce costs in kernels and waits, measured where only one GPU exists: the
    cfg-2 stage cut into `size` shards (tp.shard_shape), every shard a stage of THIS process on its own stream of the
    ONE device, exchange buffers = plain device memory (so the "peer" stores and counters are local: no NVLink time in
    this number).  The two ranks' steps run concurrently as far as the SMs allow, so the step time is about the sum
    of the shards' work: compare with the un-sharded stage on the same box (the default workload)."""
    import torch
    from paper_2606_18600_b200 import binding, synth, tp as tpmod
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    K, W = args.steps, args.warmup
    ctx0 = ctx_fn(args.seed).astype(np.int32)
    B = len(ctx0)
    total = K + W + 4
    pb = synth.paged_batch(np.random.default_rng(args.seed), ctx0, extra_tokens=total + 1)
    sshape = tpmod.shard_shape(shape, size)
    lib = binding.load_library()
    xchg = [torch.empty(lib.ss_tp_xchg_bytes(size), dtype=torch.uint8, device=dev) for _ in range(size)]
    stages = []
    g = torch.Generator(device=dev)
    g.manual_seed(args.seed + 99)
    for r in range(size):
        layers = gpu_weights(sshape, dev, args.seed + 1000 * r)
        dims = binding.make_dims(sshape, max_tokens=B, max_seqs=B, max_blocks=pb.max_blocks,
                                 max_pos=int(ctx0.max()) + total + 64)
        st = binding.Stage(dims, 0, sshape.n_layers, layers, None, n_pages=pb.n_pages_pool, device=dev)
        _fill_randn(st.kv_pool.view(-1), g)
        stages.append(st)
    for r, st in enumerate(stages):
        st.set_tp_fused(r, size, [b.data_ptr() for b in xchg])
    x = torch.randn((B, shape.hidden), generator=g, device=dev, dtype=torch.float32).to(torch.bfloat16)
    bt = torch.from_numpy(pb.block_tables).to(dev)
    ctxs = torch.from_numpy(ctx0[None, :] + np.arange(total, dtype=np.int32)[:, None]).to(dev).contiguous()
    outs = [torch.empty((B, shape.hidden), dtype=torch.bfloat16, device=dev) for _ in range(size)]
    torch.cuda.synchronize(dev)
    no = [0]

    def step():
        for r, st in enumerate(stages):
            st.decode(B, bt, ctxs[no[0]], hidden=x, out_hidden=outs[r])
        no[0] += 1

    for _ in range(W):
        step()
    torch.cuda.synchronize(dev)
    sampler = ClockSampler(0)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in stages]
    n0 = sum(st.launch_count() for st in stages)
    for (e0, _), st in zip(ev, stages):
        e0.record(st.stream)
    for _ in range(K):
        step()
    for (_, e1), st in zip(ev, stages):
        e1.record(st.stream)
    torch.cuda.synchronize(dev)
    ms = max(e0.elapsed_time(e1) for e0, e1 in ev)
    clocks = sampler.stop()
    launches = sum(st.launch_count() for st in stages) - n0
    same = all(torch.equal(outs[r], outs[0]) for r in range(size))
    graphs = [st.graph_count() for st in stages]
    for st in stages:
        st.destroy()
    byts = decode_bytes_per_step(shape, ctx0 + W + K // 2)
    return {"ms_per_step": ms / K, "tokens_per_s": B * K / (ms * 1e-3), "launches": int(launches), "clocks": clocks,
            "ranks_bit_identical": bool(same), "decode_graphs_per_rank": graphs, "bytes_per_step": float(byts), "B": B,
            "size": size}


def run_online(args, shape, rank, world):
    """cfg5: online mixed batches (96 decode rows + <= 4 prefill chunks of <= 512 tokens per ss_stage_prefill call)
    driven by paper_2606_18600_b200/online.py over a page pool at ~85% occupancy; K timed iterations."""
    import torch
    from paper_2606_18600_b200 import binding, online
    dev = torch.device(f"cuda:{int(os.environ.get('LOCAL_RANK', 0))}")
    torch.cuda.set_device(dev)
    K, W = args.steps, args.warmup
    n_pages = online.OnlineDriver.pool_pages(args.seed)
    S = online.N_DECODE + online.N_PREFILL
    Tmax = online.N_DECODE + online.N_PREFILL * online.CHUNK
    max_blocks = (8192 + 2048 + online.CHUNK) // 16 + 2
    layers = gpu_weights(shape, dev, args.seed)
    dims = binding.make_dims(shape, max_tokens=Tmax, max_seqs=S, max_blocks=max_blocks,
                             max_pos=8192 + 2048 + online.CHUNK + 64)
    st = binding.Stage(dims, 0, shape.n_layers, layers, None, n_pages=n_pages, device=dev)
    g = torch.Generator(device=dev)
    g.manual_seed(args.seed + 99)
    _fill_randn(st.kv_pool.view(-1), g)
    bank = torch.randn((Tmax, shape.hidden), generator=g, device=dev, dtype=torch.float32).to(torch.bfloat16)
    out = torch.empty((Tmax, shape.hidden), dtype=torch.bfloat16, device=dev)
    drv = online.OnlineDriver(st, shape, seed=args.seed, max_blocks=max_blocks, device=dev)
    for _ in range(W):
        drv.step(bank, out)
    torch.cuda.synchronize(dev)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    d0, p0, n0 = drv.stats["decode_tokens"], drv.stats["prefill_tokens"], st.launch_count()
    t0 = time.perf_counter()
    for _ in range(K):                       # each step ends with a stream sync (the scheduler reads the results)
        drv.step(bank, out)
    ms = (time.perf_counter() - t0) * 1e3
    clocks = sampler.stop()
    occ = drv.stats["occupancy"][W:]
    res = {"ms": ms, "decode_tokens": drv.stats["decode_tokens"] - d0, "prefill_tokens": drv.stats["prefill_tokens"] - p0,
           "launches": st.launch_count() - n0, "clocks": clocks, "occupancy": [min(occ), float(np.mean(occ)), max(occ)],
           "dropped": drv.stats["dropped"], "preempted": drv.stats["preempted"], "finished": drv.stats["finished"],
           "pages": n_pages}
    st.destroy()
    return res


# ---------------------------------------------------------------------------------------------------------------
# CPU oracle timing (cpu_baseline leg and --impl reference): the oracle as it stands, on a bounded sample
# ---------------------------------------------------------------------------------------------------------------
def oracle_sample(workload, seed, layers_sample=1, repeats=1):
    """Time `layers_sample` decoder layers of the workload's step on the host cores with the oracle; returns
    (seconds per full-depth step extrapolated by L / layers_sample, cores, description)."""
    from oracle import Oracle, OracleDims
    from paper_2606_18600_b200 import synth
    import torch
    shape, len_fn, kind = workload_spec(workload)
    orc = Oracle("f32")
    lens = len_fn(seed).astype(np.int32)
    rng = np.random.default_rng(seed)
    dims = OracleDims(shape.hidden, shape.n_q, shape.n_kv, shape.d, shape.ffn, shape.vocab, shape.eps, shape.theta,
                      shape.qk_norm, 0)
    if kind == "decode":
        B = len(lens)
        pb = synth.paged_batch(rng, lens, extra_tokens=2)
        cu = np.arange(B + 1, dtype=np.int32)
        ctx = lens
        T = B
        desc = f"{layers_sample} of {shape.n_layers} layers of one full-batch decode step (B={B}, all contexts)"
    else:
        # prefill: the 2 shortest requests only (SURVEY §8(d) sub-instance), all their tokens
        order = np.argsort(lens)[:2]
        lens = lens[order]
        pb = synth.paged_batch(rng, lens, extra_tokens=1)
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        ctx = np.zeros_like(lens)
        T = int(lens.sum())
        desc = f"{layers_sample} of {shape.n_layers} layers, the 2 shortest of 32 requests ({T} tokens)"
    g = torch.Generator().manual_seed(seed + 5)
    pool = synth.bits(torch.randn((2, pb.n_pages_pool, shape.n_kv, 16, shape.d), generator=g).to(torch.bfloat16)).copy()
    x = synth.bf16_bits_to_f32(synth.bits(synth.hidden_rows(T, shape.hidden, seed))).copy()
    best = None
    for l in range(layers_sample):
        w = {k: (None if v is None else synth.bits(v)) for k, v in synth.layer_weights(shape, l, seed).items()}
        for _ in range(repeats):
            xx = x.copy()
            t0 = time.perf_counter()
            orc.layer(dims, w, pool[0], pool[1], cu, ctx, pb.block_tables, xx)
            dt = time.perf_counter() - t0
            best = dt if best is None else min(best, dt)
    sec_full = best * shape.n_layers
    return sec_full, T, orc.threads(), desc


def main():
    args = parse()
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    shape, len_fn, kind = workload_spec(args.workload, args.layers)
    pk = peaks()
    unit = "tokens/s"
    metric = ("stage decode tokens/s" if kind == "decode" else "migration-recompute prefill tokens/s")
    cfg = {"workload": {"cfg2": "configs[1]: Llama-3.1-70B-shaped 20-layer decode stage, B=64, ctx lognormal(med 1024)",
                        "cfg3": "configs[2]: Qwen3-32B-shaped 16-layer decode stage, B=128, ctx lognormal(med 768)",
                        "cfg4": "configs[3]: migration recompute prefill, 70B shapes, 32 requests lognormal(med 1200)",
                        "cfg5": "configs[4]: online mixed batches, Qwen3-32B shapes",
                        "migrate": "migration of one request: recomputation vs KV transfer",
                        "pipeline": "80-layer 70B-shaped model in 4 stages (even / uneven), per-stage decode latency",
                        "estimator": "estimator accuracy (Fig. 8 protocol), 70B shapes",
                        "gemm": "prefill projections alone, 70B layer shapes, T = 40,173",
                        "tp_emul": "cfg-2 stage sharded D_TP = 2, both ranks on ONE GPU (fused all-reduce exercised, no NVLink)",
                        "tiny": "configs[0]: tiny Llama-style stage"}[args.workload],
           "layers": shape.n_layers, "hidden": shape.hidden, "ffn": shape.ffn, "heads": f"{shape.n_q}/{shape.n_kv}",
           "page_size": 16, "seed": args.seed, "parallelism": f"replicas x{world}",
           "l2_policy": "inputs larger than L2 (weights 34 GB / KV streamed once per step)"}
    if args.layers:
        cfg["debug_layers_override"] = args.layers
    if args.batch_invariant:
        cfg["mode"] = "batch-invariant (ss_stage_set_batch_invariant: bit-exact migration; not the headline mode)"

    # ---------------- reference arm: the CPU oracle, rank 0 only ----------------
    if args.impl == "reference":
        if rank != 0:
            return
        if kind in ("online", "migrate", "pipeline", "estimator"):
            raise SystemExit("--impl reference covers cfg2/cfg3/cfg4/tiny (the oracle has no online driver)")
        ts = []
        T = cores = desc = None
        for i in range(max(1, min(args.steps, 3)) + min(args.warmup, 1)):
            sec, T, cores, desc = oracle_sample(args.workload, args.seed, layers_sample=1)
            ts.append(sec)
        sec = float(np.mean(ts[min(args.warmup, 1):]))
        val = T / sec
        line = {"impl": "reference", "metric": metric, "value": val, "unit": unit, "n_gpus": 0, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": cfg,
                # what actually ran: each "step" is a bounded SAMPLE (one decoder layer of the step, timed, x layers)
                "steps_run": len(ts) - min(args.warmup, 1), "warmup_run": min(args.warmup, 1), "layers_run": 1,
                "layers_per_step": shape.n_layers, "extrapolated": "ms_per_step = measured layer time x layers",
                "cpu_baseline": {"value": val, "unit": unit, "cores": cores, "kind": "oracle",
                                 "sample": desc + "; time x layers (extrapolated)"},
                "e2e": {"value": val, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line))
        return

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{int(os.environ.get('LOCAL_RANK', 0))}"))

    if kind == "migrate":
        if rank != 0:
            return
        rows = run_migrate(args, shape)
        print(json.dumps({"metric": "migration of one request: recomputation vs KV transfer (ms)", "n_gpus": 1,
                          "dtype": "bf16", "data": "synthetic",
                          "config": {"workload": "70B-shaped 20-layer stage, one request, contexts 1K-64K",
                                     "link": "modelled: NVLink 5, 900 GB/s per direction (single-GPU box)"},
                          "rows": rows}))
        return
    if kind == "tp_emul":
        if rank != 0:
            return
        r = run_tp_emulated(args, shape, len_fn)
        gbs = r["bytes_per_step"] / (r["ms_per_step"] * 1e-3) / 1e9
        print(json.dumps({"metric": "stage decode tokens/s, stage sharded D_TP = 2 with both ranks on one GPU (fused "
                                    "all-reduce path exercised end to end; no NVLink in this number)",
                          "value": r["tokens_per_s"], "unit": "tokens/s", "n_gpus": 1, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
                          "dtype": "bf16", "data": "synthetic", "gpu_launches": r["launches"], "clocks": r["clocks"],
                          "ranks_bit_identical": r["ranks_bit_identical"], "decode_graphs_per_rank": r["decode_graphs_per_rank"],
                          "step_roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm_gbs"], "unit": "GB/s",
                                            "frac": gbs / pk["hbm_gbs"]},
                          "config": dict(cfg, parallelism="tp2 emulated on one GPU")}))
        return
    if kind == "gemm":
        if rank != 0:
            return
        rows = run_gemm_sustained(args, shape, len_fn)
        tot_f = sum(r["tflops_sustained"] * r["seconds"] for r in rows)
        print(json.dumps({"metric": "prefill projections alone, sustained bf16 TFLOP/s (each launched back to back >= 4 s)",
                          "unit": "TFLOP/s", "n_gpus": 1, "dtype": "bf16", "data": "synthetic",
                          "peak_sustained": pk["bf16_tflops_sustained"], "peak_burst": pk["bf16_tflops"],
                          "peak_source": pk["source"],
                          "config": {"workload": "70B layer shapes, T = 40,173 tokens (cfg-4), op-level GEMM entry points"},
                          "rows": [dict(r, frac_of_sustained_peak=r["tflops_sustained"] / pk["bf16_tflops_sustained"])
                                   for r in rows]}))
        return
    if kind == "estimator":
        if rank != 0:
            return
        r = run_estimator(args, shape)
        print(json.dumps({"metric": "MAPE of the paper's static estimator against measured stage latency (prefill of "
                                    "763 tokens + 232 decode iterations), percent", "value": r["mape_pct_calibrated"],
                          "unit": "percent", "higher_is_better": False, "n_gpus": 1, "dtype": "bf16",
                          "data": "synthetic", "gpu_launches": int(r["launches"]), "clocks": r["clocks"],
                          "mape_pct_with_measured_peaks": r["mape_pct_peaks"],
                          "mape_pct_after_one_time_calibration": r["mape_pct_calibrated"],
                          "max_err_pct_after_calibration": r["max_err_pct_calibrated"], "calibration": r["calibration"],
                          "config": {"workload": "Fig. 8 protocol on one B200: 70B shapes, stages of 10 / 20 / 40 layers "
                                                 "(PP8 / PP4 / PP2, TP1), batch 1-32, S_in 763, S_out 232",
                                     "paper_mape_pct": 6.63}, "rows": r["rows"]}))
        return
    if kind == "pipeline":
        if rank != 0:
            return
        rows, B, launches, clocks = run_pipeline(args, shape, len_fn)
        best = max(r["tokens_per_s"] for r in rows)
        print(json.dumps({"metric": "4-stage pipeline decode tokens/s, throughput = B / (max_i L^i + hop) (Eq. 5)",
                          "value": best, "unit": "tokens/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
                          "higher_is_better": True, "dtype": "bf16", "data": "synthetic", "gpu_launches": int(launches),
                          "clocks": clocks,
                          "config": {"workload": "80-layer 70B-shaped model in 4 stages, cfg-2 micro-batch (B=64) per "
                                                 "stage per tick; stages measured one at a time on one B200, hop modelled "
                                                 "(NVLink 5: 900 GB/s + 10 us)", "micro_batches": ">= 4 (pipeline full)"},
                          "rows": rows}))
        return
    if kind == "online":
        res = run_online(args, shape, rank, world)
        ms = res["ms"]
        if world > 1:
            import torch.distributed as dist
            ms = max_over_ranks([ms], "cuda")[0]
            dist.barrier()
            dist.destroy_process_group()
        if rank != 0:
            return
        toks = res["decode_tokens"] + res["prefill_tokens"]
        cfg["workload"] = "configs[4]: online mixed batches, Qwen3-32B shapes, 96 decode + 4 prefill chunks of 512"
        line = {"metric": "online mixed-batch tokens/s (decode + prefill tokens per second of wall time, host "
                          "scheduling and per-iteration H2D of block tables inside)",
                "value": whole_job_value(toks, world, ms), "unit": "tokens/s", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16", "data": "synthetic", "config": cfg, "clocks": res["clocks"],
                "gpu_launches": int(res["launches"]),
                "decode_tokens_per_s": res["decode_tokens"] * world / (ms * 1e-3),
                "prefill_tokens_per_s": res["prefill_tokens"] * world / (ms * 1e-3),
                "pool": {"pages": res["pages"], "occupancy_min_mean_max": res["occupancy"], "dropped": res["dropped"], "preempted": res["preempted"],
                         "finished": res["finished"]}}
        print(json.dumps(line))
        return
    keep_layers = None
    if kind == "decode" and args.workload == "cfg2" and not args.no_sub and not args.tp:
        dev = torch.device(f"cuda:{int(os.environ.get('LOCAL_RANK', 0))}")
        keep_layers = gpu_weights(shape, dev, args.seed)      # cfg-4 (same 70B shapes) re-uses them below
    if args.tp and (kind != "decode" or world > 8):
        raise SystemExit("--tp applies to the decode workloads (cfg2, cfg3, tiny) on at most 8 ranks")
    res = run_decode(args, shape, len_fn, rank, world, layers=keep_layers) if kind == "decode" else \
        run_prefill(args, shape, len_fn, rank, world)
    if args.tp:
        res["tp"] = True
    K = args.steps
    ms, e2e_ms = reduce_times(res, world)
    line = None
    if rank == 0:
        line = {"metric": metric, "unit": unit, "n_gpus": world, "steps": K, "warmup": args.warmup,
                "higher_is_better": True, "scaling": "strong" if args.tp else "weak", "vs_baseline": None,
                "dtype": "bf16", "data": "synthetic", "config": cfg}
        if args.tp:
            cfg["parallelism"] = f"tp{world} (one stage sharded over {world} ranks, fused all-reduce over peer memory)"
            line["decode_graphs"] = res.get("graphs")
        line.update(decode_record(res, ms, e2e_ms, world, shape, len_fn, args, pk) if kind == "decode" else
                    prefill_record(res, ms, e2e_ms, world, shape, len_fn, args, pk))
        line["build"] = source_hash()

    # ---- the rest of BASELINE.json's metric, in the same line (default workload only): migration-recompute prefill
    # tokens/s (cfg-4, on the weights already resident) and the second decode configuration (cfg-3) --------------------
    if keep_layers is not None:
        sh4, len4, _ = workload_spec("cfg4")
        r4 = run_prefill(args, sh4, len4, rank, world, layers=keep_layers, K=2, W=1)
        ms4, e4 = reduce_times(r4, world)
        if rank == 0:
            rec = prefill_record(r4, ms4, e4, world, sh4, len4, args, pk)
            rec.update({"metric": "migration-recompute prefill tokens/s", "unit": unit, "steps": 2, "warmup": 1,
                        "workload": "configs[3]: migration recompute prefill, 70B shapes, 20 layers, 32 requests "
                                    "lognormal(med 1200), 40,173 tokens"})
            line["prefill"] = rec
        del keep_layers
        torch.cuda.empty_cache()
        sh3, len3, _ = workload_spec("cfg3")
        r3 = run_decode(args, sh3, len3, rank, world, K=max(K, 10), W=max(args.warmup, 3))
        ms3, e3 = reduce_times(r3, world)
        if rank == 0:
            rec = decode_record(r3, ms3, e3, world, sh3, len3, args, pk, workload="cfg3")
            rec.update({"metric": "stage decode tokens/s", "unit": unit, "steps": r3["K"], "warmup": r3["W"],
                        "workload": "configs[2]: Qwen3-32B-shaped 16-layer decode stage, B=128, ctx lognormal(med 768)"})
            line["cfg3"] = rec
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    if not args.no_cpu_baseline and world == 1:
        sec, T, cores, desc = oracle_sample(args.workload, args.seed, layers_sample=1)
        line["cpu_baseline"] = {"value": T / sec, "unit": unit, "cores": cores, "kind": "oracle",
                                "sample": desc + "; time x layers (extrapolated)"}
    print(json.dumps(line))


def reduce_times(res, world):
    """(device-timed ms, e2e ms per step) as the MAX over ranks (replicas: the slowest one is the job's time)."""
    ms = res["ms"]
    e2e_ms = res["e2e"]["ms_per_step"] if res["e2e"] else None
    if world > 1:
        ms, e2e_max = max_over_ranks([ms, e2e_ms or 0.0], "cuda")
        e2e_ms = e2e_max if e2e_ms is not None else None
    return ms, e2e_ms


def _common_record(res, ms, e2e_ms, world):
    K = res["K"]
    if res.get("tp"):
        world = 1            # tensor parallelism: the N ranks process ONE batch together
    rec = {"value": whole_job_value(res["tokens"], world, ms), "ms_per_step": ms / K, "clocks": res["clocks"],
           "gpu_launches": res["launches"], "output_checksum_mean_abs": res["checksum"]}
    if res["e2e"]:
        rec["e2e"] = {"value": res["tokens"] * world / K / (e2e_ms * 1e-3), "unit": "tokens/s",
                      "h2d_bytes_per_step": int(res["e2e"]["h2d"]), "d2h_bytes_per_step": int(res["e2e"]["d2h"])}
    return rec


def decode_record(res, ms, e2e_ms, world, shape, len_fn, args, pk, workload=None):
    from paper_2606_18600_b200 import estimator
    K = res["K"]
    rec = _common_record(res, ms, e2e_ms, world)
    dom = res["dominant"]
    if dom:
        ach = dom["bytes"] / (dom["us"] * 1e-6) / 1e9
        traffic, label = ncu_traffic(workload or args.workload)
        rec["roofline"] = {"bound": "hbm", "achieved": ach, "peak": pk["hbm_gbs"], "unit": "GB/s",
                           "frac": ach / pk["hbm_gbs"], "traffic": traffic, "traffic_source": label,
                           "algorithmic_bytes": dom["bytes"], "kernel": dom["kernel"], "us_per_launch": dom["us"],
                           "peak_source": pk["source"]}
    step_gbs = res["bytes_per_step"] / (ms / K * 1e-3) / 1e9
    n_hbm = world if res.get("tp") else 1      # a tensor-parallel stage streams its bytes from all N ranks' HBM
    rec["step_roofline"] = {"bound": "hbm", "algorithmic_GB_per_step": res["bytes_per_step"] / 1e9,
                            "achieved": step_gbs, "peak": pk["hbm_gbs"] * n_hbm, "unit": "GB/s",
                            "frac": step_gbs / (pk["hbm_gbs"] * n_hbm)}
    rec["paper_estimator_ms"] = estimator.decode_step_ms(shape, len_fn(args.seed), pk["bf16_tflops"] * 1e12,
                                                         pk["hbm_gbs"] * 1e9)
    return rec


def prefill_record(res, ms, e2e_ms, world, shape, len_fn, args, pk):
    from paper_2606_18600_b200 import estimator
    K = res["K"]
    rec = _common_record(res, ms, e2e_ms, world)
    tf = res["flops_per_step"] / (ms / K * 1e-3) / 1e12
    rec["roofline"] = {"bound": "tensor", "achieved": tf, "peak": pk["bf16_tflops_sustained"], "unit": "TFLOP/s",
                       "frac": tf / pk["bf16_tflops_sustained"], "traffic": None,
                       "kernel": "whole prefill step (GEMMs 98.4% of flops)", "peak_source": pk["source"],
                       "peak_kind": "sustained (a >1 s step under the power cap)",
                       "frac_of_burst_peak": tf / pk["bf16_tflops"]}
    rec["paper_estimator_ms"] = estimator.prefill_ms(shape, len_fn(args.seed), pk["bf16_tflops"] * 1e12,
                                                     pk["hbm_gbs"] * 1e9)
    return rec


if __name__ == "__main__":
    main()
