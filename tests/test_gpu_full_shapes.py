"""Parity at BASELINE.json's FULL layer shapes, in the launch configuration bench.py times (148-CTA stream-K GEMMs
with two issuers at decode, band-rasterised 128x256 tiles at prefill, CUDA-graph replay with PDL edges), against
the CPU oracle.  The oracle cannot run 20 layers x 34 GB in a test, so each case runs a 1-2 layer stage of the real
width (hidden 8192 / 5120, FFN 28672 / 25600, 64/8 heads of 128) on the seed-0 workload draws; every decode row is
compared, and for the 40,173-token recompute the rows of the two shortest requests (sequences are independent:
oracle pin P9).  Tolerances: north_star's 2e-2 per stage / 1e-2 per layer (reading A15), KV pages per reading A13.
"""
import numpy as np
import pytest
import torch

from oracle import Oracle
from paper_2606_18600_b200 import synth
from tests import helpers as hp

pytestmark = pytest.mark.gpu
F32 = Oracle("f32")
ESCAPE_FRAC = 2e-2   # at most this fraction of first-layer K/V values may rely on the absolute bound (reading A13 ii)


def _sub(shape, L):
    return synth.ModelShape(shape.name, shape.hidden, shape.n_q, shape.n_kv, shape.d, shape.ffn, L, shape.eps,
                            shape.theta, shape.qk_norm, shape.vocab)


def _check_new_kv(gh, shape, pool_before, pool_oracle_r1, pool_gpu, ctx, bt, layer0_only=True):
    """A13: (i) the GPU modified exactly the slots the oracle modified; (iii) layer-0 values equal or adjacent."""
    changed_gpu = pool_gpu != pool_before
    changed_orc = pool_oracle_r1 != pool_before
    # a slot whose new value happens to equal the old bits is not 'changed' on either side: compare supports via
    # the slot mask the block table defines
    mask = np.zeros(pool_before.shape[2:5:2], dtype=bool)  # [pages, 16]
    for b, c in enumerate(ctx):
        mask[bt[b, c >> 4], c & 15] = True
    outside = ~mask[None, None, :, None, :, None]
    assert not (changed_gpu & outside).any(), "GPU wrote outside the new tokens' slots"
    assert not (changed_orc & outside).any()
    sel = np.broadcast_to(mask[None, None, :, None, :, None], pool_before.shape)
    L = pool_before.shape[0]
    ulp = gh.bf16_ulp_distance(pool_gpu[sel], pool_oracle_r1[sel]).reshape(L, -1)
    a = synth.bf16_bits_to_f32(pool_gpu[sel]).reshape(L, -1)
    b = synth.bf16_bits_to_f32(pool_oracle_r1[sel]).reshape(L, -1)
    # near zero (cancellation in RoPE / the projections) an absolute bound replaces the ulp bound, as in
    # tests/test_gpu_parity.py::_check_kv
    esc0 = (ulp[0] > 1) & (np.abs(a[0] - b[0]) <= 2e-3 * np.abs(b[0]).max())
    ok0 = (ulp[0] <= 1) | esc0
    eq0 = float((ulp[0] == 0).mean())
    print(f"new KV, layer 0: equal {eq0:.4f}, <= 1 ulp {float((ulp[0] <= 1).mean()):.4f}, only via the 2e-3 absolute "
          f"bound {float(esc0.mean()):.4f}, outside both: {int((~ok0).sum())}; "
          f"deeper layers max abs diff {float(np.abs(a - b).max()):.3e} (scale {float(np.abs(b).max()):.2f})")
    # at K = 8192 the tensor cores' fp32 accumulation differs from the CPU loop by ~2e-4 relative, so ~6% of the
    # bf16 roundings land on the neighbouring value (measured 0.94 equal at cfg-2; 0.97+ at the tiny width); values
    # near zero differ by more than one of THEIR ulps and pass through the absolute bound: counted, bounded (A13 ii)
    assert ok0.all() and eq0 >= 0.90 and esc0.mean() <= ESCAPE_FRAC
    assert (np.abs(a - b) <= 1e-2 * np.abs(b).max()).all()


@pytest.mark.parametrize("name", ["cfg2", "cfg3"])
def test_full_width_decode_step_vs_oracle(name):
    from tests import gpu_helpers as gh
    full, ctx_fn = (synth.LLAMA70B, synth.cfg2_contexts) if name == "cfg2" else (synth.QWEN32B, synth.cfg3_contexts)
    shape = _sub(full, 2)
    ctx = ctx_fn(0).astype(np.int32)
    B = len(ctx)
    rng = np.random.default_rng(0)
    pb = synth.paged_batch(rng, ctx, extra_tokens=2)
    P = gh.Problem(shape, 0, n_pages=pb.n_pages_pool, max_tokens=B, max_seqs=B, max_blocks=pb.max_blocks,
                   pool_fill="random")
    try:
        x = synth.bits(synth.hidden_rows(B, shape.hidden, 0))
        pool_before = P.pool_cpu.copy()
        pool_r0 = pool_before.copy()
        want, _ = hp.run_oracle_decode(F32, shape, P.wb, pool_r0, ctx, pb.block_tables, x)
        pool_r1 = pool_before.copy()
        hp.run_oracle_decode(F32, shape, P.wb, pool_r1, ctx, pb.block_tables, x, rounding=1)
        got = P.decode(ctx, pb.block_tables, x)
        got2 = P.decode(ctx, pb.block_tables, x)          # graph replay on the same inputs: same bits
        assert np.array_equal(got, got2)
        err = hp.rel_err_rows(got, want)
        l2 = float(np.linalg.norm(got - want) / np.linalg.norm(want))
        print(f"{name}: 2-layer full-width decode, B={B}: max row rel err {err:.3e}, l2 rel {l2:.3e}")
        assert err < 2e-2
        _check_new_kv(gh, shape, pool_before, pool_r1, P.pool_bits(), ctx, pb.block_tables)
    finally:
        P.close()


@pytest.mark.parametrize("name,b_max,batches", [("cfg3", 256, (1, 5, 32, 33, 96, 129, 224, 256)),
                                                ("cfg2", 160, (1, 3, 17, 48, 65, 128, 160))])
def test_full_width_decode_batch_sizes_vs_oracle(name, b_max, batches):
    """The decode plans change with the batch size (GEMM token-tile width 32 ... 256, stream-K grids, consumer-side
    reduction, attention page split); bench.py times only B = 64 / 128.  Rows are independent of the batch they sit in
    (oracle pin P9), so the oracle runs once on b_max rows and every prefix B of them, decoded by the GPU from the same
    pool, is held to the stage tolerance; graph replay of the same batch gives the same bits."""
    from tests import gpu_helpers as gh
    full = synth.LLAMA70B if name == "cfg2" else synth.QWEN32B
    shape = _sub(full, 2)
    rng = np.random.default_rng(5)
    ctx = synth.lognormal_lengths(rng, b_max, 400, 16, 2048).astype(np.int32)
    pb = synth.paged_batch(rng, ctx, extra_tokens=2)
    P = gh.Problem(shape, 0, n_pages=pb.n_pages_pool, max_tokens=b_max, max_seqs=b_max, max_blocks=pb.max_blocks,
                   pool_fill="random")
    try:
        x = synth.bits(synth.hidden_rows(b_max, shape.hidden, 5))
        pool_before = P.pool_cpu.copy()
        want, _ = hp.run_oracle_decode(F32, shape, P.wb, pool_before.copy(), ctx, pb.block_tables, x)
        snap = P.stage.pool_view().clone()
        for B in batches:
            P.stage.pool_view().copy_(snap)
            torch.cuda.synchronize()
            got = P.decode(ctx[:B], pb.block_tables[:B], x[:B])
            P.stage.pool_view().copy_(snap)
            torch.cuda.synchronize()
            assert np.array_equal(got, P.decode(ctx[:B], pb.block_tables[:B], x[:B]))
            err = hp.rel_err_rows(got, want[:B])
            print(f"{name} width, 2 layers, B={B}: max row rel err vs R0 {err:.3e}")
            assert np.isfinite(got).all() and err < 2e-2, (B, err)
    finally:
        P.close()


def test_full_width_recompute_prefill_and_migration_vs_oracle():
    """cfg-4: one ss_stage_prefill over all 32 migrated requests (40,173 tokens, packed varlen), then one decode
    step; the oracle follows the two shortest requests through the same two calls."""
    from tests import gpu_helpers as gh
    shape = _sub(synth.LLAMA70B, 1)
    lens = synth.cfg4_lengths(0).astype(np.int32)
    n, T = len(lens), int(lens.sum())
    rng = np.random.default_rng(0)
    pb = synth.paged_batch(rng, lens, extra_tokens=2)
    P = gh.Problem(shape, 0, n_pages=pb.n_pages_pool, max_tokens=T, max_seqs=n, max_blocks=pb.max_blocks)
    try:
        g = torch.Generator().manual_seed(77)
        x = synth.bits(synth.randn_bf16((T + n, shape.hidden), 1.0, g))
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        got = P.prefill(lens, pb.block_tables, x[:T])
        assert np.isfinite(got).all()
        got_d = P.decode(lens, pb.block_tables, x[T:])
        assert np.isfinite(got_d).all()
        pool_gpu = P.pool_bits()

        pick = np.argsort(lens)[:2]
        rows = np.concatenate([np.arange(cu[s], cu[s + 1]) for s in pick])
        sub_lens, sub_bt = lens[pick], pb.block_tables[pick]
        pool = hp.new_pool(shape, pb.n_pages_pool, 1)
        want, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool, sub_lens, sub_bt, x[rows])
        pool_r1 = hp.new_pool(shape, pb.n_pages_pool, 1)
        want1, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool_r1, sub_lens, sub_bt, x[rows], rounding=1)
        err, err1, floor = (hp.rel_err_rows(got[rows], want), hp.rel_err_rows(got[rows], want1),
                            hp.rel_err_rows(want1, want))
        print(f"cfg4: recompute prefill, {len(rows)} oracle-checked rows of {T}: max row rel err vs R0 {err:.3e}, "
              f"vs R1 {err1:.3e}; R1 vs R0 (what bf16 operands alone cost) {floor:.3e}")
        # DESIGN.md reading A15b: at this width and with N(0, 0.02) weights (activations grow ~5x per layer, sharp
        # softmax) rounding the GEMM operands to bf16 — which the paper's BF16 engine does and the oracle's R1 mode
        # restates — moves a layer's output by 1.5e-2 of the row maximum by itself, so the 1e-2 per-layer bound is
        # judged against R1 here; against R0 the 1-layer stage must meet the stage bound and not exceed that floor.
        assert err1 < 1e-2 and err < 2e-2 and err <= 1.1 * floor
        want_d, _ = hp.run_oracle_decode(F32, shape, P.wb, pool, sub_lens, sub_bt, x[T + pick])
        want_d1, _ = hp.run_oracle_decode(F32, shape, P.wb, pool_r1, sub_lens, sub_bt, x[T + pick], rounding=1)
        err_d, err_d1 = hp.rel_err_rows(got_d[pick], want_d), hp.rel_err_rows(got_d[pick], want_d1)
        print(f"cfg4: decode step after the recompute, 2 oracle-checked rows: vs R0 {err_d:.3e}, vs R1 {err_d1:.3e}")
        assert err_d1 < 1e-2 and err_d < 2e-2
        # logical KV of the two requests (prompt + the decoded token): equal or adjacent bf16 values (A13 iii)
        for i, s in enumerate(pick):
            for kv in range(2):
                a = hp.logical_kv(pool_gpu[0, kv], pb.block_tables[s], int(lens[s]) + 1)
                b = hp.logical_kv(pool_r1[0, kv], sub_bt[i], int(lens[s]) + 1)
                ulp = gh.bf16_ulp_distance(a, b)
                fa, fb = synth.bf16_bits_to_f32(a), synth.bf16_bits_to_f32(b)
                esc = (ulp > 1) & (np.abs(fa - fb) <= 2e-3 * np.abs(fb).max())
                ok = (ulp <= 1) | esc
                print(f"request {int(s)} {'KV'[kv]}: equal {float((ulp == 0).mean()):.4f}, <= 1 ulp "
                      f"{float((ulp <= 1).mean()):.4f}, only via the absolute bound {float(esc.mean()):.4f}")
                assert ok.all() and (ulp == 0).mean() >= 0.90 and esc.mean() <= ESCAPE_FRAC, (int(s), kv, int((~ok).sum()))
        # pages of no sequence keep the sentinel (indexing, A13 i)
        used = np.zeros(pb.n_pages_pool, dtype=bool)
        for s in range(n):
            used[pb.block_tables[s, : (int(lens[s]) + 1 + 15) // 16]] = True
        assert (pool_gpu[:, :, ~used] == 0x7FC1).all()
    finally:
        P.close()


@pytest.mark.parametrize("T_target", [120, 300, 512, 513, 777, 1100, 2144, 5000])
def test_full_width_prefill_token_counts_vs_oracle(T_target):
    """The prefill plans change with the token count: one token tile up to 256, single-CTA tiles / stream-K up to 512,
    CTA pairs above (256-token tiles with a ragged last one), few or many attention items.  bench.py times 40,173 tokens
    only.  A packed batch of T_target tokens (two short sequences and fillers of mixed lengths) at the cfg-2 layer
    shapes; the oracle follows the two short sequences (sequences are independent, pin P9)."""
    from tests import gpu_helpers as gh
    shape = _sub(synth.LLAMA70B, 1)
    rng = np.random.default_rng(T_target)
    lens = [23, 40]
    while sum(lens) < T_target:
        lens.append(int(min(rng.integers(1, 700), T_target - sum(lens))))
    lens = np.array(lens, dtype=np.int32)
    order = rng.permutation(len(lens))
    lens = lens[order]
    n, T = len(lens), int(lens.sum())
    assert T == T_target
    pb = synth.paged_batch(rng, lens, extra_tokens=2)
    P = gh.Problem(shape, 0, n_pages=pb.n_pages_pool, max_tokens=T, max_seqs=max(n, 16), max_blocks=pb.max_blocks)
    try:
        g = torch.Generator().manual_seed(T_target)
        x = synth.bits(synth.randn_bf16((T, shape.hidden), 1.0, g))
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        got = P.prefill(lens, pb.block_tables, x)
        assert np.isfinite(got).all()
        assert np.array_equal(got, P.prefill(lens, pb.block_tables, x))   # same call again: same bits
        pick = np.argsort(lens, kind="stable")[:2]
        rows = np.concatenate([np.arange(cu[s], cu[s + 1]) for s in pick])
        pool = hp.new_pool(shape, pb.n_pages_pool, 1)
        want, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool, lens[pick], pb.block_tables[pick], x[rows])
        pool_r1 = hp.new_pool(shape, pb.n_pages_pool, 1)
        want1, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool_r1, lens[pick], pb.block_tables[pick], x[rows], rounding=1)
        err, err1, floor = (hp.rel_err_rows(got[rows], want), hp.rel_err_rows(got[rows], want1),
                            hp.rel_err_rows(want1, want))
        print(f"T={T} ({n} sequences): {len(rows)} oracle-checked rows: vs R0 {err:.3e}, vs R1 {err1:.3e}, floor {floor:.3e}")
        # per-layer bound against R1 (reading A15b), stage bound against R0, and within 1.3 x the oracle's own floor
        # (the factor of reading A15d) where that floor exceeds the per-layer bound
        assert err1 < 1e-2 and err < 2e-2 and err <= 1.3 * max(floor, 1e-2)
        used = np.zeros(pb.n_pages_pool, dtype=bool)
        for s in range(n):
            used[pb.block_tables[s, : (int(lens[s]) + 15) // 16]] = True
        assert (P.pool_bits()[:, :, ~used] == 0x7FC1).all()
    finally:
        P.close()


def test_full_width_migration_recompute_equals_incremental_on_gpu():
    """The migration invariant (oracle pin P7) GPU against GPU at the paper's width: the two shortest
    cfg-4 requests, one 70B-shaped layer.  (a) recompute = one ss_stage_prefill over prompt + 3 generated tokens;
    (b) incremental = prefill of the prompt, then 3 ss_stage_decode steps.  The two must leave the same logical KV
    (equal or within 2 bf16 ulp; the prefill tiles schedule and the decode stream-K cut sum in different orders) and
    the same next-token hidden state within the stage tolerance; both match the oracle, for which the two paths are
    bit-identical."""
    from tests import gpu_helpers as gh
    shape = _sub(synth.LLAMA70B, 1)
    lens_all = synth.cfg4_lengths(0).astype(np.int32)
    lens = np.sort(lens_all)[:2].astype(np.int32)
    gen = 3
    prompt = lens - gen
    n, T = len(lens), int(lens.sum())
    pb = synth.paged_batch(np.random.default_rng(5), lens, extra_tokens=2)
    mk = lambda: gh.Problem(shape, 0, n_pages=pb.n_pages_pool, max_tokens=T, max_seqs=n, max_blocks=pb.max_blocks)
    P, Q = mk(), mk()
    try:
        g = torch.Generator().manual_seed(78)
        x = synth.bits(synth.randn_bf16((T + n, shape.hidden), 1.0, g))
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
        bt = pb.block_tables
        P.prefill(lens, bt, x[:T])                                                     # (a)
        rows = np.concatenate([np.arange(cu[s], cu[s] + prompt[s]) for s in range(n)])
        Q.prefill(prompt, bt, x[rows])                                                 # (b)
        for k in range(gen):
            Q.decode(prompt + k, bt, x[np.array([cu[s] + prompt[s] + k for s in range(n)])])
        pa, pq = P.pool_bits(), Q.pool_bits()
        for s in range(n):
            for kv in range(2):
                a = hp.logical_kv(pa[0, kv], bt[s], int(lens[s]))
                b = hp.logical_kv(pq[0, kv], bt[s], int(lens[s]))
                ulp = gh.bf16_ulp_distance(a, b)
                fa, fb = synth.bf16_bits_to_f32(a), synth.bf16_bits_to_f32(b)
                esc = (ulp > 2) & (np.abs(fa - fb) <= 4e-3 * np.abs(fb).max())
                print(f"request {s} {'KV'[kv]} recompute vs incremental: equal {float((ulp == 0).mean()):.4f}, <= 2 ulp "
                      f"{float((ulp <= 2).mean()):.4f}, only via the absolute bound {float(esc.mean()):.4f}")
                assert ((ulp <= 2) | esc).all() and (ulp == 0).mean() >= 0.90 and esc.mean() <= ESCAPE_FRAC
        ya, yq = P.decode(lens, bt, x[T:]), Q.decode(lens, bt, x[T:])
        pool = hp.new_pool(shape, pb.n_pages_pool, 1)
        hp.run_oracle_prefill(F32, shape, P.wb, pool, lens, bt, x[:T])
        want, _ = hp.run_oracle_decode(F32, shape, P.wb, pool, lens, bt, x[T:])
        e_ab, e_a, e_b = hp.rel_err_rows(ya, yq), hp.rel_err_rows(ya, want), hp.rel_err_rows(yq, want)
        print(f"next-token hidden: recompute vs incremental {e_ab:.3e}; vs oracle R0 {e_a:.3e} / {e_b:.3e}")
        assert e_ab < 2e-2 and e_a < 2e-2 and e_b < 2e-2
    finally:
        P.close()
        Q.close()


def test_full_vocab_logits_and_argmax_vs_oracle():
    """S11 at the real width (Table 2 'Logits Calculation'; reading A12: V = 128,256 with the
    Llama shapes, A14 for the argmax): a 1-layer stage with final norm + lm_head, one decode step of 64 rows."""
    from tests import gpu_helpers as gh
    shape = _sub(synth.LLAMA70B, 1)
    assert shape.vocab == 128256
    ctx = np.minimum(synth.cfg2_contexts(0), 600).astype(np.int32)      # the tail does not depend on the context
    B = len(ctx)
    rng = np.random.default_rng(1)
    pb = synth.paged_batch(rng, ctx, extra_tokens=2)
    P = gh.Problem(shape, 0, n_pages=pb.n_pages_pool, max_tokens=B, max_seqs=B, max_blocks=pb.max_blocks,
                   pool_fill="random", with_edge=True)
    try:
        x = synth.bits(synth.hidden_rows(B, shape.hidden, 3))
        eb = {k: synth.bits(v) for k, v in P.edge_cpu.items()}
        pool = P.pool_cpu.copy()
        y, _ = hp.run_oracle_decode(F32, shape, P.wb, pool, ctx, pb.block_tables, x)
        wl, wa, wm = F32.logits(hp.odims(shape), y, eb["final_norm"], eb["lm_head"])
        _, lg, am = P.decode(ctx, pb.block_tables, x, logits=True)
        # (i) the argmax kernel is bit-exact on the GPU's own fp32 logits, ties -> lowest index
        assert np.array_equal(am, np.argmax(lg, axis=1).astype(np.int32))
        # (ii) ids equal the oracle's wherever the oracle's top-2 margin exceeds 8x the measured logit error
        lerr = float(np.abs(lg - wl).max())
        safe = wm > 8 * lerr
        print(f"V={shape.vocab}: logit max abs err {lerr:.3e} (logit scale {float(np.abs(wl).max()):.2f}); "
              f"rows over margin {int(safe.sum())}/{B}; argmax equal on {int((am == wa).sum())}/{B} rows")
        assert np.array_equal(am[safe], wa[safe])
        assert hp.rel_err_rows(lg, wl) < 2e-2
    finally:
        P.close()
