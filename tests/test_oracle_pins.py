"""Pins of the CPU oracle (oracle/stage_oracle.c) to things other than itself — DESIGN.md "Pins" P1-P13.

Each test cites what it pins.  None of these touches CUDA.  Library routines used as independent second
implementations: numpy float64 matmul / einsum, torch CPU scaled_dot_product_attention, and randomly initialised
`transformers` Llama / Qwen3 decoder layers loaded with the same tensors (conventions A10, A11, A16).
"""
import numpy as np
import pytest
import torch

from oracle import Oracle, OracleDims
from paper_2606_18600_b200 import synth
from tests import helpers as hp

F32 = Oracle("f32")
F64 = Oracle("f64")


def f32_of_bits(b):
    return synth.bf16_bits_to_f32(np.asarray(b))


# ---------------------------------------------------------------------------------------------------------------
# bf16 conversion: exact widening, round-to-nearest-even on store (arithmetic contract; reading A13)
# ---------------------------------------------------------------------------------------------------------------
def test_bf16_rne_golden_ties():
    # golden/bf16_rne.txt: hand-derived from the IEEE-754 bit layout (8-bit mantissa of bf16), cited there
    rows = [l.split() for l in open("tests/golden/bf16_rne.txt") if l.strip() and not l.startswith("#")]
    assert len(rows) >= 8
    for f32_hex, bf16_hex in rows:
        f = np.array([int(f32_hex, 16)], dtype=np.uint32).view(np.float32)[0]
        assert F32.f32_to_bf16(float(f)) == int(bf16_hex, 16), (f32_hex, bf16_hex)


def test_bf16_rne_matches_torch_conversion():
    g = torch.Generator().manual_seed(1)
    x = torch.randn(20000, generator=g) * torch.logspace(-20, 20, 20000)
    want = x.to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    got = np.array([F32.f32_to_bf16(float(v)) for v in x.numpy()], dtype=np.uint16)
    assert np.array_equal(got, want)
    back = np.array([F32.bf16_to_f32(int(b)) for b in got[:2000]], dtype=np.float32)
    assert np.array_equal(back, f32_of_bits(got[:2000]))


# ---------------------------------------------------------------------------------------------------------------
# P1: projections vs numpy float64 matmul, incl. K = 688 / N = 688 tails (Table 2 GEMM rows)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T,N,K", [(1, 8, 16), (5, 688, 256), (7, 256, 688), (3, 33, 1000), (64, 130, 17)])
def test_P1_matmul_vs_numpy(T, N, K):
    rng = np.random.default_rng(T * 1000 + N + K)
    x = rng.standard_normal((T, K))
    w = torch.from_numpy(rng.standard_normal((N, K)).astype(np.float32)).to(torch.bfloat16)
    wb = synth.bits(w)
    want = x @ f32_of_bits(wb).astype(np.float64).T
    got64 = F64.matmul(x, wb)
    assert np.allclose(got64, want, rtol=1e-12, atol=1e-12)
    got32 = F32.matmul(x.astype(np.float32), wb)
    want32 = x.astype(np.float32).astype(np.float64) @ f32_of_bits(wb).astype(np.float64).T
    assert np.allclose(got32, want32, rtol=0, atol=2e-5 * np.sqrt(K))
    # a transposed operand or a dropped tail fails: perturb the last k and the last n
    x2 = x.copy()
    x2[:, -1] += 1.0
    d = F64.matmul(x2, wb) - got64
    assert np.allclose(d, f32_of_bits(wb)[:, -1].astype(np.float64)[None, :].repeat(T, 0), atol=1e-12)


# ---------------------------------------------------------------------------------------------------------------
# P2: RMSNorm closed forms and invariants (steps S1/S8; the paper is silent, reading A1/A8)
# ---------------------------------------------------------------------------------------------------------------
def test_P2_rmsnorm_closed_forms():
    n, eps = 256, 1e-5
    ones = synth.bits(torch.ones(n).to(torch.bfloat16))
    gains = synth.bits(synth.randn_bf16((n,), 0.02, torch.Generator().manual_seed(3), mean=1.0))
    gv = f32_of_bits(gains).astype(np.float64)
    for c in (0.5, -3.0, 17.0):
        out = F64.rmsnorm(np.full((2, n), c), gains, eps)
        assert np.allclose(out, c / np.sqrt(c * c + eps) * gv[None, :], rtol=1e-13)
    rng = np.random.default_rng(0)
    x = rng.standard_normal((9, n)) * 3.0
    out = F64.rmsnorm(x, ones, eps)
    ms = (x * x).mean(axis=1)
    assert np.allclose(np.sqrt((out * out).mean(axis=1)), 1 / np.sqrt(1 + eps / ms), rtol=1e-12)
    # scale invariance up to the eps term
    assert np.allclose(F64.rmsnorm(1e3 * x, gains, eps), F64.rmsnorm(x, gains, eps), rtol=1e-4)
    # library second opinion
    want = torch.nn.functional.rms_norm(torch.from_numpy(x), (n,), torch.from_numpy(gv), eps).numpy()
    assert np.allclose(F64.rmsnorm(x, gains, eps), want, rtol=1e-12)
    assert np.allclose(F32.rmsnorm(x.astype(np.float32), gains, eps), want, rtol=2e-5, atol=1e-6)


def test_P2_head_rmsnorm_is_rmsnorm_per_head():
    rng = np.random.default_rng(4)
    u = rng.standard_normal((5, 3, 64))
    g = synth.bits(synth.randn_bf16((64,), 0.02, torch.Generator().manual_seed(5), mean=1.0))
    got = F64.head_rmsnorm(u, g, 1e-6)
    want = F64.rmsnorm(u.reshape(15, 64), g, 1e-6).reshape(5, 3, 64)
    assert np.array_equal(got, want)


# ---------------------------------------------------------------------------------------------------------------
# P3: RoPE invariants (step S4; reading A10: rotate-half pairing, no frequency rescaling)
# ---------------------------------------------------------------------------------------------------------------
def test_P3_rope_invariants():
    rng = np.random.default_rng(7)
    d, theta = 64, 5e5
    q = rng.standard_normal((6, 2, d))
    k = rng.standard_normal((6, 2, d))
    # position 0 is the identity
    assert np.array_equal(F64.rope(q, np.zeros(6, np.int32), theta), q)
    pos_m = np.array([3, 10, 100, 1000, 4000, 8000], dtype=np.int32)
    pos_n = np.array([1, 7, 50, 999, 17, 8191], dtype=np.int32)
    qm, kn = F64.rope(q, pos_m, theta), F64.rope(k, pos_n, theta)
    # per-pair norm preserved
    h = d // 2
    assert np.allclose(qm[..., :h] ** 2 + qm[..., h:] ** 2, q[..., :h] ** 2 + q[..., h:] ** 2, rtol=1e-12)
    # <R_m q, R_n k> depends only on m - n: shift both by 123
    qm2, kn2 = F64.rope(q, pos_m + 123, theta), F64.rope(k, pos_n + 123, theta)
    assert np.allclose((qm * kn).sum(-1), (qm2 * kn2).sum(-1), rtol=1e-9, atol=1e-9)
    # R_a R_b = R_{a+b}
    assert np.allclose(F64.rope(F64.rope(q, pos_m, theta), pos_n, theta), F64.rope(q, pos_m + pos_n, theta),
                       rtol=1e-9, atol=1e-9)
    # explicit angle for one element: pair (c, c+h) at position p rotates by p * theta^(-2c/d)
    c, p = 5, 1000
    e = np.zeros((1, 1, d))
    e[0, 0, c] = 1.0
    r = F64.rope(e, np.array([p], np.int32), theta)
    ang = p * theta ** (-2.0 * c / d)
    assert np.allclose([r[0, 0, c], r[0, 0, c + h]], [np.cos(ang), np.sin(ang)], atol=1e-12)
    # inv_freq override is used verbatim
    inv = (theta ** (-2.0 * np.arange(h) / d)).astype(np.float32)
    # fp32 inv_freq: angle error <= pos * 2^-24 ~ 5e-4 rad at pos 8000
    assert np.allclose(F64.rope(q, pos_m, theta, inv), qm, rtol=0, atol=4e-3)
    assert np.allclose(F64.rope(q[:2], pos_m[:2], theta, inv[:]), qm[:2], rtol=0, atol=1e-5)


# ---------------------------------------------------------------------------------------------------------------
# helpers for attention pins
# ---------------------------------------------------------------------------------------------------------------
def _rand_pool(n_pages, n_kv, d, seed):
    g = torch.Generator().manual_seed(seed)
    kp = synth.bits(torch.randn((n_pages, n_kv, 16, d), generator=g).to(torch.bfloat16)).copy()
    vp = synth.bits(torch.randn((n_pages, n_kv, 16, d), generator=g).to(torch.bfloat16)).copy()
    return kp, vp


def _dense_attention(q, kp, vp, cu, ctx_before, bt, n_q, n_kv, d):
    """P5 brute force: gather pages to dense, full masked score matrix, softmax, multiply — numpy float64."""
    G = n_q // n_kv
    out = np.zeros((cu[-1], n_q, d))
    for s in range(len(ctx_before)):
        qs = q[cu[s]:cu[s + 1]]                                   # [ql, n_q, d]
        ql = qs.shape[0]
        Ltot = ctx_before[s] + ql
        K = f32_of_bits(hp.logical_kv(kp, bt[s], Ltot)).astype(np.float64)   # [L, n_kv, d]
        V = f32_of_bits(hp.logical_kv(vp, bt[s], Ltot)).astype(np.float64)
        K = np.repeat(K, G, axis=1)
        V = np.repeat(V, G, axis=1)
        S = np.einsum("ihc,jhc->hij", qs, K) / np.sqrt(d)          # [n_q, ql, L]
        ii = ctx_before[s] + np.arange(ql)[:, None]
        jj = np.arange(Ltot)[None, :]
        S = np.where(jj <= ii, S, -np.inf)
        P = np.exp(S - S.max(-1, keepdims=True))
        P /= P.sum(-1, keepdims=True)
        out[cu[s]:cu[s + 1]] = np.einsum("hij,jhc->ihc", P, V)
    return out


# ---------------------------------------------------------------------------------------------------------------
# P4: softmax rows, degenerate cases (step S6; north_star: "softmax rows summing to 1")
# ---------------------------------------------------------------------------------------------------------------
def test_P4_softmax_rows_sum_to_one_and_special_cases():
    n_kv, d = 2, 64
    kp, vp = _rand_pool(12, n_kv, d, 11)
    rng = np.random.default_rng(12)
    bt_row = rng.permutation(12).astype(np.int32)
    for p in (0, 1, 15, 16, 17, 130):
        qv = rng.standard_normal(d) * 4
        w64 = F64.attention_weights(qv, kp, bt_row, p, 1)
        assert abs(w64.sum() - 1.0) < 1e-12 and (w64 >= 0).all()
        w32 = F32.attention_weights(qv.astype(np.float32), kp, bt_row, p, 1)
        assert abs(w32.astype(np.float64).sum() - 1.0) < 1e-6
    # all keys equal -> uniform weights -> output = mean of V
    kp2 = kp.copy()
    kp2[:, :, :, :] = kp[0, 0, 0, :]
    L = 37
    q = rng.standard_normal((1, 4, d))
    o = F64.attention(q, kp2, vp, [0, 1], [L - 1], bt_row[None, :])
    V = f32_of_bits(hp.logical_kv(vp, bt_row, L)).astype(np.float64)
    assert np.allclose(o[0, 0], V[:, 0].mean(0), rtol=1e-12) and np.allclose(o[0, 3], V[:, 1].mean(0), rtol=1e-12)
    # ctx = 0 -> o = the (bf16) v of the only key, exactly
    o0 = F32.attention(q.astype(np.float32), kp, vp, [0, 1], [0], bt_row[None, :])
    assert np.array_equal(o0[0, 1], f32_of_bits(vp[bt_row[0], 0, 0]))
    assert np.array_equal(o0[0, 2], f32_of_bits(vp[bt_row[0], 1, 0]))


# ---------------------------------------------------------------------------------------------------------------
# P5: brute-force dense attention + torch SDPA (north_star: "checked against brute-force dense attention")
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_q,n_kv,d", [(4, 2, 64), (8, 1, 128), (4, 4, 64)])
def test_P5_attention_vs_dense_bruteforce_and_sdpa(n_q, n_kv, d):
    rng = np.random.default_rng(n_q * 100 + d)
    ctx_before = np.array([0, 5, 31, 16], dtype=np.int32)
    q_len = np.array([20, 1, 3, 33], dtype=np.int32)
    cu = np.concatenate([[0], np.cumsum(q_len)]).astype(np.int32)
    pb = synth.paged_batch(rng, ctx_before + q_len, pool_factor=1.5)
    kp, vp = _rand_pool(pb.n_pages_pool, n_kv, d, 21)
    q = rng.standard_normal((cu[-1], n_q, d)) * 2.0
    got = F64.attention(q, kp, vp, cu, ctx_before, pb.block_tables)
    want = _dense_attention(q, kp, vp, cu, ctx_before, pb.block_tables, n_q, n_kv, d)
    assert np.allclose(got, want, rtol=1e-11, atol=1e-12)
    got32 = F32.attention(q.astype(np.float32), kp, vp, cu, ctx_before, pb.block_tables)
    assert np.allclose(got32, want, rtol=0, atol=2e-5)
    # torch SDPA on one sequence with prior context, GQA by repeating kv heads
    s = 3
    Ltot = int(ctx_before[s] + q_len[s])
    K = torch.from_numpy(f32_of_bits(hp.logical_kv(kp, pb.block_tables[s], Ltot)).astype(np.float64))
    V = torch.from_numpy(f32_of_bits(hp.logical_kv(vp, pb.block_tables[s], Ltot)).astype(np.float64))
    G = n_q // n_kv
    K = K.repeat_interleave(G, 1).permute(1, 0, 2)[None]
    V = V.repeat_interleave(G, 1).permute(1, 0, 2)[None]
    Q = torch.from_numpy(q[cu[s]:cu[s + 1]]).permute(1, 0, 2)[None]
    mask = (torch.arange(Ltot)[None, :] <= (ctx_before[s] + torch.arange(int(q_len[s])))[:, None])
    ref = torch.nn.functional.scaled_dot_product_attention(Q, K, V, attn_mask=mask)[0].permute(1, 0, 2).numpy()
    assert np.allclose(got[cu[s]:cu[s + 1]], ref, rtol=1e-10, atol=1e-12)


# ---------------------------------------------------------------------------------------------------------------
# P10: GQA reductions: MHA (n_kv = n_q), MQA (n_kv = 1), replicated-kv-heads equivalence (reading A16)
# ---------------------------------------------------------------------------------------------------------------
def test_P10_gqa_equals_mha_with_replicated_kv_heads():
    rng = np.random.default_rng(5)
    n_q, n_kv, d = 8, 2, 64
    G = n_q // n_kv
    lens = np.array([40, 9], dtype=np.int32)
    cu = np.array([0, 1, 2], dtype=np.int32)
    pb = synth.paged_batch(rng, lens + 1)
    kp, vp = _rand_pool(pb.n_pages_pool, n_kv, d, 31)
    q = rng.standard_normal((2, n_q, d)).astype(np.float32)
    a = F32.attention(q, kp, vp, cu, lens, pb.block_tables)
    kp_r = np.ascontiguousarray(np.repeat(kp, G, axis=1))
    vp_r = np.ascontiguousarray(np.repeat(vp, G, axis=1))
    b = F32.attention(q, kp_r, vp_r, cu, lens, pb.block_tables)
    assert np.array_equal(a, b)
    # MQA: all q heads read kv head 0
    kp1, vp1 = np.ascontiguousarray(kp[:, :1]), np.ascontiguousarray(vp[:, :1])
    c = F32.attention(q, kp1, vp1, cu, lens, pb.block_tables)
    assert np.array_equal(c[:, :G], a[:, :G]) and not np.array_equal(c[:, G:], a[:, G:])


# ---------------------------------------------------------------------------------------------------------------
# P11: SwiGLU closed forms (step S9)
# ---------------------------------------------------------------------------------------------------------------
def test_P11_swiglu_closed_forms():
    one = np.ones(5)
    assert np.array_equal(F64.swiglu(np.zeros(5), one * 3), np.zeros(5))
    assert np.allclose(F64.swiglu(one * 40.0, one), one * 40.0, rtol=1e-15)
    assert np.allclose(F64.swiglu(one * -40.0, one), 0.0, atol=1e-15)
    x = np.linspace(-9, 9, 101)
    assert np.allclose(F64.swiglu(x, np.ones_like(x)) - F64.swiglu(-x, np.ones_like(x)), x, rtol=1e-13,
                       atol=1e-13)
    u = np.linspace(-2, 2, 101)
    want = (torch.nn.functional.silu(torch.from_numpy(x)) * torch.from_numpy(u)).numpy()
    assert np.allclose(F64.swiglu(x, u), want, rtol=1e-13, atol=1e-15)


# ---------------------------------------------------------------------------------------------------------------
# whole-stage fixtures
# ---------------------------------------------------------------------------------------------------------------
def _tiny_problem(shape, seed=0, proj_std=0.02, lens=None):
    rng = np.random.default_rng(seed)
    lens = synth.cfg1_contexts(seed) if lens is None else np.asarray(lens)
    pb = synth.paged_batch(rng, lens, extra_tokens=4, pool_factor=2.0)
    _, wb = hp.weights_bits(shape, seed, proj_std)
    x = synth.bits(synth.hidden_rows(int(lens.sum()) + 64, shape.hidden, seed))
    return lens.astype(np.int32), pb, wb, x


# ---------------------------------------------------------------------------------------------------------------
# P6: page-permutation invariance, bitwise (step S5/S6; block-table indexing)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape", [synth.TINY, synth.TINY_QWEN])
def test_P6_page_permutation_invariance_bitwise(shape):
    lens, pb, wb, x = _tiny_problem(shape)
    T = int(lens.sum())
    pool_a = hp.new_pool(shape, pb.n_pages_pool)
    ya, _, _ = hp.run_oracle_prefill(F32, shape, wb, pool_a, lens, pb.block_tables, x[:T])
    perm = np.random.default_rng(99).permutation(pb.n_pages_pool).astype(np.int32)
    bt_b = perm[pb.block_tables]
    pool_b = hp.new_pool(shape, pb.n_pages_pool)
    yb, _, _ = hp.run_oracle_prefill(F32, shape, wb, pool_b, lens, bt_b, x[:T])
    assert np.array_equal(ya, yb)
    for s in range(len(lens)):
        for l in range(shape.n_layers):
            for kv in (0, 1):
                assert np.array_equal(hp.logical_kv(pool_a[l, kv], pb.block_tables[s], lens[s]),
                                      hp.logical_kv(pool_b[l, kv], bt_b[s], lens[s]))
    # P16: bytes outside the written slots are untouched
    written = np.zeros(pool_a.shape[2:5:2], dtype=bool)   # [pages,16]
    for s in range(len(lens)):
        for p in range(lens[s]):
            written[pb.block_tables[s, p >> 4], p & 15] = True
    untouched = pool_a[:, :, ~written.any(axis=1)]
    assert (untouched == 0x7FC1).all()
    m = np.broadcast_to(written[None, None, :, None, :, None], pool_a.shape)
    assert (pool_a[~m] == 0x7FC1).all() and (pool_a[m] != 0x7FC1).all()


# ---------------------------------------------------------------------------------------------------------------
# P7: the migration invariant, bitwise in the oracle (recomputation from input + already-
# generated tokens reconstructs the KV cache) — prefill(L) == prefill(P) + (L-P) decode steps
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,rounding", [(synth.TINY, 0), (synth.TINY_QWEN, 1)])
def test_P7_migration_invariant_bitwise(shape, rounding):
    lens, pb, wb, x = _tiny_problem(shape)
    T = int(lens.sum())
    gen = 3                                            # tokens "already generated" before the interruption
    # (a) recompute: one prefill over prompt+generated
    pool_a = hp.new_pool(shape, pb.n_pages_pool)
    ya, _, cu = hp.run_oracle_prefill(F32, shape, wb, pool_a, lens, pb.block_tables, x[:T], rounding=rounding)
    # (b) incremental: prefill the prompt, then decode the generated tokens one at a time
    pool_b = hp.new_pool(shape, pb.n_pages_pool)
    prompt = lens - gen
    rows = np.concatenate([np.arange(cu[s], cu[s] + prompt[s]) for s in range(len(lens))])
    yb, _, cub = hp.run_oracle_prefill(F32, shape, wb, pool_b, prompt, pb.block_tables, x[rows],
                                       rounding=rounding)
    last = None
    for g in range(gen):
        rows = np.array([cu[s] + prompt[s] + g for s in range(len(lens))])
        last, _ = hp.run_oracle_decode(F32, shape, wb, pool_b, prompt + g, pb.block_tables, x[rows],
                                       rounding=rounding)
    assert np.array_equal(pool_a, pool_b)
    assert np.array_equal(last, ya[cu[1:] - 1])
    # the prompt rows agree too (causality)
    for s in range(len(lens)):
        assert np.array_equal(ya[cu[s]:cu[s] + prompt[s]], yb[cub[s]:cub[s + 1]])


# ---------------------------------------------------------------------------------------------------------------
# P8: chunked-prefill invariance, P9: batch-composition invariance (bitwise)
# ---------------------------------------------------------------------------------------------------------------
def test_P8_chunked_prefill_invariance_bitwise():
    shape = synth.TINY
    lens, pb, wb, x = _tiny_problem(shape, lens=[77])
    pool_a = hp.new_pool(shape, pb.n_pages_pool)
    ya, _, _ = hp.run_oracle_prefill(F32, shape, wb, pool_a, lens, pb.block_tables, x[:77])
    pool_b = hp.new_pool(shape, pb.n_pages_pool)
    done, outs = 0, []
    for c in (1, 7, 16, 40, 13):
        y, _, _ = hp.run_oracle_prefill(F32, shape, wb, pool_b, [done + c], pb.block_tables, x[done:done + c],
                                        ctx_before=[done])
        outs.append(y)
        done += c
    assert done == 77
    assert np.array_equal(np.concatenate(outs), ya) and np.array_equal(pool_a, pool_b)


def test_P9_batch_composition_invariance_bitwise():
    shape = synth.TINY
    lens, pb, wb, x = _tiny_problem(shape)
    T = int(lens.sum())
    pool_a = hp.new_pool(shape, pb.n_pages_pool)
    ya, _, cu = hp.run_oracle_prefill(F32, shape, wb, pool_a, lens, pb.block_tables, x[:T])
    order = [2, 0]                                      # drop sequences 1 and 3, permute the rest
    rows = np.concatenate([np.arange(cu[s], cu[s + 1]) for s in order])
    pool_b = hp.new_pool(shape, pb.n_pages_pool)
    yb, _, cub = hp.run_oracle_prefill(F32, shape, wb, pool_b, lens[order], pb.block_tables[order], x[rows])
    for i, s in enumerate(order):
        assert np.array_equal(yb[cub[i]:cub[i + 1]], ya[cu[s]:cu[s + 1]])


# ---------------------------------------------------------------------------------------------------------------
# P12: whole-layer second opinion — `transformers` Llama / Qwen3 decoder layers with the same tensors
# (conventions: RoPE pairing A10, QK-norm order A11, GQA head mapping A16, no biases A7)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape", [synth.TINY, synth.TINY_QWEN])
def test_P12_layer_vs_transformers(shape):
    tf = pytest.importorskip("transformers")
    if shape.qk_norm:
        from transformers.models.qwen3.modeling_qwen3 import (Qwen3Config as Cfg, Qwen3DecoderLayer as Layer,
                                                              Qwen3RotaryEmbedding as Rot)
    else:
        from transformers.models.llama.modeling_llama import (LlamaConfig as Cfg, LlamaDecoderLayer as Layer,
                                                              LlamaRotaryEmbedding as Rot)
    cfg = Cfg(hidden_size=shape.hidden, intermediate_size=shape.ffn, num_attention_heads=shape.n_q,
              num_key_value_heads=shape.n_kv, head_dim=shape.d, rms_norm_eps=shape.eps, rope_theta=shape.theta,
              num_hidden_layers=2, vocab_size=shape.vocab, attention_bias=False, max_position_embeddings=8192)
    cfg._attn_implementation = "eager"
    tw, wb = hp.weights_bits(shape, seed=5, proj_std=0.08)      # "sharp" variant: peaked softmax (A21)
    L = 45
    x_bits = synth.bits(synth.hidden_rows(L, shape.hidden, 5))
    x = torch.from_numpy(f32_of_bits(x_bits).astype(np.float64))[None]
    pos = torch.arange(L)[None]
    rot = Rot(cfg)
    cos, sin = rot(x, pos)
    mask = torch.full((L, L), float("-inf"), dtype=torch.float64).triu(1)[None, None]
    names = {"self_attn.q_proj.weight": "wq", "self_attn.k_proj.weight": "wk", "self_attn.v_proj.weight": "wv",
             "self_attn.o_proj.weight": "wo", "mlp.gate_proj.weight": "w_gate", "mlp.up_proj.weight": "w_up",
             "mlp.down_proj.weight": "w_down", "input_layernorm.weight": "ln1",
             "post_attention_layernorm.weight": "ln2", "self_attn.q_norm.weight": "q_norm",
             "self_attn.k_norm.weight": "k_norm"}
    h = x
    for li in range(2):
        layer = Layer(cfg, li).double()
        with torch.no_grad():
            for n, p in layer.named_parameters():
                p.copy_(tw[li][names[n]].to(torch.float64))
            h = layer(h, attention_mask=mask, position_ids=pos, position_embeddings=(cos.double(), sin.double()))
            h = h[0] if isinstance(h, tuple) else h
    want = h[0].numpy()
    pb = synth.paged_batch(np.random.default_rng(5), [L], pool_factor=2.0)
    pool = hp.new_pool(shape, pb.n_pages_pool)
    got, _, _ = hp.run_oracle_prefill(F64, shape, wb, pool, [L], pb.block_tables, x_bits)
    # the only intended difference: the oracle stores K/V as bf16 (contract), transformers keeps them in fp64
    err = hp.rel_err_rows(got, want)
    print("P12 rel err", shape.name, err)
    assert err < 8e-3
    # with weights that make K/V exactly representable the difference vanishes: covered by the dense pin P5;
    # here check that conventions are right by breaking one: swapping kv-head mapping or RoPE pairing moves
    # the error to O(1)
    assert np.abs(got - want).max() < 0.05 * np.abs(want).max()


# ---------------------------------------------------------------------------------------------------------------
# P13: the fp32 build against the fp64 build on cfg-1 (oracle's own rounding error)
# ---------------------------------------------------------------------------------------------------------------
def test_P13_f32_build_vs_f64_build_on_cfg1():
    shape = synth.TINY
    lens, pb, wb, x = _tiny_problem(shape)
    T = int(lens.sum())
    p32 = hp.new_pool(shape, pb.n_pages_pool)
    p64 = hp.new_pool(shape, pb.n_pages_pool)
    y32, _, _ = hp.run_oracle_prefill(F32, shape, wb, p32, lens, pb.block_tables, x[:T])
    y64, _, _ = hp.run_oracle_prefill(F64, shape, wb, p64, lens, pb.block_tables, x[:T])
    assert hp.rel_err_rows(y32, y64) < 1e-5 * 40   # K/V bf16 rounding can flip on a boundary: allow slack
    # KV: identical except for rare rounding-boundary flips of one bf16 ulp
    diff = (p32 != p64)
    assert diff.mean() < 2e-3
    a = f32_of_bits(p32[diff]).astype(np.float64)
    b = f32_of_bits(p64[diff]).astype(np.float64)
    assert (np.abs(a - b) <= np.abs(b) * 2.0 ** -7 + 1e-5).all()   # 1 ulp, or cancellation noise near 0


# ---------------------------------------------------------------------------------------------------------------
# logits tail (step S11; Table 2 "Logits Calculation"): argmax = lowest index among maxima
# ---------------------------------------------------------------------------------------------------------------
def test_logits_argmax_lowest_index_and_margin():
    shape = synth.TINY
    ew = synth.edge_weights(shape, 0)
    d = hp.odims(shape)
    y = np.random.default_rng(3).standard_normal((6, shape.hidden)).astype(np.float32)
    lm = synth.bits(ew["lm_head"]).copy()
    lm[7] = lm[3]                                        # duplicate row -> exact tie between ids 3 and 7
    logits, am, margin = F32.logits(d, y, synth.bits(ew["final_norm"]), lm)
    z = F32.rmsnorm(y, synth.bits(ew["final_norm"]), shape.eps)
    want = z.astype(np.float64) @ f32_of_bits(lm).astype(np.float64).T
    assert np.allclose(logits, want, atol=1e-4)
    assert np.array_equal(logits[:, 3], logits[:, 7])
    assert np.array_equal(am, np.argmax(logits, axis=1))   # numpy argmax returns the first maximum
    lm2 = lm.copy()
    lm2[3] = synth.bits((ew["lm_head"][am[0]].float() * 50).to(torch.bfloat16))
    lm2[7] = lm2[3]
    _, am2, mg2 = F32.logits(d, y[:1], synth.bits(ew["final_norm"]), lm2)
    assert am2[0] == 3 and mg2[0] == 0.0
    s = np.sort(logits, axis=1)
    assert np.allclose(margin, s[:, -1] - s[:, -2], atol=1e-6)


# ---------------------------------------------------------------------------------------------------------------
# embedding gather (S0)
# ---------------------------------------------------------------------------------------------------------------
def test_embed_gather():
    emb = synth.bits(synth.randn_bf16((50, 32), 1.0, torch.Generator().manual_seed(1)))
    ids = np.array([3, 49, 0, 3], dtype=np.int32)
    assert np.array_equal(F32.embed(emb, ids, 32), f32_of_bits(emb)[ids])
