"""Parity of the CUDA path (through the C-ABI) with the CPU oracle on the same seeded inputs.  All -m gpu.

Tolerances (north_star): stage-output hidden max relative error 2e-2 (reading A15: per row ||g-r||inf / ||r||inf),
per layer 1e-2, bit-exact KV indexing / page bytes outside written slots / argmax kernel; KV values vs the R1
oracle per reading A13(iii).
"""
import numpy as np
import pytest
import torch

from oracle import Oracle
from paper_2606_18600_b200 import synth
from tests import helpers as hp

pytestmark = pytest.mark.gpu

F32 = Oracle("f32")
STAGE_TOL = 2e-2
LAYER_TOL = 1e-2
ESCAPE_FRAC = 5e-3   # at most this fraction of first-layer K/V values may rely on the absolute bound (A13 ii)


def _gh():
    from tests import gpu_helpers
    return gpu_helpers


def f32b(b):
    return synth.bf16_bits_to_f32(np.asarray(b))


# ---------------------------------------------------------------------------------------------------------------
# op level: the tcgen05 GEMM against the oracle's projection (Table 2 GEMM rows)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T,N,K", [
    (64, 256, 256), (4, 512, 256), (7, 688, 256), (5, 256, 688), (64, 1024, 2048), (130, 384, 512), (300, 200, 1000),
    (16, 128, 64), (1, 8, 64), (33, 3000, 4096), (64, 128, 28672), (128, 640, 5120), (1000, 2048, 512),
    (2500, 40000, 128), (257, 130, 200),
    # every token-tile width: 96, 160, 192, 224 columns, and two ragged tiles of 160 / 224
    (65, 700, 1024), (96, 512, 8192), (129, 1300, 2048), (160, 256, 4096), (190, 4000, 512), (224, 640, 1024),
    (300, 900, 1536), (420, 520, 768),
    # the CTA-pair kernel (cta_group::2, 256 x 256 pair tiles): odd row-tile count, ragged T / N, long K
    (1100, 9000, 1024), (2049, 4224, 2048), (513, 38000, 512), (3000, 8192, 4096),
])
def test_op_gemm_vs_oracle(T, N, K):
    """Covers both schedules: stream-K with in-kernel fix-up (few tiles; one tile cut across up to 148 CTAs at
    K = 28672) and band-rasterised whole tiles (>= 4 x #SM tiles), ragged T / N / K tails."""
    from paper_2606_18600_b200 import binding
    g = torch.Generator().manual_seed(T * 7 + N + K)
    x = synth.randn_bf16((T, K), 1.0, g)
    w = synth.randn_bf16((N, K), 0.05, g)
    want = F32.matmul(f32b(synth.bits(x)), synth.bits(w))
    got = binding.op_gemm_bf16(x.cuda(), w.cuda())
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    scale = np.abs(want).max()
    assert np.abs(got - want).max() <= 2e-5 * scale * np.sqrt(K / 64) + 1e-6


@pytest.mark.gpu
@pytest.mark.parametrize("dual,T,N,K", [(True, 64, 19072, 8192), (False, 64, 8192, 8192), (True, 128, 18944, 5120),
                                        (False, 128, 5120, 8192),
                                        # the CTA-pair kernel at prefill sizes: every SM pair busy, long K
                                        (False, 2100, 8192, 8192), (True, 1500, 6144, 5120)])
def test_op_gemm_full_grid_long_k_is_stable(dual, T, N, K):
    """Regression for a pipeline race: with two MMA issuers and an odd ring size a ring slot used to change hands
    between the issuers, and the single mbarrier phase bit then let a fast issuer consume a tile still in flight
    (intermittent launch failure / garbage at decode shapes: every SM busy, >100 k-blocks per CTA, each tile cut
    across several CTAs).  20 launches must agree bit for bit with each other and match a sampled oracle check."""
    from paper_2606_18600_b200 import binding
    g = torch.Generator().manual_seed(11 + T + N)
    x = synth.randn_bf16((T, K), 1.0, g)
    w0 = synth.randn_bf16((N, K), 0.05, g)
    w1 = synth.randn_bf16((N, K), 0.05, g) if dual else None
    xd, w0d = x.cuda(), w0.cuda()
    w1d = w1.cuda() if dual else None
    torch.cuda.synchronize()
    first = None
    for _ in range(20):
        got = binding.op_gemm_swiglu_bf16(xd, w0d, w1d) if dual else binding.op_gemm_bf16(xd, w0d)
        torch.cuda.synchronize()
        if first is None:
            first = got.clone()
        else:
            assert torch.equal(got, first)
    cols = np.unique(np.concatenate([np.arange(0, N, 997), [N - 1, 127, 128]]))
    xs = f32b(synth.bits(x))
    gw = F32.matmul(xs, synth.bits(w0[cols]))
    if dual:
        want = F32.swiglu(gw, F32.matmul(xs, synth.bits(w1[cols])))
        gotc = first[:, cols].float().cpu().numpy()
        assert np.abs(gotc - want).max() <= 1e-2 * np.abs(want).max()
    else:
        gotc = first[:, cols].cpu().numpy()
        assert np.abs(gotc - gw).max() <= 2e-5 * np.abs(gw).max() * np.sqrt(K / 64) + 1e-6


@pytest.mark.parametrize("T,F,K", [(64, 256, 256), (4, 688, 256), (130, 1376, 512), (300, 200, 1000), (16, 128, 64),
                                   (64, 384, 8192), (128, 3000, 1024), (700, 20000, 128), (96, 1000, 2048),
                                   (150, 640, 4096), (192, 384, 1024), (200, 2000, 512), (310, 300, 1024),
                                   (1300, 12000, 768), (2100, 9100, 2048)])   # CTA-pair kernel
def test_op_gemm_swiglu_vs_oracle(T, F, K):
    from paper_2606_18600_b200 import binding
    g = torch.Generator().manual_seed(T + F + K)
    x = synth.randn_bf16((T, K), 1.0, g)
    wg = synth.randn_bf16((F, K), 0.08, g)
    wu = synth.randn_bf16((F, K), 0.08, g)
    xf = f32b(synth.bits(x))
    want = F32.swiglu(F32.matmul(xf, synth.bits(wg)), F32.matmul(xf, synth.bits(wu)))
    got = binding.op_gemm_swiglu_bf16(x.cuda(), wg.cuda(), wu.cuda())
    torch.cuda.synchronize()
    got = f32b(got.cpu().view(torch.int16).numpy().view(np.uint16))
    # output is bf16: half an ulp (2^-9 relative) plus accumulation noise
    assert np.abs(got - want).max() <= 2.0 ** -8 * np.abs(want).max() + 1e-6
    assert np.abs(got - want).mean() <= 2.0 ** -9 * np.abs(want).mean() + 1e-7


# ---------------------------------------------------------------------------------------------------------------
# whole stage on the tiny configs (cfg-1 of BASELINE.json and variants)
# ---------------------------------------------------------------------------------------------------------------
def _problem(shape, seed=0, proj_std=0.02, lens=None, with_edge=False, extra=4):
    gh = _gh()
    rng = np.random.default_rng(seed)
    lens = synth.cfg1_contexts(seed) if lens is None else np.asarray(lens)
    pb = synth.paged_batch(rng, lens, extra_tokens=extra, pool_factor=2.0)
    P = gh.Problem(shape, seed, proj_std, n_pages=pb.n_pages_pool, max_tokens=int(lens.sum()) + 64,
                   max_seqs=max(16, len(lens)), max_blocks=pb.max_blocks, with_edge=with_edge)
    x = synth.bits(synth.hidden_rows(int(lens.sum()) + 64, shape.hidden, seed))
    return P, lens.astype(np.int32), pb, x


def _written_mask(pool_shape, bt, lens):
    written = np.zeros((pool_shape[2], 16), dtype=bool)
    for s in range(len(lens)):
        for p in range(lens[s]):
            written[bt[s, p >> 4], p & 15] = True
    return np.broadcast_to(written[None, None, :, None, :, None], pool_shape)


def _check_kv(pool_gpu, pool_r1, mask, first_layer_only_ulp=True):
    # A13(i): indexing strict — bytes outside the written slots are untouched, written slots are all written
    assert (pool_gpu[~mask] == 0x7FC1).all(), "a byte outside the written KV slots changed"
    assert (pool_gpu[mask] != 0x7FC1).all(), "a KV slot that must be written still holds the sentinel"
    # A13(iii): values vs the R1 oracle: first layer equal or adjacent bf16 values; deeper layers close
    gh = _gh()
    ulp = gh.bf16_ulp_distance(pool_gpu[0][mask[0]], pool_r1[0][mask[0]])
    a, b = f32b(pool_gpu[0][mask[0]]), f32b(pool_r1[0][mask[0]])
    # near zero (cancellation in RoPE / projections) an absolute bound replaces the ulp bound; the elements that pass
    # ONLY through it are counted, printed and bounded (so "<= 1 ulp" is what is asserted for all but that fraction)
    esc = (ulp > 1) & (np.abs(a - b) <= 2e-3 * np.abs(b).max())
    ok = (ulp <= 1) | esc
    print(f"first-layer K/V: equal {float((ulp == 0).mean()):.4f}, <= 1 ulp {float((ulp <= 1).mean()):.4f}, "
          f"only via the absolute bound {float(esc.mean()):.5f} ({int(esc.sum())} of {ulp.size})")
    assert ok.all(), f"first-layer KV differs by more than 1 bf16 ulp in {np.count_nonzero(~ok)} elements"
    assert (ulp == 0).mean() > 0.97 and esc.mean() <= ESCAPE_FRAC
    for l in range(1, pool_gpu.shape[0]):
        a, b = f32b(pool_gpu[l][mask[l]]).astype(np.float64), f32b(pool_r1[l][mask[l]]).astype(np.float64)
        assert np.abs(a - b).max() <= 1e-2 * np.abs(b).max()


# groups of 12 and 16 query heads per kv head: rows 8-15 of the decode kernel's MMA tile are live (its HI variant)
G12 = synth.ModelShape("tiny-g12", 256, 12, 1, 64, 688, 2, 1e-5, 5e5, 0, 512)
G16 = synth.ModelShape("tiny-g16-d128", 512, 16, 1, 128, 1024, 2, 1e-6, 1e6, 1, 512)


@pytest.mark.parametrize("shape,proj_std,ref", [(synth.TINY, 0.02, 0), (synth.TINY, 0.08, 0), (synth.TINY, 0.16, 1),
                                                (synth.TINY_QWEN, 0.02, 0), (synth.TINY128, 0.05, 0),
                                                (G12, 0.04, 0), (G16, 0.04, 0)])
def test_stage_prefill_then_decode_vs_oracle(shape, proj_std, ref):
    """ref = 0: judged against the plain fp32 oracle (R0).  ref = 1: the 'sharp' variant of reading A21 (weights x8,
    peaked softmax), reading A15c: there the oracle's own R1-vs-R0 distance (printed and asserted below as
    `floor`) is several times 2e-2 — any engine that materialises bf16 activations is that far from R0 — so the 2e-2
    bound is held against R1, and against R0 the GPU must stay within 1.3 x that floor (the same rule as the
    full-depth test, reading A15d)."""
    P, lens, pb, x = _problem(shape, proj_std=proj_std)
    try:
        T = int(lens.sum())
        bt = pb.block_tables
        # ---- prefill (migration recompute path)
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        want, _, cu = hp.run_oracle_prefill(F32, shape, P.wb, pool0, lens, bt, x[:T])
        pool1 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        want1, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool1, lens, bt, x[:T], rounding=1)
        got = P.prefill(lens, bt, x[:T])
        err, err1, floor = hp.rel_err_rows(got, want), hp.rel_err_rows(got, want1), hp.rel_err_rows(want1, want)
        print(f"{shape.name} std={proj_std} prefill stage rel err vs R0 {err:.3e}, vs R1 {err1:.3e}; oracle floor "
              f"(R1 vs R0) {floor:.3e}")
        if ref == 1:
            assert floor > STAGE_TOL, "the sharp case no longer needs reading A15c: judge it against R0"
            assert err1 < STAGE_TOL and err <= 1.3 * floor
        else:
            assert err < STAGE_TOL
        mask = _written_mask(pool0.shape, bt, lens)
        _check_kv(P.pool_bits(), pool1, mask)
        # ---- two decode steps on top (both sides continue from their own pools)
        for step in range(2):
            xs = x[T + step * len(lens): T + (step + 1) * len(lens)]
            want_d, _ = hp.run_oracle_decode(F32, shape, P.wb, pool0, lens + step, bt, xs)
            want_d1, _ = hp.run_oracle_decode(F32, shape, P.wb, pool1, lens + step, bt, xs, rounding=1)
            got_d = P.decode(lens + step, bt, xs)
            err, err1, floor = (hp.rel_err_rows(got_d, want_d), hp.rel_err_rows(got_d, want_d1),
                                hp.rel_err_rows(want_d1, want_d))
            print(f"{shape.name} decode step {step} stage rel err vs R0 {err:.3e}, vs R1 {err1:.3e}; floor {floor:.3e}")
            if ref == 1:
                assert err1 < STAGE_TOL and err <= max(STAGE_TOL, 1.3 * floor)
            else:
                assert err < STAGE_TOL
        mask = _written_mask(pool0.shape, bt, lens + 2)
        _check_kv(P.pool_bits(), pool1, mask)
    finally:
        P.close()


@pytest.mark.parametrize("shape", [synth.TINY, synth.TINY_QWEN, synth.TINY128])
@pytest.mark.parametrize("phase", ["decode", "prefill"])
def test_per_layer_teacher_forced_vs_oracle(shape, phase):
    """Reading A15 'per layer', 1e-2 against the plain fp32 oracle R0: a 1-layer GPU stage holding layer l's weights is
    run from the oracle's layer-l input (rounded to bf16, the stage-boundary dtype) over the oracle's KV pool of that
    layer, for every layer, at decode (one new token per sequence on top of a prefilled context) and at prefill (the
    whole prompt; causal attention + S5 append in qkv_post); Llama-style, Qwen3-style (QK-norm) and d = 128 shapes.
    The full-width layers of both models are checked the same way in tests/test_gpu_full_depth.py."""
    gh = _gh()
    rng = np.random.default_rng(3)
    lens = synth.cfg1_contexts(3).astype(np.int32)
    pb = synth.paged_batch(rng, lens, extra_tokens=2, pool_factor=1.5)
    _, wb_all = hp.weights_bits(shape, 3)
    T = int(lens.sum())
    x = synth.bits(synth.hidden_rows(T + 8, shape.hidden, 3))
    pool = hp.new_pool(shape, pb.n_pages_pool)
    pool_empty = pool.copy()
    _, ptaps, cu = hp.run_oracle_prefill(F32, shape, wb_all, pool, lens, pb.block_tables, x[:T], taps=True)
    xs = x[T:T + len(lens)]
    pool_prefilled = pool.copy()
    _, dtaps = hp.run_oracle_decode(F32, shape, wb_all, pool, lens, pb.block_tables, xs, taps=True)
    dec = phase == "decode"
    taps, x0, pool_before = (dtaps, xs, pool_prefilled) if dec else (ptaps, x[:T], pool_empty)
    ctx = lens if dec else np.zeros_like(lens)
    cu_q = np.arange(len(lens) + 1, dtype=np.int32) if dec else cu
    sub = synth.ModelShape(shape.name, shape.hidden, shape.n_q, shape.n_kv, shape.d, shape.ffn, 1, shape.eps,
                           shape.theta, shape.qk_norm, shape.vocab)
    for l in range(shape.n_layers):
        # oracle input of layer l, rounded to bf16 (the stage boundary dtype), and the oracle's own answer from it
        x_in = f32b(x0) if l == 0 else taps[l - 1]["out"]
        x_in_bits = synth.bits(torch.from_numpy(np.ascontiguousarray(x_in, dtype=np.float32)).to(torch.bfloat16))
        pool_l = pool_before[l:l + 1].copy()
        want = f32b(x_in_bits).copy()
        F32.layer(hp.odims(shape), wb_all[l], pool_l[0, 0], pool_l[0, 1], cu_q, ctx, pb.block_tables, want)
        # GPU: 1-layer stage holding layer l's weights and the oracle's KV for that layer
        P = gh.Problem(sub, 3, n_pages=pb.n_pages_pool, max_tokens=T + 64, max_seqs=16, max_blocks=pb.max_blocks)
        try:
            tw = synth.layer_weights(shape, l, 3)
            for k, v in tw.items():
                if v is not None:
                    P.dw[0][k].copy_(v.to("cuda:0"))
            P.stage.pool_view().copy_(torch.from_numpy(pool_before[l:l + 1].view(np.int16).copy())
                                      .view(torch.bfloat16).to("cuda:0"))
            got = P.decode(lens, pb.block_tables, x_in_bits) if dec else P.prefill(lens, pb.block_tables, x_in_bits)
        finally:
            P.close()
        err = hp.rel_err_rows(got, want)
        print(f"{shape.name} layer {l} teacher-forced {phase} rel err vs R0 {err:.3e}")
        assert err < LAYER_TOL


def test_ss_debug_device_contract_checks(monkeypatch):
    """SS_DEBUG=1 (include/shuntstage.h, ss_stage_debug_info): a page id outside the pool, a
    context beyond the listed pages, a position beyond max_pos, a token id outside the vocabulary and a malformed cu_q
    are caught on the device BEFORE anything is enqueued — the call returns SS_ERR_INVALID_ARG, the violation is
    reported, the pool keeps every sentinel byte — and a valid call still matches the oracle."""
    from paper_2606_18600_b200 import binding
    monkeypatch.setenv("SS_DEBUG", "1")
    shape = synth.TINY
    P, lens, pb, x = _problem(shape, seed=5, with_edge=True)
    try:
        on, info = P.stage.debug_info()
        assert on and info == [0, 0, 0, 0]
        bt = pb.block_tables
        T, n = int(lens.sum()), len(lens)
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        n_pages = P.stage.num_pages()
        out = torch.empty((T, shape.hidden), dtype=torch.bfloat16, device="cuda:0")
        hid = P.bf16(x[:T])

        def prefill(bt_=bt, cu_=cu, ctx_=np.zeros(n, np.int32), ids=None, T_=T):
            kw = dict(token_ids=P.i32(ids)) if ids is not None else dict(hidden=hid[:T_])
            rc = P.stage.prefill(n, P.i32(cu_), P.i32(ctx_), P.i32(bt_), T_, out_hidden=out[:T_], check=False, **kw)
            P.stage.synchronize()
            return rc, P.stage.debug_info()[1]

        bad = bt.copy(); bad[2, 1] = n_pages                       # first page id past the pool
        assert prefill(bt_=bad) == (-1, [1, 2, 1, n_pages])
        bad = bt.copy(); bad[0, 0] = -3
        assert prefill(bt_=bad) == (-1, [1, 0, 0, -3])
        far = np.zeros(n, np.int32); far[1] = bt.shape[1] * 16      # ctx + q_len beyond the listed pages
        rc, info = prefill(ctx_=far)
        assert rc == -1 and info[0] == 2 and info[1] == 1
        cu_bad = cu.copy(); cu_bad[2] = cu_bad[1]                   # an empty sequence
        rc, info = prefill(cu_=cu_bad)
        assert rc == -1 and info[0] == 5
        ids = np.arange(T, dtype=np.int32) % shape.vocab; ids[7] = shape.vocab
        assert prefill(ids=ids) == (-1, [4, -1, 7, shape.vocab])
        # decode: context that puts the new token beyond max_pos; a bad page id in ss_kv_export
        ctx_far = lens.copy(); ctx_far[3] = P.dims.max_pos
        o2 = torch.empty((n, shape.hidden), dtype=torch.bfloat16, device="cuda:0")
        rc = P.stage.decode(n, P.i32(bt), P.i32(ctx_far), hidden=hid[:n], out_hidden=o2, check=False)
        assert rc == -1 and P.stage.debug_info()[1][0] in (2, 3) and P.stage.debug_info()[1][1] == 3
        buf = torch.empty(2 * P.stage.page_bytes // 2, dtype=torch.bfloat16, device="cuda:0")
        assert P.stage.kv_export(P.i32([1, n_pages + 5]), buf, check=False) == -1
        assert P.stage.debug_info()[1] == [1, -1, 1, n_pages + 5]
        # nothing was enqueued by any rejected call: every pool byte still holds the sentinel
        assert (P.pool_bits() == 0x7FC1).all()
        # a valid call under SS_DEBUG=1 works and matches the oracle
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        want, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool0, lens, bt, x[:T])
        got = P.prefill(lens, bt, x[:T])
        assert hp.rel_err_rows(got, want) < STAGE_TOL
    finally:
        P.close()
    monkeypatch.delenv("SS_DEBUG")
    Q, _, _, _ = _problem(shape, seed=5)
    try:
        assert Q.stage.debug_info()[0] is False
    finally:
        Q.close()


def test_migration_invariant_on_gpu():
    """recompute (one prefill over prompt + generated tokens) must reproduce incremental decode:
    same next-token hidden state within tolerance, KV pages equal or adjacent bf16 values."""
    shape = synth.TINY
    gh = _gh()
    P, lens, pb, x = _problem(shape, seed=1)
    Q, _, _, _ = _problem(shape, seed=1)
    try:
        bt = pb.block_tables
        T = int(lens.sum())
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        gen = 3
        prompt = lens - gen
        # (a) recompute
        P.prefill(lens, bt, x[:T])
        # (b) incremental
        rows = np.concatenate([np.arange(cu[s], cu[s] + prompt[s]) for s in range(len(lens))])
        Q.prefill(prompt, bt, x[rows])
        for g in range(gen):
            rows = np.array([cu[s] + prompt[s] + g for s in range(len(lens))])
            Q.decode(prompt + g, bt, x[rows])
        pa, pq = P.pool_bits(), Q.pool_bits()
        mask = _written_mask(pa.shape, bt, lens)
        assert (pa[~mask] == 0x7FC1).all() and (pq[~mask] == 0x7FC1).all()
        ulp = gh.bf16_ulp_distance(pa[mask], pq[mask])
        a, b = f32b(pa[mask]), f32b(pq[mask])
        esc = (ulp > 2) & (np.abs(a - b) <= 4e-3 * np.abs(b).max())
        print(f"recompute vs incremental K/V: equal {float((ulp == 0).mean()):.4f}, <= 2 ulp "
              f"{float((ulp <= 2).mean()):.4f}, only via the absolute bound {float(esc.mean()):.5f}")
        assert ((ulp <= 2) | esc).all()
        assert (ulp == 0).mean() > 0.9 and esc.mean() <= 2 * ESCAPE_FRAC
        # next decode step from both states
        xs = x[T:T + len(lens)]
        ya = P.decode(lens, bt, xs)
        yq = Q.decode(lens, bt, xs)
        assert hp.rel_err_rows(ya, yq) < STAGE_TOL
        # and both match the oracle's (bitwise-invariant) answer
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        hp.run_oracle_prefill(F32, shape, P.wb, pool0, lens, bt, x[:T])
        want, _ = hp.run_oracle_decode(F32, shape, P.wb, pool0, lens, bt, xs)
        assert hp.rel_err_rows(ya, want) < STAGE_TOL and hp.rel_err_rows(yq, want) < STAGE_TOL
    finally:
        P.close()
        Q.close()


@pytest.mark.parametrize("shape", [synth.TINY, synth.TINY_QWEN, synth.TINY128])
def test_migration_is_bit_exact_in_batch_invariant_mode(shape):
    """ss_stage_set_batch_invariant (include/shuntstage.h; SURVEY 8(f) "later": batch-invariant summation).  The paper's
    migration is output-PRESERVING: in this mode the GPU meets that bit for bit — recompute (one
    prefill over prompt + generated tokens), a chunked recompute with another batch composition, and incremental decode
    (prefill of the prompt + decode steps) leave IDENTICAL KV pages, and the next decode step from each state returns
    identical hidden-state bits; all of it still matches the oracle within the stage tolerance."""
    P, lens, pb, x = _problem(shape, seed=1)
    Q, _, _, _ = _problem(shape, seed=1)
    R, _, _, _ = _problem(shape, seed=1)
    try:
        for S in (P, Q, R):
            S.stage.set_batch_invariant(True)
        bt = pb.block_tables
        n, T = len(lens), int(lens.sum())
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        gen = 3
        prompt = lens - gen
        # (a) recompute: one prefill over everything
        P.prefill(lens, bt, x[:T])
        # (b) incremental: prompt, then one decode step per generated token
        rows = np.concatenate([np.arange(cu[s], cu[s] + prompt[s]) for s in range(n)])
        Q.prefill(prompt, bt, x[rows])
        for g in range(gen):
            Q.decode(prompt + g, bt, x[np.array([cu[s] + prompt[s] + g for s in range(n)])])
        # (c) chunked recompute in another batch composition: sequences 0-1 first, then 2-3, each in two chunks
        for grp in (np.arange(0, n // 2), np.arange(n // 2, n)):
            half = lens[grp] // 2
            r1 = np.concatenate([np.arange(cu[s], cu[s] + lens[s] // 2) for s in grp])
            r2 = np.concatenate([np.arange(cu[s] + lens[s] // 2, cu[s + 1]) for s in grp])
            R.prefill(half, bt[grp], x[r1])
            R.prefill(lens[grp], bt[grp], x[r2], ctx_before=half)
        pa, pq, pr = P.pool_bits(), Q.pool_bits(), R.pool_bits()
        assert np.array_equal(pa, pq), f"recompute vs incremental: {int((pa != pq).sum())} KV elements differ"
        assert np.array_equal(pa, pr), f"recompute vs chunked recompute: {int((pa != pr).sum())} KV elements differ"
        mask = _written_mask(pa.shape, bt, lens)
        assert (pa[~mask] == 0x7FC1).all() and (pa[mask] != 0x7FC1).all()
        xs = x[T:T + n]
        ya, yq, yr = P.decode(lens, bt, xs), Q.decode(lens, bt, xs), R.decode(lens, bt, xs)
        assert np.array_equal(ya, yq) and np.array_equal(ya, yr)
        # a decode step of a sub-batch returns the same bits for its rows (batch composition)
        sub = np.array([2, 0])
        P2, _, _, _ = _problem(shape, seed=1)
        try:
            P2.stage.set_batch_invariant(True)
            P2.prefill(lens, bt, x[:T])
            ys = P2.decode(lens[sub], bt[sub], xs[sub])
            assert np.array_equal(ys, ya[sub])
        finally:
            P2.close()
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        hp.run_oracle_prefill(F32, shape, P.wb, pool0, lens, bt, x[:T])
        want, _ = hp.run_oracle_decode(F32, shape, P.wb, pool0, lens, bt, xs)
        err = hp.rel_err_rows(ya, want)
        print(f"{shape.name}: batch-invariant mode, next-token hidden vs oracle R0 {err:.3e}")
        assert err < STAGE_TOL
        # back in the default mode the stage still works (graphs re-captured)
        P.stage.set_batch_invariant(False)
        yd = P.decode(lens + 1, bt, xs)
        assert np.isfinite(yd).all()
    finally:
        P.close()
        Q.close()
        R.close()


# odd groups and no grouping at all: the prefill attention pairs the q heads of a GQA group per CTA, an odd group leaves
# its last head alone, MHA (G = 1) leaves every head alone
G3 = synth.ModelShape("tiny-g3", 192, 3, 1, 64, 384, 2, 1e-5, 5e5, 0, 512)
MHA = synth.ModelShape("tiny-mha-d128", 256, 2, 2, 128, 512, 2, 1e-6, 1e6, 1, 512)


@pytest.mark.parametrize("shape,lens,first", [
    (G3, [300, 1, 129, 64], [0, 0, 0, 0]),                       # odd group; 1-row tile; a tile boundary at 128 / 64
    (MHA, [257, 128, 65], [0, 0, 0]),                            # MHA, d = 128, a 1-row last tile (257 = 2 x 128 + 1)
    (synth.TINY128, [700, 33], [517, 20]),                       # chunk on top of a long prior context, unaligned start
    (synth.TINY, [2100, 2049], [2000, 0]),                       # > 2,048 keys: 33 ring stages per tile, ring wrap-around
    (synth.TINY, [9001, 40], [0, 0]),                            # one long sequence: items of 1 ... 141 stages, 71 query tiles
    (synth.TINY128, [8200, 300], [7900, 290]),                   # short chunks on top of ~8K tokens of prior context
])
def test_prefill_attention_edge_shapes_vs_oracle(shape, lens, first):
    """Edge cases of the tcgen05 prefill attention (two heads per CTA, 128-row query tiles, 64-key stages, lazy maximum,
    dead rows of the last page zeroed): whole 2-layer stage vs the oracle, KV pages strict."""
    lens, first = np.array(lens, dtype=np.int32), np.array(first, dtype=np.int32)
    P, lens, pb, x = _problem(shape, seed=9, lens=lens, extra=4)
    try:
        bt = pb.block_tables
        n = len(lens)
        cu_full = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        if first.any():   # prior context first (sequences with first == 0 take no part in that call)
            keep = first > 0
            rows1 = np.concatenate([np.arange(cu_full[s], cu_full[s] + first[s]) for s in range(n) if keep[s]])
            w1, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool0, first[keep], bt[keep], x[rows1])
            g1 = P.prefill(first[keep], bt[keep], x[rows1])
            assert hp.rel_err_rows(g1, w1) < STAGE_TOL
        rows2 = np.concatenate([np.arange(cu_full[s] + first[s], cu_full[s + 1]) for s in range(n)])
        w2, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool0, lens, bt, x[rows2], ctx_before=first)
        g2 = P.prefill(lens, bt, x[rows2], ctx_before=first)
        err = hp.rel_err_rows(g2, w2)
        print(f"{shape.name} lens {lens.tolist()} after {first.tolist()}: prefill rel err vs R0 {err:.3e}")
        assert np.isfinite(g2).all() and err < STAGE_TOL
        mask = _written_mask(pool0.shape, bt, lens)
        pg = P.pool_bits()
        assert (pg[~mask] == 0x7FC1).all() and (pg[mask] != 0x7FC1).all()
    finally:
        P.close()


@pytest.mark.gpu
@pytest.mark.parametrize("shape,n_seqs,long_len", [
    (G3, 230, 700),          # odd group, d = 64: the items of a CTA alternate between two heads and a lone head
    (MHA, 200, 600),         # MHA, d = 128: tile B is absent in every item
    (synth.TINY128, 400, 1500),   # G = 8, d = 128: 4 head pairs per tile, ~2,000 items
])
def test_prefill_attention_persistent_ctas_take_several_items_vs_oracle(shape, n_seqs, long_len):
    """The prefill attention is persistent: one CTA per SM walks the heaviest-first list of (query tile, head pair) items
    in snake order, and its barrier phases, ring slots and S / O buffers carry on from one item to the next.  The other
    attention cases have fewer items than SMs; here every CTA takes several, of very different weights (a few long
    sequences among many of 1-130 tokens, so 1-row tiles, 1-stage items and ring wrap-arounds meet in one CTA), with and
    without the second head of the pair.  Whole 2-layer stage vs the oracle, KV pages strict."""
    rng = np.random.default_rng(n_seqs)
    lens = rng.integers(1, 131, size=n_seqs).astype(np.int32)
    lens[rng.choice(n_seqs, size=5, replace=False)] = [long_len, long_len - 63, 257, 129, 128]
    P, lens, pb, x = _problem(shape, seed=13, lens=lens, extra=4)
    try:
        bt = pb.block_tables
        pairs = (shape.n_q // shape.n_kv + 1) // 2
        n_items = int(((lens + 127) // 128).sum()) * shape.n_kv * pairs
        assert n_items > 2 * 148, n_items        # several items per CTA on a 148-SM part
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        want, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool0, lens, bt, x[:int(lens.sum())])
        got = P.prefill(lens, bt, x[:int(lens.sum())])
        err = hp.rel_err_rows(got, want)
        print(f"{shape.name}: {n_seqs} sequences, {int(lens.sum())} tokens, {n_items} attention items: rel err vs R0 {err:.3e}")
        assert np.isfinite(got).all() and err < STAGE_TOL
        mask = _written_mask(pool0.shape, bt, lens)
        pg = P.pool_bits()
        assert (pg[~mask] == 0x7FC1).all() and (pg[mask] != 0x7FC1).all()
        again = P.prefill(lens, bt, x[:int(lens.sum())])   # same call again: same bits (no state left behind in the CTAs' walk)
        assert np.array_equal(again, got)
    finally:
        P.close()


@pytest.mark.parametrize("shape,lens,first", [
    (synth.TINY128, [1500, 333, 64], [0, 0, 0]),
    (synth.TINY, [700, 2100], [300, 2000]),
    (G3, [400, 129], [0, 100]),
])
def test_prefill_attention_rescale_path_vs_oracle_and_default(monkeypatch, shape, lens, first):
    """The prefill attention rescales its O accumulator in tensor memory only when a key tile exceeds a row's running
    maximum by more than 2^16 — rare on these inputs.  SS_ATTN_LAZY=0 makes every growth of the maximum take that path
    (tcgen05.ld / scale / tcgen05.st of O after waiting for the previous P.V): the result must still match the oracle, and
    the default build's result up to rounding (O / l is the same quotient)."""
    gh = _gh()
    lens, first = np.array(lens, dtype=np.int32), np.array(first, dtype=np.int32)
    P, lens, pb, x = _problem(shape, seed=17, lens=lens, extra=4)
    monkeypatch.setenv("SS_ATTN_LAZY", "0")
    Q = gh.Problem(shape, 17, n_pages=pb.n_pages_pool, max_tokens=int(lens.sum()) + 64, max_seqs=16, max_blocks=pb.max_blocks)
    monkeypatch.delenv("SS_ATTN_LAZY")
    try:
        bt, n = pb.block_tables, len(lens)
        cu_full = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        if first.any():
            keep = first > 0
            rows1 = np.concatenate([np.arange(cu_full[s], cu_full[s] + first[s]) for s in range(n) if keep[s]])
            hp.run_oracle_prefill(F32, shape, P.wb, pool0, first[keep], bt[keep], x[rows1])
            P.prefill(first[keep], bt[keep], x[rows1])
            Q.prefill(first[keep], bt[keep], x[rows1])
        rows2 = np.concatenate([np.arange(cu_full[s] + first[s], cu_full[s + 1]) for s in range(n)])
        want, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool0, lens, bt, x[rows2], ctx_before=first)
        a = P.prefill(lens, bt, x[rows2], ctx_before=first)
        b = Q.prefill(lens, bt, x[rows2], ctx_before=first)
        ea, eb, d = hp.rel_err_rows(a, want), hp.rel_err_rows(b, want), hp.rel_err_rows(b, a)
        print(f"{shape.name} lens {lens.tolist()}: default vs R0 {ea:.3e}, always-rescale vs R0 {eb:.3e}, between them {d:.3e}")
        assert np.isfinite(b).all() and ea < STAGE_TOL and eb < STAGE_TOL and d < 1e-2   # (bf16 outputs: single-step flips)
        assert not np.array_equal(a, b), "SS_ATTN_LAZY=0 changed nothing: the rescale path was not taken"
    finally:
        P.close()
        Q.close()


def test_chunked_prefill_and_mixed_batch_on_gpu():
    """Prior context (ctx_before > 0) and q_len = 1 rows in a prefill call (mixed iteration, reading A19)."""
    shape = synth.TINY_QWEN
    P, lens, pb, x = _problem(shape, seed=2, lens=[70, 33, 150, 16])
    try:
        bt = pb.block_tables
        first = np.array([40, 33 - 1, 100, 15], dtype=np.int32)      # chunk 1
        cu_full = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        rows1 = np.concatenate([np.arange(cu_full[s], cu_full[s] + first[s]) for s in range(4)])
        rows2 = np.concatenate([np.arange(cu_full[s] + first[s], cu_full[s + 1]) for s in range(4)])
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        w1, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool0, first, bt, x[rows1])
        w2, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool0, lens, bt, x[rows2], ctx_before=first)
        g1 = P.prefill(first, bt, x[rows1])
        g2 = P.prefill(lens, bt, x[rows2], ctx_before=first)    # seqs 1 and 3 have q_len = 1
        assert hp.rel_err_rows(g1, w1) < STAGE_TOL
        assert hp.rel_err_rows(g2, w2) < STAGE_TOL
        mask = _written_mask(pool0.shape, bt, lens)
        pg = P.pool_bits()
        assert (pg[~mask] == 0x7FC1).all() and (pg[mask] != 0x7FC1).all()
    finally:
        P.close()


@pytest.mark.parametrize("shape", [synth.TINY, synth.TINY_QWEN])
def test_stage_mixed_decode_rows_first_vs_oracle(shape):
    """ss_stage_mixed (continuous batching; reading A19): 3 decode rows (q_len 1, routed to the
    decode attention kernel, their K/V appended by qkv_post) followed by 2 prefill chunks, one call; then the same
    state advanced again with every row a decode row (n_decode_rows == n_seqs)."""
    from paper_2606_18600_b200 import binding
    lens = np.array([37, 16, 129, 90, 50], dtype=np.int32)           # totals after the mixed call
    P, lens, pb, x = _problem(shape, seed=4, lens=lens, extra=8)
    try:
        bt = pb.block_tables
        before = np.array([36, 15, 128, 30, 0], dtype=np.int32)       # rows 0-2 decode (q_len 1), 3-4 chunks
        cu_full = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        rows1 = np.concatenate([np.arange(cu_full[s], cu_full[s] + before[s]) for s in range(5)])
        rows2 = np.concatenate([np.arange(cu_full[s] + before[s], cu_full[s + 1]) for s in range(5)])
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        keep = before > 0
        hp.run_oracle_prefill(F32, shape, P.wb, pool0, before[keep], bt[keep], x[rows1])
        w2, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool0, lens, bt, x[rows2], ctx_before=before)
        P.prefill(before[keep], bt[keep], x[rows1])
        q = lens - before
        cu = np.concatenate([[0], np.cumsum(q)]).astype(np.int32)
        T = int(cu[-1])
        out = torch.empty((T, shape.hidden), dtype=torch.bfloat16, device="cuda:0")
        a = (P.i32(cu), P.i32(before), P.i32(bt), P.bf16(x[rows2]))
        torch.cuda.synchronize()
        P.stage.mixed(3, 5, a[0], a[1], a[2], T, hidden=a[3], out_hidden=out)
        P.stage.synchronize()
        g2 = f32b(out.cpu().view(torch.int16).numpy().view(np.uint16))
        assert hp.rel_err_rows(g2, w2) < STAGE_TOL
        mask = _written_mask(pool0.shape, bt, lens)
        pg = P.pool_bits()
        assert (pg[~mask] == 0x7FC1).all() and (pg[mask] != 0x7FC1).all()
        # every row a decode row, through ss_stage_mixed
        xs = x[int(lens.sum()):int(lens.sum()) + 5]
        w3, _ = hp.run_oracle_decode(F32, shape, P.wb, pool0, lens, bt, xs)
        out3 = torch.empty((5, shape.hidden), dtype=torch.bfloat16, device="cuda:0")
        b = (P.i32(np.arange(6)), P.i32(lens), P.bf16(xs))
        torch.cuda.synchronize()
        P.stage.mixed(5, 5, b[0], b[1], a[2], 5, hidden=b[2], out_hidden=out3)
        P.stage.synchronize()
        assert hp.rel_err_rows(f32b(out3.cpu().view(torch.int16).numpy().view(np.uint16)), w3) < STAGE_TOL
        # host-detectable misuse
        assert P.stage.mixed(6, 5, b[0], b[1], a[2], 5, hidden=b[2], out_hidden=out3, check=False) == -1
        assert P.stage.mixed(-1, 5, b[0], b[1], a[2], 5, hidden=b[2], out_hidden=out3, check=False) == -1
    finally:
        P.close()


def test_P17_dyadic_case_kv_bits_exact():
    """Reading A13, strict value pin: with projection weights +-2^-k, unit gains and small-integer hidden rows every
    fp32 partial sum of the K/V projections is exact, so the result cannot depend on the summation order (tensor
    core vs CPU loop): V at every position and K at position 0 (RoPE = identity there) must equal the oracle's
    pages BIT FOR BIT."""
    shape = synth.TINY
    gh = _gh()
    lens = np.array([1, 5, 16, 33], dtype=np.int32)
    P, lens, pb, _ = _problem(shape, seed=9, lens=lens)
    try:
        g = torch.Generator().manual_seed(123)
        for name in ("wq", "wk", "wv", "wo", "w_gate", "w_up", "w_down"):
            w = P.tw[0][name]
            sign = torch.randint(0, 2, w.shape, generator=g) * 2 - 1
            expo = torch.randint(4, 8, w.shape, generator=g)
            w.copy_((sign.float() * torch.pow(2.0, -expo.float())).to(torch.bfloat16))
        for name in ("ln1", "ln2"):
            for l in range(P.L):
                P.tw[l][name].fill_(1.0)
        for l in range(P.L):
            for k, v in P.tw[l].items():
                if v is not None:
                    P.dw[l][k].copy_(v.to("cuda:0"))
        wb = [{k: (None if v is None else synth.bits(v)) for k, v in w.items()} for w in P.tw]
        T = int(lens.sum())
        xi = torch.randint(-4, 5, (T, shape.hidden), generator=g).float()
        xi[xi == 0] = 1.0
        x = synth.bits(xi.to(torch.bfloat16))
        pool = hp.new_pool(shape, pb.n_pages_pool, P.L)
        hp.run_oracle_prefill(F32, shape, wb, pool, lens, pb.block_tables, x, rounding=1)
        P.prefill(lens, pb.block_tables, x)
        pg = P.pool_bits()
        for s, n in enumerate(lens):
            v_gpu = hp.logical_kv(pg[0, 1], pb.block_tables[s], int(n))
            v_orc = hp.logical_kv(pool[0, 1], pb.block_tables[s], int(n))
            assert np.array_equal(v_gpu, v_orc), f"V bits differ in sequence {s}"
            k_gpu = hp.logical_kv(pg[0, 0], pb.block_tables[s], 1)
            k_orc = hp.logical_kv(pool[0, 0], pb.block_tables[s], 1)
            assert np.array_equal(k_gpu, k_orc), f"K bits at position 0 differ in sequence {s}"
    finally:
        P.close()


def test_migration_by_kv_transfer_is_bit_exact():
    """instead of recomputing, move a request's KV pages to another stage
    instance (ss_kv_export -> copy -> ss_kv_import into freshly allocated pages).  The exported message equals the
    numpy gather of the pool byte for byte, the importer's logical KV equals the exporter's, and the next decode
    step on the destination is bit-identical to the same step on the source."""
    shape = synth.TINY_QWEN
    gh = _gh()
    A, lens, pb, x = _problem(shape, seed=6, lens=[70, 33, 150, 16], extra=20)
    B = gh.Problem(shape, 6, n_pages=pb.n_pages_pool + 7, max_tokens=64, max_seqs=16, max_blocks=pb.max_blocks)
    try:
        bt = pb.block_tables
        T = int(lens.sum())
        A.prefill(lens, bt, x[:T])
        need = [(int(n) + 1 + 15) // 16 for n in lens]                # pages incl. the next token's slot
        src_ids = np.concatenate([bt[s, :need[s]] for s in range(len(lens))]).astype(np.int32)
        n = len(src_ids)
        page_bytes = A.L * 2 * shape.n_kv * 16 * shape.d * 2
        buf = torch.empty(n * page_bytes // 2, dtype=torch.bfloat16, device="cuda:0")
        A.stage.kv_export(A.i32(src_ids), buf)
        A.stage.synchronize()
        msg = buf.cpu().view(torch.int16).numpy().view(np.uint16).reshape(A.L, 2, n, shape.n_kv, 16, shape.d)
        assert np.array_equal(msg, A.pool_bits()[:, :, src_ids])      # byte-exact gather
        # destination: its own allocator hands out the pages (a different physical placement)
        B.stage.kv_alloc(5)                                           # shift the ids
        dst_ids = np.array(B.stage.kv_alloc(n), dtype=np.int32)[::-1].copy()
        B.stage.kv_import(B.i32(dst_ids), buf)
        bt_b = np.zeros_like(bt)
        o = 0
        for s in range(len(lens)):
            bt_b[s, :need[s]] = dst_ids[o:o + need[s]]
            o += need[s]
        pa, pq = A.pool_bits(), B.pool_bits()
        for s, ln in enumerate(lens):
            for l in range(A.L):
                for kv in range(2):
                    assert np.array_equal(hp.logical_kv(pa[l, kv], bt[s], int(ln)), hp.logical_kv(pq[l, kv], bt_b[s], int(ln)))
        xs = x[T:T + len(lens)]
        ya = A.decode(lens, bt, xs)
        yb = B.decode(lens, bt_b, xs)
        assert np.array_equal(ya, yb)                                 # output-preserving, bit for bit
        # misuse
        assert B.stage.kv_import(B.i32(dst_ids), buf[:8], check=False) == -3      # SS_ERR_CAPACITY
        assert B.stage.kv_export(B.i32(dst_ids[:0]), buf, check=False) == -1      # n <= 0
    finally:
        A.close()
        B.close()


@pytest.mark.parametrize("invariant", [False, True])
def test_generation_then_migration_recompute_gives_the_same_tokens(invariant):
    """BASELINE.json configs[3] end to end, on the tiny model run as ONE stage with its embedding and lm_head: requests
    generate greedily (token ids in, argmax out, fed back) for k steps; the request is then 'migrated': a fresh stage
    instance recomputes prompt + generated tokens in one prefill and continues.  Output-preserving
    means the tokens after the migration equal the ones the original instance goes on to produce.  In batch-invariant
    mode that must hold for every row, bit for bit in the logits; in the default mode for every row whose top-2 logit margin
    exceeds the recompute-vs-incremental logit difference (reading A14), which is printed."""
    shape = synth.TINY_QWEN
    k_before, k_after = 6, 4
    P, lens, pb, _ = _problem(shape, seed=9, with_edge=True, extra=k_before + k_after + 2)
    Q, _, _, _ = _problem(shape, seed=9, with_edge=True, extra=k_before + k_after + 2)
    try:
        for st in (P.stage, Q.stage):
            st.set_batch_invariant(invariant)
        n, bt = len(lens), pb.block_tables
        rng = np.random.default_rng(9)
        prompt = rng.integers(0, shape.vocab, int(lens.sum())).astype(np.int32)
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        dev = "cuda:0"

        def prefill(stage, ids, cu_q):
            lg = torch.empty((n, shape.vocab), dtype=torch.float32, device=dev)
            am = torch.empty((n,), dtype=torch.int32, device=dev)
            stage.prefill(n, P.i32(cu_q), P.i32(np.zeros(n)), P.i32(bt), int(cu_q[-1]), token_ids=P.i32(ids), out_logits=lg,
                          out_argmax=am)
            stage.synchronize()
            return lg.cpu().numpy(), am.cpu().numpy()

        def decode(stage, ctx, ids):
            lg = torch.empty((n, shape.vocab), dtype=torch.float32, device=dev)
            am = torch.empty((n,), dtype=torch.int32, device=dev)
            stage.decode(n, P.i32(bt), P.i32(ctx), token_ids=P.i32(ids), out_logits=lg, out_argmax=am)
            stage.synchronize()
            return lg.cpu().numpy(), am.cpu().numpy()

        # ---- the original instance: prompt, then k_before + k_after greedy steps
        _, tok = prefill(P.stage, prompt, cu)
        gen, logit_log = [tok], []
        for step in range(k_before + k_after):
            lg, tok = decode(P.stage, lens + step, gen[-1])
            gen.append(tok)
            logit_log.append(lg)
        gen = np.stack(gen, axis=1)                                  # [n, 1 + k_before + k_after]
        # ---- migration after k_before generated tokens have been CONSUMED: recompute prompt + gen[:, :k_before] ...
        lens2 = lens + k_before
        cu2 = np.concatenate([[0], np.cumsum(lens2)]).astype(np.int32)
        ids2 = np.concatenate([np.concatenate([prompt[cu[s]:cu[s + 1]], gen[s, :k_before]]) for s in range(n)]).astype(np.int32)
        lg_m, tok_m = prefill(Q.stage, ids2, cu2)
        # ... whose last-row logits are those of incremental step k_before - 1 (input gen[:, k_before - 1])
        ref = logit_log[k_before - 1]
        diff = float(np.abs(lg_m - ref).max())
        top2 = np.sort(ref, axis=1)[:, -2:]
        safe = (top2[:, 1] - top2[:, 0]) > 4 * diff
        print(f"invariant={invariant}: recompute vs incremental logits max abs diff {diff:.3e} (scale {float(np.abs(ref).max()):.2f}); "
              f"rows over margin {int(safe.sum())}/{n}")
        if invariant:
            assert np.array_equal(lg_m, ref) and np.array_equal(tok_m, gen[:, k_before])
        else:
            assert hp.rel_err_rows(lg_m, ref) < STAGE_TOL and np.array_equal(tok_m[safe], gen[safe, k_before])
        # ---- and the migrated instance continues with the same tokens
        follow = safe if not invariant else np.ones(n, dtype=bool)
        tok = gen[:, k_before].copy()                # feed the original's token (rows off the margin may differ by a near-tie)
        for step in range(k_before, k_before + k_after):
            lg, tok_n = decode(Q.stage, lens + step, tok)
            ref = logit_log[step]
            if invariant:
                assert np.array_equal(lg, ref), step
            else:
                d = float(np.abs(lg - ref).max())
                t2 = np.sort(ref, axis=1)[:, -2:]
                follow = follow & ((t2[:, 1] - t2[:, 0]) > 4 * d)
                assert hp.rel_err_rows(lg, ref) < STAGE_TOL
            assert np.array_equal(tok_n[follow], gen[follow, step + 1]), step
            tok = gen[:, step + 1]
        assert follow.sum() >= n // 2
    finally:
        P.close()
        Q.close()


def test_token_ids_logits_and_argmax():
    """S0 embedding gather and S11 logits/argmax (Table 2 'Logits Calculation'; reading A14)."""
    shape = synth.TINY
    gh = _gh()
    P, lens, pb, _ = _problem(shape, seed=4, with_edge=True)
    try:
        bt = pb.block_tables
        T = int(lens.sum())
        rng = np.random.default_rng(4)
        ids = rng.integers(0, shape.vocab, T + len(lens)).astype(np.int32)
        eb = {k: synth.bits(v) for k, v in P.edge_cpu.items()}
        cu = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        y, _ = F32.stage(hp.odims(shape), P.wb, pool0, cu, np.zeros_like(lens), bt, token_ids=ids[:T],
                         embed=eb["embed"])
        wl, wa, wm = F32.logits(hp.odims(shape), y[cu[1:] - 1], eb["final_norm"], eb["lm_head"])
        out = torch.empty((T, shape.hidden), dtype=torch.bfloat16, device="cuda:0")
        lg = torch.empty((len(lens), shape.vocab), dtype=torch.float32, device="cuda:0")
        am = torch.empty((len(lens),), dtype=torch.int32, device="cuda:0")
        a = (P.i32(cu), P.i32(np.zeros_like(lens)), P.i32(bt), P.i32(ids[:T]))
        torch.cuda.synchronize()
        P.stage.prefill(len(lens), a[0], a[1], a[2], T, token_ids=a[3], out_hidden=out, out_logits=lg,
                        out_argmax=am)
        P.stage.synchronize()
        got = f32b(out.cpu().view(torch.int16).numpy().view(np.uint16))
        assert hp.rel_err_rows(got, y) < STAGE_TOL
        lg, am = lg.cpu().numpy(), am.cpu().numpy()
        # (i) the argmax kernel is bit-exact on the GPU's own logits, ties -> lowest index
        assert np.array_equal(am, np.argmax(lg, axis=1).astype(np.int32))
        # (ii) ids equal the oracle's wherever the oracle's top-2 margin exceeds 8x the measured logit error
        lerr = np.abs(lg - wl).max()
        safe = wm > 8 * lerr
        print(f"logit max err {lerr:.3e}; rows over margin {safe.sum()}/{len(safe)}")
        assert np.array_equal(am[safe], wa[safe])
        assert hp.rel_err_rows(lg, wl) < STAGE_TOL
        # decode with token ids + logits
        ids_d = ids[T:]
        yd, _ = F32.stage(hp.odims(shape), P.wb, pool0, np.arange(len(lens) + 1, dtype=np.int32), lens, bt,
                          token_ids=ids_d, embed=eb["embed"])
        wl2, wa2, wm2 = F32.logits(hp.odims(shape), yd, eb["final_norm"], eb["lm_head"])
        lg2 = torch.empty((len(lens), shape.vocab), dtype=torch.float32, device="cuda:0")
        am2 = torch.empty((len(lens),), dtype=torch.int32, device="cuda:0")
        a2 = (P.i32(bt), P.i32(lens), P.i32(ids_d))
        torch.cuda.synchronize()
        P.stage.decode(len(lens), a2[0], a2[1], token_ids=a2[2], out_logits=lg2, out_argmax=am2)
        P.stage.synchronize()
        lg2, am2 = lg2.cpu().numpy(), am2.cpu().numpy()
        assert np.array_equal(am2, np.argmax(lg2, axis=1).astype(np.int32))
        assert hp.rel_err_rows(lg2, wl2) < STAGE_TOL
        safe2 = wm2 > 8 * np.abs(lg2 - wl2).max()
        assert np.array_equal(am2[safe2], wa2[safe2])
    finally:
        P.close()


def test_decode_graph_replay_is_deterministic_and_pointer_safe():
    """The decode step is replayed from a CUDA graph; user pointers change between calls (device-side arg block)."""
    shape = synth.TINY
    P, lens, pb, x = _problem(shape, seed=5)
    try:
        bt = pb.block_tables
        T = int(lens.sum())
        P.prefill(lens, bt, x[:T])
        xs = x[T:T + len(lens)]
        snap = P.stage.pool_view().clone()
        y1 = P.decode(lens, bt, xs)
        n1 = P.stage.launch_count()
        P.stage.pool_view().copy_(snap)
        torch.cuda.synchronize()
        y2 = P.decode(lens, bt, xs)            # new tensors -> new pointers, same values
        n2 = P.stage.launch_count()
        assert np.array_equal(y1, y2)
        assert n2 - n1 > 0 and (n2 - n1) == 2 + shape.n_layers * 9
    finally:
        P.close()


@pytest.mark.parametrize("shape", [synth.TINY128, synth.TINY_QWEN])
def test_decode_batch_size_sweep_vs_oracle(shape):
    """Decode batches across every size boundary of the path: the GEMM's token-tile width (32 ... 256 columns, then
    several token tiles), the stream-K pieces left to the consumer kernels or not, the variants of the residual + RMSNorm
    and qkv_post kernels, one CUDA graph per batch size, the decode attention's page split over few or many rows.  One
    stage holds 300 sequences; a prefix of B of them takes one decode step (the others' pages must not change)."""
    n = 300
    rng = np.random.default_rng(21)
    lens = rng.integers(1, 90, size=n).astype(np.int32)
    lens[[0, 7, 130]] = [300, 1, 16]
    P, lens, pb, _ = _problem(shape, seed=6, lens=lens, extra=4)
    try:
        T = int(lens.sum())
        x = synth.bits(synth.hidden_rows(T + n, shape.hidden, 6))
        bt = pb.block_tables
        pool = hp.new_pool(shape, pb.n_pages_pool, P.L)
        hp.run_oracle_prefill(F32, shape, P.wb, pool, lens, bt, x[:T])
        P.prefill(lens, bt, x[:T])
        snap_gpu = P.stage.pool_view().clone()
        worst = 0.0
        for B in (1, 2, 3, 5, 17, 32, 33, 64, 65, 100, 128, 129, 200, 256, 257, 300):
            P.stage.pool_view().copy_(snap_gpu)          # every batch starts from the prefilled pool
            torch.cuda.synchronize()
            pool_b = pool.copy()
            xs = x[T:T + B]
            want, _ = hp.run_oracle_decode(F32, shape, P.wb, pool_b, lens[:B], bt[:B], xs)
            got = P.decode(lens[:B], bt[:B], xs)
            err = hp.rel_err_rows(got, want)
            worst = max(worst, err)
            assert np.isfinite(got).all() and err < STAGE_TOL, (B, err)
            mask = _written_mask(pool.shape, bt[:B], lens[:B] + 1) | _written_mask(pool.shape, bt, lens)
            pg = P.pool_bits()
            assert (pg[~mask] == 0x7FC1).all() and (pg[mask] != 0x7FC1).all(), B
        print(f"{shape.name}: decode batches 1..300, worst stage rel err vs R0 {worst:.3e}")
    finally:
        P.close()


def test_stage_create_destroy_cycles_leak_nothing_on_the_device():
    """A serving process re-creates stages (the paper's reconfiguration after a spot interruption): each
    cycle builds a stage, runs a prefill and two decode steps (which captures and replays a CUDA graph) and destroys it.
    The stage allocates no device memory of its own, so after the first cycles the device's free memory must not move
    and every cycle must give the same bits."""
    import gc
    shape = synth.TINY_QWEN

    def cycle():
        P, lens, pb, x = _problem(shape, seed=4, lens=[40, 17, 70, 3])
        try:
            T = int(lens.sum())
            P.prefill(lens, pb.block_tables, x[:T])
            y = P.decode(lens, pb.block_tables, x[T:T + len(lens)])
            y = P.decode(lens + 1, pb.block_tables, x[T:T + len(lens)])
            return y.copy()
        finally:
            P.close()

    first = cycle()
    for _ in range(2):
        cycle()
    gc.collect()
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(25):
        assert np.array_equal(cycle(), first)
    gc.collect()
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    free1 = torch.cuda.mem_get_info()[0]
    print(f"free device memory before / after 25 cycles: {free0} / {free1}")
    assert free0 - free1 <= 2 << 20   # nothing accumulates (2 MiB of slack for the driver's own pools)


def test_edge_cases_and_error_codes():
    shape = synth.TINY
    gh = _gh()
    from paper_2606_18600_b200 import binding
    # single sequence, single token prompt (ctx = 0), then decode across a page boundary
    P, lens, pb, x = _problem(shape, seed=6, lens=[1], extra=40)
    try:
        bt = pb.block_tables
        pool0 = hp.new_pool(shape, pb.n_pages_pool, P.L)
        want, _, _ = hp.run_oracle_prefill(F32, shape, P.wb, pool0, lens, bt, x[:1])
        got = P.prefill(lens, bt, x[:1])
        assert hp.rel_err_rows(got, want) < STAGE_TOL
        for step in range(18):
            xs = x[1 + step: 2 + step]
            want, _ = hp.run_oracle_decode(F32, shape, P.wb, pool0, lens + step, bt, xs)
            got = P.decode(lens + step, bt, xs)
            assert hp.rel_err_rows(got, want) < STAGE_TOL, step
        # error codes
        st = P.stage
        out = torch.empty((1, shape.hidden), dtype=torch.bfloat16, device="cuda:0")
        btd, cx, hx = P.i32(bt), P.i32(lens), P.bf16(x[:1])
        assert st.decode(1, btd, cx, hidden=None, token_ids=None, out_hidden=out, check=False) == -1
        assert st.decode(1, btd, cx, hidden=hx, token_ids=cx, out_hidden=out, check=False) == -1
        assert st.decode(1, btd, cx, token_ids=cx, out_hidden=out, check=False) == -1      # no embed
        assert st.decode(1, btd, cx, hidden=hx, out_argmax=cx, check=False) == -1           # no lm_head
        assert st.decode(10 ** 6, btd, cx, hidden=hx, out_hidden=out, check=False) == -3
        assert st.prefill(1, cx, cx, btd, 10 ** 7, hidden=hx, out_hidden=out, check=False) == -3
    finally:
        P.close()
    # unsupported dims
    bad = binding.make_dims(synth.TINY, 64, 4, 8)
    bad.head_dim = 96
    lib = binding.load_library()
    import ctypes as C
    assert lib.ss_stage_workspace_bytes(C.byref(bad), 0, 2) == 0


def test_decode_at_maximum_context_many_segments():
    """Contexts at the top of the paper's range (8,192 tokens, BASELINE.json configs[1]) with a tiny batch: every
    (sequence, kv head) pair is cut across hundreds of worker warps, so the split-K partials and the merge carry the
    whole result; plus a 1-token context beside it (a pair that is a single page)."""
    shape = synth.TINY128
    gh = _gh()
    ctx = np.array([8191, 0, 4097], dtype=np.int32)
    rng = np.random.default_rng(8)
    pb = synth.paged_batch(rng, ctx, extra_tokens=2)
    P = gh.Problem(shape, 8, n_pages=pb.n_pages_pool, max_tokens=8, max_seqs=8, max_blocks=pb.max_blocks,
                   pool_fill="random")
    try:
        x = synth.bits(synth.hidden_rows(3, shape.hidden, 8))
        pool = P.pool_cpu.copy()
        want, _ = hp.run_oracle_decode(F32, shape, P.wb, pool, ctx, pb.block_tables, x)
        # max_pos must cover position 8191
        got = P.decode(ctx, pb.block_tables, x)
        assert hp.rel_err_rows(got, want) < STAGE_TOL
    finally:
        P.close()


def test_op_gemm_random_shapes_property():
    """Property test (hypothesis): random ragged (T, N, K) — token tails, weight-row tails, K tails that are only
    multiples of 8 — through both schedules and both epilogues, against a float64 matmul of the same bf16 bits."""
    from hypothesis import given, settings, strategies as st
    from paper_2606_18600_b200 import binding

    @settings(max_examples=30, deadline=None)
    @given(st.integers(1, 700), st.integers(1, 90), st.integers(1, 160), st.booleans(), st.integers(0, 10 ** 6))
    def run(T, n8, k8, dual, seed):
        N, K = 8 * n8, 8 * k8
        g = torch.Generator().manual_seed(seed)
        x = synth.randn_bf16((T, K), 1.0, g)
        w0 = synth.randn_bf16((N, K), 0.06, g)
        xd = x.cuda()
        ref0 = x.double() @ w0.double().T
        if dual:
            w1 = synth.randn_bf16((N, K), 0.06, g)
            got = binding.op_gemm_swiglu_bf16(xd, w0.cuda(), w1.cuda()).float().cpu().double()
            ref = torch.nn.functional.silu(ref0) * (x.double() @ w1.double().T)
            tol = 1e-2 * ref.abs().max() + 1e-6
        else:
            got = binding.op_gemm_bf16(xd, w0.cuda()).cpu().double()
            ref = ref0
            tol = 2e-5 * ref.abs().max() * np.sqrt(max(K, 64) / 64) + 1e-6
        torch.cuda.synchronize()
        assert (got - ref).abs().max() <= tol, (T, N, K, dual)

    run()


def test_graph_replay_equals_stream_launches_bit_for_bit(monkeypatch):
    """The decode step captured into a CUDA graph (with its programmatic-dependency edges) and the same kernels
    launched one by one on the stream produce identical bits, hidden state and KV pool."""
    shape = synth.TINY_QWEN
    gh = _gh()
    P, lens, pb, x = _problem(shape, seed=12)
    monkeypatch.setenv("SS_NO_GRAPH", "1")
    Q = gh.Problem(shape, 12, n_pages=pb.n_pages_pool, max_tokens=int(lens.sum()) + 64, max_seqs=16,
                   max_blocks=pb.max_blocks)
    monkeypatch.delenv("SS_NO_GRAPH")
    try:
        T = int(lens.sum())
        a, b = P.prefill(lens, pb.block_tables, x[:T]), Q.prefill(lens, pb.block_tables, x[:T])
        assert np.array_equal(a, b)
        for step in range(3):
            xs = x[T + step * len(lens): T + (step + 1) * len(lens)]
            ya, yb = P.decode(lens + step, pb.block_tables, xs), Q.decode(lens + step, pb.block_tables, xs)
            assert np.array_equal(ya, yb), step
        assert np.array_equal(P.pool_bits(), Q.pool_bits())
    finally:
        P.close()
        Q.close()


def test_kv_allocator_invariants():
    """P15: alloc/free conserve the page multiset; double free / over-allocation return the documented errors."""
    shape = synth.TINY
    P, lens, pb, x = _problem(shape, seed=7)
    try:
        st = P.stage
        n = st.num_pages()
        assert st.num_free() == n
        a = st.kv_alloc(5)
        b = st.kv_alloc(n - 5)
        assert sorted(a + b) == list(range(n)) and st.num_free() == 0
        import ctypes as C
        one = (C.c_int32 * 1)()
        assert st.lib.ss_kv_alloc(st.h, 1, one) == -4
        st.kv_free(a)
        assert st.num_free() == 5
        arr = (C.c_int32 * 2)(a[0], a[1])
        assert st.lib.ss_kv_free(st.h, 2, arr) == -5 and st.num_free() == 5          # already free
        arr = (C.c_int32 * 2)(b[0], b[0])
        assert st.lib.ss_kv_free(st.h, 2, arr) == -5 and st.num_free() == 5          # duplicate in one call
        arr = (C.c_int32 * 1)(n)
        assert st.lib.ss_kv_free(st.h, 1, arr) == -5                                  # out of range
        c = st.kv_alloc(5)
        assert sorted(c) == sorted(a)
        st.kv_free(b + c)
        assert st.num_free() == n
        rng = np.random.default_rng(0)
        held = []
        for _ in range(200):
            if held and rng.random() < 0.5:
                k = int(rng.integers(1, len(held) + 1))
                idx = rng.permutation(len(held))[:k]
                st.kv_free([held[i] for i in idx])
                held = [h for i, h in enumerate(held) if i not in set(idx.tolist())]
            else:
                k = int(rng.integers(0, st.num_free() + 1))
                got = st.kv_alloc(k)
                assert not set(got) & set(held)
                held += got
            assert st.num_free() + len(held) == n and len(set(held)) == len(held)
    finally:
        P.close()
