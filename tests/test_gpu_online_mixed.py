"""BASELINE.json configs[4] ("cfg-5"): online mixed batches on Qwen3-32B layer shapes — each iteration ONE
ss_stage_prefill call of 96 decode rows + up to 4 prefill chunks of <= 512 tokens, over a page pool sized for 85%
occupancy and churned through ss_kv_alloc/free by the driver in paper_2606_18600_b200/online.py.  A 2-layer stage of
the real width; iteration 0 and a late iteration are checked against the oracle on sampled sequences (a sequence's
rows depend on no other sequence: pin P9), starting from a snapshot of the GPU pool taken before the call."""
import numpy as np
import pytest
import torch

from oracle import Oracle
from paper_2606_18600_b200 import binding, online, synth
from tests import helpers as hp

pytestmark = pytest.mark.gpu
F32 = Oracle("f32")
DEV = "cuda:0"


def _pool_bits(stage):
    stage.synchronize()
    return stage.pool_view().cpu().view(torch.int16).numpy().view(np.uint16)


def _check_iteration(shape, wb, pool_before, it, x_bits, got, picks, tag):
    lens = it.ctx_before + (it.cu_q[1:] - it.cu_q[:-1])
    worst = 0.0
    for s in picks:
        rows = np.arange(it.cu_q[s], it.cu_q[s + 1])
        pool = pool_before.copy() if len(picks) == 1 else pool_before.copy()
        want, _, _ = hp.run_oracle_prefill(F32, shape, wb, pool, lens[s:s + 1], it.block_tables[s:s + 1], x_bits[rows],
                                           ctx_before=it.ctx_before[s:s + 1])
        err = hp.rel_err_rows(got[rows], want)
        worst = max(worst, err)
        print(f"{tag}: seq {s} (ctx {int(it.ctx_before[s])}, q_len {len(rows)}): max row rel err {err:.3e}")
    assert worst < 2e-2


def test_online_mixed_batches_vs_oracle_and_pool_invariants():
    full = synth.QWEN32B
    shape = synth.ModelShape(full.name, full.hidden, full.n_q, full.n_kv, full.d, full.ffn, 2, full.eps, full.theta,
                             full.qk_norm, full.vocab)
    seed, iters = 0, 10
    tw, wb = hp.weights_bits(shape, seed)
    dw = [{k: (None if v is None else v.to(DEV)) for k, v in w.items()} for w in tw]
    n_pages = online.OnlineDriver.pool_pages(seed)
    S = online.N_DECODE + online.N_PREFILL
    Tmax = online.N_DECODE + online.N_PREFILL * online.CHUNK
    max_blocks = (8192 + 2048 + online.CHUNK) // 16 + 2
    dims = binding.make_dims(shape, max_tokens=Tmax, max_seqs=S, max_blocks=max_blocks, n_layers_total=2,
                             max_pos=8192 + 2048 + online.CHUNK + 64)
    st = binding.Stage(dims, 0, 2, dw, None, n_pages=n_pages, device=DEV)
    try:
        g = torch.Generator(device=DEV).manual_seed(5)
        pool = st.pool_view()
        for l in range(2):                                    # random KV pre-fill N(0,1) (reading A21)
            pool[l].copy_(torch.randn(pool[l].shape, generator=g, device=DEV, dtype=torch.float32).to(torch.bfloat16))
        drv = online.OnlineDriver(st, shape, seed=seed, max_blocks=max_blocks, device=DEV)
        assert 0.75 <= drv.occupancy() <= 0.86
        out = torch.empty((Tmax, shape.hidden), dtype=torch.bfloat16, device=DEV)
        for i in range(iters):
            x = synth.hidden_rows(Tmax, shape.hidden, seed, idx=100 + i)
            checked = i in (0, iters - 1)
            before = _pool_bits(st).copy() if checked else None
            it = drv.step(x.to(DEV), out)
            # allocator invariants (P15) while the pool churns: no page owned twice, free + owned = all
            owned = [p for r in drv.decode + drv.prefill + list(drv.fifo) for p in r.pages]
            assert len(owned) == len(set(owned)) and len(owned) + st.num_free() == n_pages
            if checked:
                got = synth.bf16_bits_to_f32(out[:it.T].cpu().view(torch.int16).numpy().view(np.uint16))
                assert np.isfinite(got).all()
                q = it.cu_q[1:] - it.cu_q[:-1]
                dec = np.argsort(it.ctx_before[:online.N_DECODE])[:2]           # two shortest decode rows
                chunks = np.arange(online.N_DECODE, it.n_seqs)
                picks = list(dec) + ([int(chunks[np.argmin(q[chunks])])] if len(chunks) else [])
                _check_iteration(shape, wb, before, it, synth.bits(x), got, picks, f"iteration {i}")
        occ = drv.stats["occupancy"]
        print(f"cfg5 x{iters}: decode tokens {drv.stats['decode_tokens']}, prefill tokens {drv.stats['prefill_tokens']}, "
              f"finished {drv.stats['finished']}, dropped {drv.stats['dropped']}, occupancy min/max "
              f"{min(occ):.3f}/{max(occ):.3f}")
        assert drv.stats["decode_tokens"] == online.N_DECODE * iters and drv.stats["prefill_tokens"] > 0
        assert max(occ) <= 0.93
    finally:
        st.destroy()
