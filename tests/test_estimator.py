"""P14: the paper's Eq. 1 / Table 2 estimator (report-only host arithmetic) against hand-checkable values."""
from paper_2606_18600_b200 import estimator as est, synth


def golden():
    return {l.split()[0]: float(l.split()[1]) for l in open("tests/golden/estimator_p14.txt")
            if l.strip() and not l.startswith("#")}


def test_P14_estimator_values():
    g = golden()
    F, BW = 1616.2e12, 6545e9
    rows = est.decode_rows(synth.LLAMA70B, synth.cfg2_contexts(0), F, BW)
    assert abs(rows["up_gate"] * 1e6 - g["up_gate_us"]) < 0.05
    # the closed form retyped from Table 2's memory column: (B*H + 2*H*H_ffn) * E / BW
    assert abs(rows["up_gate"] - (64 * 8192 + 2 * 8192 * 28672) * 2 / BW) < 1e-12
    assert abs(est.decode_step_ms(synth.LLAMA70B, synth.cfg2_contexts(0), F, BW) - g["cfg2_ms"]) < 2e-3
    assert abs(est.decode_step_ms(synth.QWEN32B, synth.cfg3_contexts(0), F, BW) - g["cfg3_ms"]) < 2e-3
    assert abs(est.prefill_ms(synth.LLAMA70B, synth.cfg4_lengths(0), F, BW) / 1e3 - g["cfg4_s"]) < 1e-3
    assert abs(est.decode_step_ms(synth.LLAMA70B, synth.cfg2_contexts(0), 4500e12, 7700e9) - g["cfg2_ms_table1_b200"]) < 2e-3


def test_seed0_workload_draws_match_design():
    c2, c3, l4 = synth.cfg2_contexts(0), synth.cfg3_contexts(0), synth.cfg4_lengths(0)
    assert (len(c2), int(c2.sum()), int(c2.min()), int(c2.max())) == (64, 84035, 201, 4039)
    assert (len(c3), int(c3.sum())) == (128, 127041)
    assert (len(l4), int(l4.sum()), int(l4.min()), int(l4.max())) == (32, 40173, 256, 3123)
    # decode is memory-bound on every row, prefill compute-bound on every GEMM row
    rows = est.decode_rows(synth.LLAMA70B, c2, 1616.2e12, 6545e9)
    assert max(rows, key=rows.get) == "up_gate"


def test_bench_estimator_column_agrees_with_libshuntplace_on_uniform_batches():
    """Two restatements of Eq. 1 + Table 2 in this repo — the per-sequence report column of bench.py (estimator.py) and
    the placement library's stage latency (csrc/placement.cpp) — must give the same number where both apply: one
    decode iteration (S_out = 1) or one prefill of a batch of equal lengths, D_TP = 1, no communication, no logits."""
    import numpy as np
    from paper_2606_18600_b200 import estimator, placement as pl, synth
    for shape in (synth.LLAMA70B, synth.QWEN32B):
        m = pl.sp_model(shape.hidden, shape.hq, shape.hkv, shape.ffn, 0, shape.n_layers, 2)
        g = pl.sp_instance(1624.1e12, 6545.3e9, 180e9, 1, 0.0, 1.0, 1.0)
        for B, S in ((64, 1313), (128, 992), (1, 17), (32, 1255)):
            o = pl.sp_opts(float(S), 1.0, 0.0, 1e30, 0.0, 0.0, 0.0, 1, 8, 0)
            dec = pl.stage_latency(m, g, o, shape.n_layers, B, 1, False, False) * 1e3
            want = estimator.decode_step_ms(shape, np.full(B, S), g.flops, g.mem_bw)
            assert abs(dec - want) <= 1e-12 * want
            pre = pl.stage_latency(m, g, o, shape.n_layers, B, 0, False, False) * 1e3
            want_p = estimator.prefill_ms(shape, np.full(B, S), g.flops, g.mem_bw)
            assert abs(pre - want_p) <= 1e-12 * want_p
