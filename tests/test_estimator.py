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
