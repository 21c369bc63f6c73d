"""libshuntplace.so (the paper's estimator + Algorithm 1) against the Python oracle
(oracle/placement_oracle.py), and the oracle against values fixed by the paper's formulas computed by hand.
CPU only."""
import ctypes as C
import random
import subprocess

import pytest

from oracle import placement_oracle as po
from paper_2606_18600_b200 import placement as pl

LLAMA70B = dict(hidden=8192, hq=8192, hkv=1024, ffn=28672, vocab=128256, n_layers=80, elem_bytes=2)
# PAPER.md:66-75 (Table 1): GB, TFLOPS (BF16 non-sparse), GB/s
TABLE1 = {"L4": (24, 121, 300), "A10G": (24, 70, 600), "L40S": (48, 362, 864), "B200": (180, 4500, 7700)}


def _c_model(m: po.Model):
    return pl.sp_model(m.hidden, m.hq, m.hkv, m.ffn, m.vocab, m.n_layers, m.elem_bytes)


def _c_inst(g: po.Instance):
    return pl.sp_instance(g.flops, g.mem_bw, g.mem_bytes, g.n_gpus, g.alpha_intra, g.beta_intra, g.cost)


def _c_opts(o: po.Opts, beam=1):
    return pl.sp_opts(o.s_in, o.s_out, o.alpha_inter, o.beta_inter, o.act_bytes, o.gamma, o.slo, beam, o.max_stages,
                      o.max_batch)


def test_library_exports_every_declared_symbol():
    lib = pl.load_library()
    import re
    hdr = open(pl._build.HERE.parent / "include" / "shuntplace.h").read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sp_[a-z_]+)\s*\(", hdr))
    assert declared == set(pl.EXPORTS)
    out = subprocess.run(["nm", "-D", "--defined-only", str(pl._build.PLACE_LIB)], capture_output=True, text=True).stdout
    for s in declared:
        assert f" T {s}" in out and hasattr(lib, s)


# ---- pins of the oracle: the paper's formulas worked by hand -----------------------------------------------------
def test_oracle_table2_literals():
    m = po.Model(**LLAMA70B)
    rows = po.table2(m, B=1, s_in=1000, s_out=1, D=1, phase="prefill")
    # QKV prefill FLOPs = B (2 S H^2 + 4 S H H_kv): 2*1000*8192^2 + 4*1000*8192*1024
    assert rows["qkv"][0] == 134_217_728_000 + 33_554_432_000
    # attention prefill: 4 B S^2 H; memory scan B S H + 2 B S H_kv
    assert rows["attention"] == (4 * 1000 * 1000 * 8192, 1000 * 8192 + 2 * 1000 * 1024)
    # up and gate: 4 B S H H_ffn ; B S H + 2 H H_ffn
    assert rows["up_gate"] == (4 * 1000 * 8192 * 28672, 1000 * 8192 + 2 * 8192 * 28672)
    dec = po.table2(m, B=3, s_in=10, s_out=2, D=1, phase="decode")
    # decode attention: sum_{t=1..2} 4 B (S_in + t) H = 4*3*8192*(11 + 12); memory sum_t (B H + 2 B (S_in + t) H_kv)
    assert dec["attention"][0] == 4 * 3 * 8192 * 23
    assert dec["attention"][1] == 2 * 3 * 8192 + 2 * 3 * 23 * 1024
    # tensor parallelism divides weights and FLOPs, not the replicated activation term of the FFN rows
    tp = po.table2(m, B=1, s_in=1000, s_out=1, D=4, phase="prefill")
    assert tp["up_gate"] == (4 * 1000 * 8192 * 28672 / 4, 1000 * 8192 + 2 * 8192 * 28672 / 4)


def test_oracle_p14_gate_up_memory_term_and_roofline_max():
    """DESIGN.md pin P14: cfg-2 gate/up at decode is memory-bound: (64*8192 + 2*8192*28672) * 2 B / 6545 GB/s = 143.7 us."""
    m = po.Model(**{**LLAMA70B, "vocab": 0, "n_layers": 1})
    g = po.Instance(flops=1616.2e12, mem_bw=6545e9, mem_bytes=180e9)
    f, mem = po.table2(m, 64, 1024, 1, 1, "decode")["up_gate"]
    assert abs(mem * 2 / g.mem_bw - 143.7e-6) < 0.1e-6 and f / g.flops < mem * 2 / g.mem_bw
    # Eq. 1 takes the max: a prefill of 4096 tokens is compute-bound on the same row
    f2, mem2 = po.table2(m, 1, 4096, 1, 1, "prefill")["up_gate"]
    assert f2 / g.flops > mem2 * 2 / g.mem_bw
    lat = po.stage_latency(m, g, po.Opts(4096, 1), 1, 1, "prefill", False, False)
    rows = po.table2(m, 1, 4096, 1, 1, "prefill")
    assert abs(lat - sum(max(a / g.flops, b * 2 / g.mem_bw) for k, (a, b) in rows.items() if k != "logits")) < 1e-15


def test_oracle_communication_and_batch_literals():
    m = po.Model(hidden=8192, hq=8192, hkv=1024, ffn=28672, vocab=0, n_layers=2)
    fast = po.Instance(flops=1e30, mem_bw=1e30, mem_bytes=80e9, n_gpus=4, alpha_intra=1e-5, beta_intra=100e9)
    o = po.Opts(s_in=1000, s_out=1, alpha_inter=2e-4, beta_inter=10e9)
    # Eq. 3: 4 (alpha + B S H E / (D beta)) (D - 1) l = 4 * (1e-5 + 16,384,000 / 4e11) * 3 * 2 = 1.22304e-3 s
    lat = po.stage_latency(m, fast, o, 2, 1, "prefill", False, False)
    assert abs(lat - 1.22304e-3) < 1e-9
    # Eq. 2 on top: alpha + B S H E / beta = 2e-4 + 16,384,000 / 1e10 = 1.8384e-3 s
    assert abs(po.stage_latency(m, fast, o, 2, 1, "prefill", False, True) - lat - 1.8384e-3) < 1e-9
    # Eq. 6 (reading A18): one GPU of 80 GB, 2 layers of 855,638,016 params in bf16, requests of 1000 + 24 tokens,
    # 2 * 1024 * 2 B of KV per token per layer: floor((80e9 - 3,422,552,064) / (2 * 1024 * 4096)) = 9128
    g1 = po.Instance(flops=1e15, mem_bw=1e12, mem_bytes=80e9)
    assert po.max_batch(m, [g1], po.Opts(1000, 24), (0,), (2,)) == (80_000_000_000 - 3_422_552_064) // (2 * 1024 * 4096)


def test_oracle_monotonicity():
    m = po.Model(**LLAMA70B)
    g = po.Instance(flops=362e12, mem_bw=864e9, mem_bytes=48e9)
    o = po.Opts(763, 232)
    l1 = po.stage_latency(m, g, o, 10, 8, "decode", False, True)
    assert po.stage_latency(m, g, o, 20, 8, "decode", False, True) > l1          # more layers
    assert po.stage_latency(m, g, o, 10, 16, "decode", False, True) > l1         # bigger batch
    faster = po.Instance(flops=724e12, mem_bw=1728e9, mem_bytes=48e9)
    assert po.stage_latency(m, faster, o, 10, 8, "decode", False, True) < l1     # faster device
    # decode is memory-bound and batches well: doubling B far less than doubles the latency
    assert po.stage_latency(m, g, o, 10, 16, "decode", False, False) < 1.2 * po.stage_latency(m, g, o, 10, 8, "decode", False, False)


# ---- the C++ library against the oracle ---------------------------------------------------------------------------
def _random_problem(rng, n_layers, n_types):
    m = po.Model(hidden=rng.choice([1024, 4096, 8192]), hq=0, hkv=rng.choice([256, 1024]), ffn=rng.choice([4096, 14336, 28672]),
                 vocab=rng.choice([0, 32000, 128256]), n_layers=n_layers)
    m.hq = rng.choice([m.hidden, 2 * m.hidden])
    types = []
    for _ in range(n_types):
        name = rng.choice(list(TABLE1))
        gb, tf, bw = TABLE1[name]
        n_gpus = rng.choice([1, 1, 2, 4])
        types.append(po.Instance(flops=tf * 1e12 * rng.uniform(0.5, 1.0), mem_bw=bw * 1e9 * rng.uniform(0.6, 1.0),
                                 mem_bytes=gb * 1e9, n_gpus=n_gpus, alpha_intra=rng.uniform(2e-6, 2e-5),
                                 beta_intra=rng.uniform(20e9, 400e9), cost=rng.uniform(0.3, 3.0) * n_gpus))
    o = po.Opts(s_in=rng.choice([128, 763, 2048]), s_out=rng.choice([1, 32, 232]), alpha_inter=rng.uniform(5e-5, 5e-4),
                beta_inter=rng.uniform(1e9, 25e9), act_bytes=rng.uniform(0, 2e9), gamma=rng.choice([0.0, 0.0, 0.5]),
                slo=rng.uniform(1.0, 30.0), max_stages=rng.choice([2, 3, 8]), max_batch=rng.choice([0, 64, 256]))
    return m, types, o


def test_stage_latency_and_evaluate_match_oracle():
    rng = random.Random(1)
    for _ in range(200):
        m, types, o = _random_problem(rng, rng.randint(2, 12), rng.randint(1, 3))
        cm, co = _c_model(m), _c_opts(o)
        for phase, pname in ((0, "prefill"), (1, "decode")):
            g = rng.choice(types)
            layers, B = rng.randint(1, m.n_layers), rng.randint(1, 300)
            last, nxt = rng.random() < 0.5, rng.random() < 0.5
            want = po.stage_latency(m, g, o, layers, B, pname, last, nxt)
            got = pl.stage_latency(cm, _c_inst(g), co, layers, B, phase, last, nxt)
            assert abs(got - want) <= 1e-12 * want
        s = rng.randint(1, min(4, m.n_layers))
        layers = rng.choice(list(po.compositions(m.n_layers, s)))
        inst = [rng.randrange(len(types)) for _ in range(s)]
        want = po.evaluate(m, types, o, inst, layers)
        got = pl.evaluate(cm, [_c_inst(g) for g in types], co, inst, layers)
        assert got.batch == want["batch"]
        for k in ("prefill_s", "decode_s", "rps", "cost", "score"):
            assert abs(getattr(got, k) - want[k]) <= 1e-12 * max(abs(want[k]), 1e-300), k


@pytest.mark.parametrize("seed", range(12))
def test_dp_with_unbounded_beam_finds_the_exhaustive_optimum(seed):
    """Algorithm 1 with k large enough to keep every candidate enumerates all placements: it must return the score
    the exhaustive search finds; with k = 1 (the paper's default) it returns a valid placement that cannot beat it."""
    rng = random.Random(100 + seed)
    m, types, o = _random_problem(rng, rng.randint(3, 7), rng.randint(1, 3))
    avail = None if seed % 3 == 0 else [rng.randint(1, 3) for _ in types]
    best = po.brute_force(m, types, o, avail)
    cm, ct = _c_model(m), [_c_inst(g) for g in types]
    rc, p = pl.optimize(cm, ct, _c_opts(o, beam=100000), avail)
    if best is None:
        assert rc == 1
        return
    assert rc == 0 and abs(p.score - best[0]["score"]) <= 1e-12 * abs(best[0]["score"])
    assert sum(p.layers[:p.n_stages]) == m.n_layers and p.n_stages <= o.max_stages
    rc1, p1 = pl.optimize(cm, ct, _c_opts(o, beam=1), avail)
    if rc1 == 0:
        assert sum(p1.layers[:p1.n_stages]) == m.n_layers and p1.score <= best[0]["score"] + 1e-12 * abs(best[0]["score"])
        chk = po.evaluate(m, types, o, list(p1.inst[:p1.n_stages]), list(p1.layers[:p1.n_stages]))
        assert abs(chk["score"] - p1.score) <= 1e-12 * abs(chk["score"])
        if avail is not None:
            assert all(list(p1.inst[:p1.n_stages]).count(t) <= avail[t] for t in range(len(types)))


def test_paper_shaped_cluster_llama70b():
    """Llama-3.1-70B (80 layers) over the paper's mid-tier instance types (Table 1 numbers, 4-GPU L4 / A10G nodes and
    L40S nodes as in its AWS g6 / g5 / g6e cluster): Algorithm 1 places all layers, respects the
    availability limits, and a larger beam never scores lower than k = 1 here."""
    m = po.Model(**LLAMA70B)
    mk = lambda n, gpus, cost: po.Instance(flops=TABLE1[n][1] * 1e12, mem_bw=TABLE1[n][2] * 1e9, mem_bytes=TABLE1[n][0] * 1e9,
                                           n_gpus=gpus, alpha_intra=1e-5, beta_intra=32e9, cost=cost)
    types = [mk("L4", 4, 1.6), mk("A10G", 4, 2.0), mk("L40S", 4, 5.0)]
    o = po.Opts(s_in=763, s_out=232, alpha_inter=2e-4, beta_inter=3e9, act_bytes=1e9, max_stages=8, max_batch=256)
    scores = []
    for k in (1, 4):
        rc, p = pl.optimize(_c_model(m), [_c_inst(g) for g in types], _c_opts(o, beam=k), [4, 4, 2])
        assert rc == 0 and sum(p.layers[:p.n_stages]) == 80 and p.batch >= 1
        inst = list(p.inst[:p.n_stages])
        assert inst.count(0) <= 4 and inst.count(1) <= 4 and inst.count(2) <= 2
        chk = po.evaluate(m, types, o, inst, list(p.layers[:p.n_stages]))
        assert abs(chk["score"] - p.score) <= 1e-12 * chk["score"]
        scores.append(p.score)
        print(f"k={k}: stages {[(['L4x4', 'A10Gx4', 'L40Sx4'][t], l) for t, l in zip(inst, p.layers[:p.n_stages])]}, "
              f"B={p.batch}, rps={p.rps:.3f}, prefill {p.prefill_s:.2f}s decode {p.decode_s:.2f}s, score {p.score:.4f}")
    assert scores[1] >= scores[0] * (1 - 1e-12)


# ---- request dispatch: weighted round-robin on pipeline throughput -------------------------------
def test_wrr_oracle_pins():
    # the textbook worked example of smooth weighted round-robin: weights 5, 1, 1 -> a a b a c a a, then it repeats
    assert po.wrr_sequence([5, 1, 1], 14) == [0, 0, 1, 0, 2, 0, 0] * 2
    # equal weights degenerate to plain round-robin; a single pipeline takes everything; all-zero -> -1
    assert po.wrr_sequence([3, 3, 3, 3], 8) == [0, 1, 2, 3, 0, 1, 2, 3]
    assert po.wrr_sequence([0.7], 3) == [0, 0, 0] and po.wrr_sequence([0, 0], 2) == [-1, -1]
    rng = random.Random(11)
    for _ in range(50):
        w = [rng.randint(0, 9) for _ in range(rng.randint(1, 6))]
        W = sum(w)
        if W == 0:
            continue
        seq = po.wrr_sequence(w, 3 * W)
        # integer weights: every window of one period holds exactly w_i picks of pipeline i ...
        for start in (0, W, 2 * W):
            assert [seq[start:start + W].count(i) for i in range(len(w))] == w
        # ... and at every prefix each pipeline is within one request of its share (what "smooth" means)
        cnt = [0] * len(w)
        for n, i in enumerate(seq, 1):
            cnt[i] += 1
            assert all(abs(cnt[j] - n * w[j] / W) < 1.0 + 1e-9 for j in range(len(w)))


def test_wrr_library_matches_oracle_including_drain_and_shunt():
    rng = random.Random(5)
    for trial in range(30):
        n = rng.randint(1, 7)
        w = [rng.choice([0.0, rng.uniform(0.1, 40.0)]) if trial % 3 else float(rng.randint(1, 9)) for _ in range(n)]
        # a pipeline is drained (weight 0) at some pick and a replacement comes up later (section 5.2)
        victim = rng.randrange(n)
        changes = {17: (victim, 0.0), 41: (victim, rng.uniform(0.5, 30.0))}
        want = po.wrr_sequence(w, 80, changes)
        d = pl.Dispatcher(w)
        got = []
        for k in range(80):
            if k in changes:
                d.set_weight(*changes[k])
            got.append(d.next())
        d.close()
        assert got == want
        assert victim not in got[17:41]
    with pytest.raises(ValueError):
        pl.Dispatcher([1.0, -2.0])
    with pytest.raises(ValueError):
        pl.Dispatcher([])
    with pytest.raises(ValueError):
        pl.Dispatcher([float("nan")])
    d = pl.Dispatcher([1.0])
    with pytest.raises(ValueError):
        d.set_weight(3, 1.0)
    d.close()
    assert pl.load_library().sp_wrr_next(None) == -1 and pl.load_library().sp_wrr_destroy(None) == -1
