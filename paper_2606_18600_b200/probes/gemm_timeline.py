"""gemm_timeline.py — per-CTA timeline of one launch of the tcgen05 GEMM (profiling aid, not part of the product path).

Needs a library built with the trace stamps compiled in:
    SS_NVCC_EXTRA=-DSS_GEMM_TRACE python -m paper_2606_18600_b200.build
    python paper_2606_18600_b200/probes/gemm_timeline.py <name> <T> <N> <K> <dual 0|1>
(rebuild without SS_NVCC_EXTRA afterwards).  The kernel then writes %globaltimer stamps per CTA — kernel start/end,
first tile landed, and per work item: MMAs issued, fix-up flags seen, accumulator complete, epilogue done, plus
per-32-token-chunk stamps inside the second item's epilogue — behind the op-level scratch buffer; this script
prints min/median/max over the 148 CTAs.  Output kept in profiles/r01_gemm_timeline.md.
"""
import os, sys, torch, numpy as np
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
from paper_2606_18600_b200 import binding
dev = torch.device("cuda:0")
name, T, N, K, dual = sys.argv[1], int(sys.argv[2]), int(sys.argv[3]), int(sys.argv[4]), sys.argv[5] == "1"
lib = binding.load_library()
nfix = lib.ss_op_gemm_scratch_bytes()
sc = torch.zeros(nfix + 256 * 64 * 8, dtype=torch.uint8, device=dev)
binding._SCRATCH[str(dev)] = sc
ws = [(torch.randn((N, K), device=dev) * 0.02).to(torch.bfloat16) for _ in range(4)]
x = torch.randn((T, K), device=dev).to(torch.bfloat16)
def one(i):
    if dual: binding.op_gemm_swiglu_bf16(x, ws[(2 * i) % 4], ws[(2 * i + 1) % 4])
    else: binding.op_gemm_bf16(x, ws[i % 4])
for i in range(4): one(i)
torch.cuda.synchronize()
sc[nfix:].zero_(); torch.cuda.synchronize()
one(5); torch.cuda.synchronize()
tr = sc[nfix:].view(torch.int64).cpu().numpy().reshape(256, 64)[:148].astype(np.float64)
t0 = tr[:, 0].min()
rel = lambda a: (a - t0) / 1e3
print(name, "kernel span us: start spread %.1f, end min/median/max %.1f %.1f %.1f" % (rel(tr[:, 0]).max(), rel(tr[:, 1]).min(), np.median(rel(tr[:, 1])), rel(tr[:, 1]).max()))
print(" setup done (barriers, TMEM) median %.2f; first TMA issued %.2f; first tile landed (issuer 0): median %.2f max %.2f" % (np.median((tr[:, 7] - tr[:, 0]) / 1e3), np.median((tr[:, 8] - tr[:, 0]) / 1e3), np.median((tr[:, 2] - tr[:, 0]) / 1e3), ((tr[:, 2] - tr[:, 0]) / 1e3).max()))
nit = int(((tr[:, 3::4][:, :8] > 0).sum(axis=1)).max())
for it in range(nit):
    b = 3 + 4 * it
    ok = tr[:, b + 3] > 0
    if ok.sum() == 0: continue
    f = lambda c: "%.1f/%.1f/%.1f" % (rel(tr[ok, c]).min(), np.median(rel(tr[ok, c])), rel(tr[ok, c]).max())
    print(f" item {it} (n={int(ok.sum())}): mma issued {f(b)}  flags ok {f(b+1)}  tfull {f(b+2)}  epi done {f(b+3)}   [min/med/max us]")
    d = (tr[ok, b + 3] - tr[ok, b + 2]) / 1e3
    w = (tr[ok, b + 2] - tr[ok, b]) / 1e3
    print("    epilogue duration med %.1f max %.1f; tfull - issued med %.1f" % (np.median(d), d.max(), np.median(w)))

ok = tr[:, 60] > 0
if ok.sum():
    base = tr[ok, 5 + 4]   # tfull of item 1
    print(" item 1 fine stamps (us after tfull, median over %d CTAs):" % ok.sum())
    for c in range(8):
        a, b2 = tr[ok, 40 + 3 * c], tr[ok, 41 + 3 * c]
        if (a > 0).sum() == 0: break
        print("   chunk %d: tmem loaded %.2f, fix-up done %.2f" % (c, np.median((a - base) / 1e3), np.median((b2 - base) / 1e3)))
    print("   stores done %.2f" % np.median((tr[ok, 60] - base) / 1e3))
