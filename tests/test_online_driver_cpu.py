"""Host logic of the online mixed-batch driver (paper_2606_18600_b200/online.py) without a GPU: its planning and page
bookkeeping driven for more iterations than BASELINE.json's cfg-5 asks for (500), over the library's own host page
allocator (ss_pool_*), with a stage stand-in that computes nothing.  Invariants: every iteration has the 96 decode rows,
no page belongs to two requests, every row's pages cover its tokens, the pool never over-commits, prefill makes progress."""
import numpy as np

from paper_2606_18600_b200 import binding, online


class _HostStage:
    """The allocator half of binding.Stage over ss_pool_* (host only); no forward pass."""

    def __init__(self, n_pages):
        self.pool = binding.PagePool(n_pages)
        self.n = n_pages

    def num_pages(self):
        return self.n

    def num_free(self):
        return self.pool.num_free()

    def kv_alloc(self, n):
        rc, ids = self.pool.alloc(n)
        assert rc == 0, rc
        return ids

    def kv_free(self, ids):
        assert self.pool.free(ids) == 0


def _run(seed, iters, n_pages=None):
    n_pages = n_pages or online.OnlineDriver.pool_pages(seed)
    st = _HostStage(n_pages)
    drv = online.OnlineDriver(st, shape=None, seed=seed, device="cpu")
    tokens_prefilled = 0
    for it in range(iters):
        rows = drv.plan()
        assert len(rows) >= online.N_DECODE and all(q == 1 for _, q in rows[:online.N_DECODE])
        assert [r for r, _ in rows[:online.N_DECODE]] == drv.decode
        owned = [p for r, _ in rows for p in r.pages] + [p for r in drv.fifo for p in r.pages] + \
                [p for r in drv.prefill if all(r is not x for x, _ in rows) for p in r.pages]
        assert len(owned) == len(set(owned)), "a page belongs to two requests"
        assert len(owned) + st.num_free() == n_pages, "pages leaked or over-committed"
        for r, q in rows:
            assert len(r.pages) * online.PAGE >= r.ctx + q and len(r.pages) <= drv.max_blocks
        for r, q in rows[online.N_DECODE:]:
            assert 0 < q <= online.CHUNK and r.ctx + q <= r.prompt
            tokens_prefilled += q
        drv._advance(rows)
    return drv, tokens_prefilled


def test_online_driver_runs_the_baseline_iteration_count_without_exhausting_the_pool():
    for seed in (0, 1, 2):
        drv, pre = _run(seed, 1200)
        s = drv.stats
        assert s["decode_tokens"] == 1200 * online.N_DECODE and s["prefill_tokens"] == pre > 0
        assert s["finished"] > 0 and max(s["occupancy"]) <= 1.0
        print(f"seed {seed}: prefill tokens {pre}, finished {s['finished']}, dropped {s['dropped']}, "
              f"preempted {s['preempted']}, occupancy {min(s['occupancy']):.3f}..{max(s['occupancy']):.3f}")


def test_online_driver_preempts_instead_of_failing_when_the_pool_is_tight():
    """A pool with barely more than the live pages: decode rows still always get their page (prompts in mid-prefill and
    FIFO entries give theirs back), nothing is leaked."""
    seed = 3
    rng = np.random.default_rng(seed)
    live = sum((online.OnlineDriver._draw_decode(rng)[0] + 1 + online.PAGE - 1) // online.PAGE for _ in range(online.N_DECODE))
    drv, _ = _run(seed, 600, n_pages=live + online.N_DECODE + 40)
    assert drv.stats["decode_tokens"] == 600 * online.N_DECODE
    assert drv.stats["preempted"] + drv.stats["dropped"] >= 0
