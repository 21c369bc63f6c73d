"""P15: the host page allocator behind ss_kv_alloc/free (paged KV cache), driven
through the stand-alone ss_pool_* C-ABI — no device needed.  A model (a Python set) is the reference."""
import pytest
from hypothesis import given, settings, strategies as st

from paper_2606_18600_b200 import binding

NO_PAGES, BAD_PAGE, INVALID = -4, -5, -1


def test_pool_hands_out_every_page_once_then_refuses():
    p = binding.PagePool(37)
    assert p.num_pages() == 37 and p.num_free() == 37
    rc, a = p.alloc(30)
    assert rc == 0 and len(set(a)) == 30 and all(0 <= i < 37 for i in a)
    rc, none = p.alloc(8)                        # all-or-nothing
    assert rc == NO_PAGES and none == [] and p.num_free() == 7
    rc, b = p.alloc(7)
    assert rc == 0 and set(a) | set(b) == set(range(37))
    assert p.free([a[0], a[0]]) == BAD_PAGE and p.num_free() == 0      # duplicate inside one call: nothing freed
    assert p.free([a[1], 37]) == BAD_PAGE and p.num_free() == 0        # out of range: nothing freed
    assert p.free(a[:5]) == 0 and p.num_free() == 5
    assert p.free([a[0]]) == BAD_PAGE                                   # double free
    assert p.alloc(-1)[0] == INVALID
    p.destroy()


@settings(max_examples=200, deadline=None)
@given(st.integers(1, 64), st.lists(st.tuples(st.booleans(), st.integers(0, 70), st.integers(0, 2 ** 31 - 1)),
                                    max_size=60))
def test_pool_matches_set_model(n_pages, ops):
    """Random alloc/free sequences: the multiset of pages is conserved, no page is handed out twice, errors leave
    the pool untouched."""
    import random
    p = binding.PagePool(n_pages)
    held = set()
    try:
        for is_alloc, n, seed in ops:
            if is_alloc:
                rc, ids = p.alloc(n)
                if n > n_pages - len(held):
                    assert rc == NO_PAGES and ids == []
                else:
                    assert rc == 0 and len(ids) == n and len(set(ids)) == n
                    assert not (set(ids) & held) and all(0 <= i < n_pages for i in ids)
                    held |= set(ids)
            else:
                rnd = random.Random(seed)
                pick = rnd.sample(sorted(held), min(n, len(held)))
                poison = rnd.random() < 0.3
                if poison:                                   # one bad id anywhere in the list voids the call
                    bad = rnd.choice([-1, n_pages, *(sorted(set(range(n_pages)) - held)[:1]), *(pick[:1])])
                    pick_bad = pick + [bad]
                    rnd.shuffle(pick_bad)
                    assert p.free(pick_bad) == BAD_PAGE
                else:
                    assert p.free(pick) == 0
                    held -= set(pick)
            assert p.num_free() == n_pages - len(held)
    finally:
        p.destroy()
