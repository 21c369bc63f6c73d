"""CPU-only checks of the boundary: libshuntstage.so builds, loads without a GPU and exports every symbol that
include/shuntstage.h declares; host-only entry points behave as documented.  No compute calls here."""
import ctypes as C
import re
from pathlib import Path

from paper_2606_18600_b200 import binding, synth

ROOT = Path(__file__).resolve().parent.parent


def declared_symbols():
    text = (ROOT / "include" / "shuntstage.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ss_[a-z0-9_]+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    lib = binding.load_library()
    syms = declared_symbols()
    assert set(syms) == set(binding.EXPORTS), (syms, binding.EXPORTS)
    for s in syms:
        assert hasattr(lib, s), s
    assert b"sm_100a" in lib.ss_version()


def test_strerror_and_workspace_query_are_host_only():
    lib = binding.load_library()
    assert lib.ss_strerror(0) == b"ok" and lib.ss_strerror(-4) == b"not enough free KV pages"
    d = binding.make_dims(synth.LLAMA70B, 64, 64, 520)
    ws = lib.ss_stage_workspace_bytes(C.byref(d), 0, 20)
    assert 0 < ws < 2 << 30
    # page bytes: (l1-l0) * 2 * n_kv * 16 * d * 2  (one page (K+V, one layer) = 65,536 B at cfg-2)
    assert lib.ss_kv_page_bytes(C.byref(d), 0, 20) == 20 * 65536
    assert lib.ss_kv_page_bytes(C.byref(d), 3, 4) == 65536
    t = binding.make_dims(synth.TINY, 64, 4, 16)
    assert lib.ss_kv_page_bytes(C.byref(t), 0, 2) == 2 * 8192
    # bad layer ranges and unsupported dims -> 0
    assert lib.ss_stage_workspace_bytes(C.byref(d), 5, 5) == 0
    assert lib.ss_stage_workspace_bytes(C.byref(d), 0, 21) == 0
    d.page_size = 32
    assert lib.ss_stage_workspace_bytes(C.byref(d), 0, 20) == 0


def test_create_rejects_bad_arguments_before_touching_cuda():
    lib = binding.load_library()
    d = binding.make_dims(synth.TINY, 64, 4, 16)
    h = C.c_void_p()
    assert lib.ss_stage_create(C.byref(h), C.byref(d), 0, 2, None, None, None, 0, None, 0, None) == -1
    assert lib.ss_stage_create(None, C.byref(d), 0, 2, None, None, None, 0, None, 0, None) == -1
    d.head_dim = 96
    arr = (binding.ss_layer_weights * 2)()
    assert lib.ss_stage_create(C.byref(h), C.byref(d), 0, 2, arr, None, 1024, 1 << 20, 1024, 1 << 20, None) == -2
    assert lib.ss_kv_num_pages(None) == -1 and lib.ss_kv_alloc(None, 1, None) == -1


def test_tp_exchange_buffer_size_is_host_only_arithmetic():
    """ss_tp_xchg_bytes (fused tensor-parallel all-reduce): 2 buffers x D_TP source regions of 320 slots of 128 x 128 fp32,
    plus one 128-byte counter line per (buffer, source); 0 for a degree outside 1..8."""
    lib = binding.load_library()
    for size in range(1, 9):
        assert lib.ss_tp_xchg_bytes(size) == 2 * size * 320 * 128 * 128 * 4 + 2 * size * 128
    assert lib.ss_tp_xchg_bytes(0) == 0 and lib.ss_tp_xchg_bytes(9) == 0 and lib.ss_tp_xchg_bytes(-1) == 0
    assert lib.ss_stage_set_tp_fused(None, 0, 1, None) == -1 and lib.ss_stage_set_batch_invariant(None, 1) == -1
