"""Thin ctypes binding of libshuntstage.so — same names as include/shuntstage.h, argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch is used here for device memory and streams
only.  There is no CPU fallback: if the library is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import torch

from . import build as _build

_HERE = Path(__file__).resolve().parent
_LIB = None

SS_OK = 0
ERRORS = {0: "SS_OK", -1: "SS_ERR_INVALID_ARG", -2: "SS_ERR_UNSUPPORTED", -3: "SS_ERR_CAPACITY",
          -4: "SS_ERR_NO_PAGES", -5: "SS_ERR_BAD_PAGE", -6: "SS_ERR_CUDA"}

EXPORTS = ["ss_stage_workspace_bytes", "ss_kv_page_bytes", "ss_stage_create", "ss_stage_destroy",
           "ss_kv_num_pages", "ss_kv_num_free", "ss_kv_alloc", "ss_kv_free", "ss_stage_prefill", "ss_stage_mixed",
           "ss_stage_decode",
           "ss_stage_launch_count", "ss_op_gemm_scratch_bytes", "ss_op_gemm_bf16", "ss_op_gemm_swiglu_bf16", "ss_op_gemm_bf16_static", "ss_strerror",
           "ss_last_cuda_error", "ss_version", "ss_debug_buffer", "ss_pool_create", "ss_pool_destroy",
           "ss_pool_num_pages", "ss_pool_num_free", "ss_pool_alloc", "ss_pool_free", "ss_kv_export", "ss_kv_import", "ss_stage_set_allreduce", "ss_stage_set_batch_invariant", "ss_tp_xchg_bytes", "ss_stage_set_tp_fused",
           "ss_stage_debug_tap", "ss_stage_debug_info", "ss_stage_graph_count", "ss_store_alloc", "ss_store_free", "ss_store_upload", "ss_store_export", "ss_store_attach", "ss_store_detach"]


ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)


class ss_model_dims(C.Structure):
    _fields_ = [("hidden", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("ffn", C.c_int32), ("n_layers_total", C.c_int32), ("vocab", C.c_int32),
                ("rms_eps", C.c_float), ("rope_theta", C.c_float), ("qk_norm", C.c_int32),
                ("page_size", C.c_int32), ("max_pos", C.c_int32), ("max_tokens", C.c_int32),
                ("max_seqs", C.c_int32), ("max_blocks_per_seq", C.c_int32)]


class ss_layer_weights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("ln1", "wq", "wk", "wv", "q_norm", "k_norm", "wo", "ln2", "w_gate",
                                          "w_up", "w_down")]


class ss_edge_weights(C.Structure):
    _fields_ = [("embed", C.c_void_p), ("final_norm", C.c_void_p), ("lm_head", C.c_void_p),
                ("inv_freq", C.c_void_p)]


class ShuntStageError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        detail = ""
        if code == -6 and _LIB is not None:
            detail = ": " + _LIB.ss_last_cuda_error().decode()
        super().__init__(f"{where} -> {ERRORS.get(code, code)}{detail}")


def lib_path() -> Path:
    return _HERE / "libshuntstage.so"


def load_library(build_if_missing: bool = True) -> C.CDLL:
    """Load libshuntstage.so (building it with nvcc when absent/stale).  Fails loudly; never falls back."""
    global _LIB
    if _LIB is not None:
        return _LIB
    if build_if_missing:
        _build.build()
    if not lib_path().exists():
        raise FileNotFoundError(f"{lib_path()} is missing: the CUDA extension was not built")
    lib = C.CDLL(str(lib_path()))
    lib.ss_stage_workspace_bytes.restype = C.c_size_t
    lib.ss_stage_workspace_bytes.argtypes = [C.POINTER(ss_model_dims), C.c_int, C.c_int]
    lib.ss_kv_page_bytes.restype = C.c_size_t
    lib.ss_kv_page_bytes.argtypes = [C.POINTER(ss_model_dims), C.c_int, C.c_int]
    lib.ss_stage_create.restype = C.c_int
    lib.ss_stage_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(ss_model_dims), C.c_int, C.c_int,
                                    C.POINTER(ss_layer_weights), C.POINTER(ss_edge_weights), C.c_void_p,
                                    C.c_size_t, C.c_void_p, C.c_size_t, C.c_void_p]
    lib.ss_stage_destroy.argtypes = [C.c_void_p]
    lib.ss_kv_num_pages.argtypes = [C.c_void_p]
    lib.ss_kv_num_free.argtypes = [C.c_void_p]
    lib.ss_kv_alloc.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int32)]
    lib.ss_kv_free.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int32)]
    lib.ss_stage_prefill.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ss_stage_mixed.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                   C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ss_stage_decode.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                    C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ss_stage_launch_count.restype = C.c_int64
    lib.ss_stage_launch_count.argtypes = [C.c_void_p]
    lib.ss_debug_buffer.argtypes = [C.c_void_p]
    lib.ss_stage_debug_info.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
    lib.ss_stage_graph_count.restype = C.c_int64
    lib.ss_stage_graph_count.argtypes = [C.c_void_p]
    lib.ss_stage_debug_tap.argtypes = [C.c_void_p, C.c_char_p, C.POINTER(C.c_void_p), C.POINTER(C.c_size_t)]
    lib.ss_stage_set_allreduce.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    lib.ss_stage_set_batch_invariant.argtypes = [C.c_void_p, C.c_int]
    lib.ss_tp_xchg_bytes.restype = C.c_size_t
    lib.ss_tp_xchg_bytes.argtypes = [C.c_int]
    lib.ss_stage_set_tp_fused.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_void_p)]
    lib.ss_kv_export.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_size_t]
    lib.ss_kv_import.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_size_t]
    lib.ss_pool_create.argtypes = [C.POINTER(C.c_void_p), C.c_int]
    lib.ss_pool_destroy.argtypes = [C.c_void_p]
    lib.ss_pool_num_pages.argtypes = [C.c_void_p]
    lib.ss_pool_num_free.argtypes = [C.c_void_p]
    lib.ss_pool_alloc.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int32)]
    lib.ss_pool_free.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int32)]
    lib.ss_store_alloc.argtypes = [C.POINTER(C.c_void_p), C.c_size_t]
    lib.ss_store_free.argtypes = [C.c_void_p]
    lib.ss_store_upload.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
    lib.ss_store_export.argtypes = [C.c_void_p, C.c_void_p]
    lib.ss_store_attach.argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
    lib.ss_store_detach.argtypes = [C.c_void_p]
    lib.ss_op_gemm_scratch_bytes.restype = C.c_size_t
    lib.ss_op_gemm_bf16.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p,
                                    C.c_size_t, C.c_void_p]
    lib.ss_op_gemm_swiglu_bf16.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                           C.c_int, C.c_void_p, C.c_size_t, C.c_void_p]
    lib.ss_op_gemm_bf16_static.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
    lib.ss_strerror.restype = C.c_char_p
    lib.ss_strerror.argtypes = [C.c_int]
    lib.ss_last_cuda_error.restype = C.c_char_p
    lib.ss_version.restype = C.c_char_p
    _LIB = lib
    return lib


def _ptr(t):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device pointer arguments must be contiguous CUDA tensors"
    return t.data_ptr()


def make_dims(shape, max_tokens, max_seqs, max_blocks, max_pos=8192 + 256, n_layers_total=None) -> ss_model_dims:
    """shape: any object with hidden, n_q, n_kv, d, ffn, n_layers, vocab, eps, theta, qk_norm attributes."""
    return ss_model_dims(shape.hidden, shape.n_q, shape.n_kv, shape.d, shape.ffn,
                         n_layers_total if n_layers_total is not None else shape.n_layers, shape.vocab, shape.eps,
                         shape.theta, shape.qk_norm, 16, max_pos, max_tokens, max_seqs, max_blocks)


class Stage:
    """ss_stage_* with torch tensors as the device buffers.  Owns the KV pool, the workspace and a CUDA stream
    (torch memory), never any arithmetic."""

    def __init__(self, dims: ss_model_dims, l0: int, l1: int, layers: list, edge: dict | None = None,
                 n_pages: int = 0, kv_pool: torch.Tensor | None = None, device="cuda:0", stream=None,
                 inv_freq=None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_18600_b200 needs a CUDA device (sm_100a); there is no CPU path")
        self.lib = load_library()
        self.dims = dims
        self.l0, self.l1 = l0, l1
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
        self._keep = [layers, edge]
        L = l1 - l0
        arr = (ss_layer_weights * L)()
        for i, w in enumerate(layers):
            for name, _ in ss_layer_weights._fields_:
                t = w.get(name)
                setattr(arr[i], name, _ptr(t))
        ew = None
        self._inv = None
        if edge is not None or inv_freq is not None:
            edge = edge or {}
            ew = ss_edge_weights(_ptr(edge.get("embed")), _ptr(edge.get("final_norm")), _ptr(edge.get("lm_head")),
                                 None)
            if inv_freq is not None:
                self._inv = (C.c_float * len(inv_freq))(*[float(v) for v in inv_freq])
                ew.inv_freq = C.cast(self._inv, C.c_void_p)
        page_bytes = self.lib.ss_kv_page_bytes(C.byref(dims), l0, l1)
        if page_bytes == 0:
            raise ShuntStageError(-2, "ss_kv_page_bytes")
        if kv_pool is None:
            kv_pool = torch.empty(n_pages * page_bytes // 2, dtype=torch.bfloat16, device=self.device)
        self.kv_pool = kv_pool
        self.page_bytes = page_bytes
        ws_bytes = self.lib.ss_stage_workspace_bytes(C.byref(dims), l0, l1)
        self.workspace = torch.empty(ws_bytes, dtype=torch.uint8, device=self.device)
        h = C.c_void_p()
        torch.cuda.synchronize(self.device)
        rc = self.lib.ss_stage_create(C.byref(h), C.byref(dims), l0, l1, arr, C.byref(ew) if ew else None,
                                      kv_pool.data_ptr(), kv_pool.numel() * kv_pool.element_size(),
                                      self.workspace.data_ptr(), ws_bytes, self.stream.cuda_stream)
        if rc != SS_OK:
            raise ShuntStageError(rc, "ss_stage_create")
        self.h = h

    # pool view: [L, 2, pages, n_kv, 16, d] bf16
    def pool_view(self) -> torch.Tensor:
        d = self.dims
        n_pages = self.num_pages()
        n = (self.l1 - self.l0) * 2 * n_pages * d.n_kv_heads * 16 * d.head_dim
        return self.kv_pool.view(-1)[:n].view(self.l1 - self.l0, 2, n_pages, d.n_kv_heads, 16, d.head_dim)

    def num_pages(self) -> int:
        return self.lib.ss_kv_num_pages(self.h)

    def num_free(self) -> int:
        return self.lib.ss_kv_num_free(self.h)

    def kv_alloc(self, n: int) -> list:
        out = (C.c_int32 * max(n, 1))()
        rc = self.lib.ss_kv_alloc(self.h, n, out)
        if rc != SS_OK:
            raise ShuntStageError(rc, "ss_kv_alloc")
        return list(out[:n])

    def kv_free(self, ids) -> None:
        ids = list(ids)
        arr = (C.c_int32 * max(len(ids), 1))(*ids)
        rc = self.lib.ss_kv_free(self.h, len(ids), arr)
        if rc != SS_OK:
            raise ShuntStageError(rc, "ss_kv_free")

    def prefill(self, n_seqs, cu_q, ctx_before, block_tables, total_tokens, hidden=None, token_ids=None,
                out_hidden=None, out_logits=None, out_argmax=None, check=True):
        rc = self.lib.ss_stage_prefill(self.h, n_seqs, _ptr(hidden), _ptr(token_ids), _ptr(cu_q), _ptr(ctx_before),
                                       _ptr(block_tables), block_tables.shape[1], total_tokens, _ptr(out_hidden),
                                       _ptr(out_logits), _ptr(out_argmax))
        if check and rc != SS_OK:
            raise ShuntStageError(rc, "ss_stage_prefill")
        return rc

    def mixed(self, n_decode_rows, n_seqs, cu_q, ctx_before, block_tables, total_tokens, hidden=None, token_ids=None,
              out_hidden=None, out_logits=None, out_argmax=None, check=True):
        rc = self.lib.ss_stage_mixed(self.h, n_decode_rows, n_seqs, _ptr(hidden), _ptr(token_ids), _ptr(cu_q),
                                     _ptr(ctx_before), _ptr(block_tables), block_tables.shape[1], total_tokens,
                                     _ptr(out_hidden), _ptr(out_logits), _ptr(out_argmax))
        if check and rc != SS_OK:
            raise ShuntStageError(rc, "ss_stage_mixed")
        return rc

    def decode(self, batch, block_tables, context_lens, hidden=None, token_ids=None, out_hidden=None,
               out_logits=None, out_argmax=None, check=True):
        rc = self.lib.ss_stage_decode(self.h, batch, _ptr(hidden), _ptr(token_ids), _ptr(block_tables),
                                      block_tables.shape[1], _ptr(context_lens), _ptr(out_hidden),
                                      _ptr(out_logits), _ptr(out_argmax))
        if check and rc != SS_OK:
            raise ShuntStageError(rc, "ss_stage_decode")
        return rc

    def set_batch_invariant(self, on: bool = True):
        rc = self.lib.ss_stage_set_batch_invariant(self.h, 1 if on else 0)
        if rc != SS_OK:
            raise ShuntStageError(rc, "ss_stage_set_batch_invariant")

    def set_tp_fused(self, rank: int, size: int, xchg_ptrs):
        """ss_stage_set_tp_fused: xchg_ptrs = device addresses (ints) of every rank's exchange buffer, indexed by rank."""
        arr = (C.c_void_p * max(size, 1))(*[int(p) for p in xchg_ptrs]) if size else None
        rc = self.lib.ss_stage_set_tp_fused(self.h, rank, size, arr)
        if rc != SS_OK:
            raise ShuntStageError(rc, "ss_stage_set_tp_fused")

    def set_allreduce(self, fn):
        """fn(partial: float32 torch view of the workspace, stream_ptr: int) -> None: enqueue an in-place sum across
        the tensor-parallel ranks on that stream (see paper_2606_18600_b200/tp.py).  None clears it."""
        if fn is None:
            self._ar_cb = None
            rc = self.lib.ss_stage_set_allreduce(self.h, None, None)
        else:
            ws, base = self.workspace, self.workspace.data_ptr()

            def tramp(ptr, count, user, stream):
                try:                                   # an exception must not be lost inside the C call
                    off = ptr - base
                    fn(ws[off:off + 4 * count].view(torch.float32), stream)
                    return 0
                except Exception as exc:               # noqa: BLE001 - reported through the return code
                    self._ar_error = exc
                    return 1

            self._ar_cb = ALLREDUCE_FN(tramp)          # keep the trampoline alive
            rc = self.lib.ss_stage_set_allreduce(self.h, C.cast(self._ar_cb, C.c_void_p), None)
        if rc != SS_OK:
            raise ShuntStageError(rc, "ss_stage_set_allreduce")

    def kv_export(self, page_ids: torch.Tensor, buf: torch.Tensor, check=True):
        rc = self.lib.ss_kv_export(self.h, page_ids.numel(), _ptr(page_ids), _ptr(buf), buf.numel() * buf.element_size())
        if check and rc != SS_OK:
            raise ShuntStageError(rc, "ss_kv_export")
        return rc

    def kv_import(self, page_ids: torch.Tensor, buf: torch.Tensor, check=True):
        rc = self.lib.ss_kv_import(self.h, page_ids.numel(), _ptr(page_ids), _ptr(buf), buf.numel() * buf.element_size())
        if check and rc != SS_OK:
            raise ShuntStageError(rc, "ss_kv_import")
        return rc

    def debug_info(self):
        """(checks_on, [code, sequence, index, value]) of ss_stage_debug_info."""
        out = (C.c_int32 * 4)()
        rc = self.lib.ss_stage_debug_info(self.h, out)
        if rc < 0:
            raise ShuntStageError(rc, "ss_stage_debug_info")
        return bool(rc), list(out)

    def debug_tap(self, name: str, rows: int) -> torch.Tensor:
        """ss_stage_debug_tap as a torch view of the workspace: the first `rows` rows of tensor `name`."""
        p, n = C.c_void_p(), C.c_size_t()
        rc = self.lib.ss_stage_debug_tap(self.h, name.encode(), C.byref(p), C.byref(n))
        if rc != SS_OK:
            raise ShuntStageError(rc, "ss_stage_debug_tap")
        off = p.value - self.workspace.data_ptr()
        d = self.dims
        cap = max(d.max_tokens, d.max_seqs)
        dt = torch.float32 if name in ("x", "qkv") else torch.bfloat16
        return self.workspace[off:off + n.value].view(dt).view(cap, -1)[:rows]

    def graph_count(self) -> int:
        return int(self.lib.ss_stage_graph_count(self.h))

    def launch_count(self) -> int:
        return int(self.lib.ss_stage_launch_count(self.h))

    def synchronize(self):
        self.stream.synchronize()

    def destroy(self):
        if getattr(self, "h", None):
            self.stream.synchronize()
            self.lib.ss_stage_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


_SCRATCH = {}


def _op_scratch(device, stream_ptr: int) -> torch.Tensor:
    """Zero-initialised stream-K fix-up scratch for the op-level GEMMs: one per (device, stream), because two GEMMs in
    flight on different streams must not share fix-up flags (torch memory)."""
    key = (str(device), stream_ptr)
    if key not in _SCRATCH:
        n = load_library().ss_op_gemm_scratch_bytes()
        _SCRATCH[key] = torch.zeros(n, dtype=torch.uint8, device=device)
        torch.cuda.synchronize(device)
    return _SCRATCH[key]


def _op_stream(stream):
    return stream if stream is not None else torch.cuda.current_stream()


def op_gemm_bf16(x: torch.Tensor, w: torch.Tensor, stream=None) -> torch.Tensor:
    """C[T,N] fp32 = x[T,K] bf16 @ w[N,K]^T bf16 through the tcgen05 GEMM kernel."""
    lib = load_library()
    T, K = x.shape
    N = w.shape[0]
    st = _op_stream(stream)
    with torch.cuda.stream(st):                      # the output belongs to the stream the kernel runs on
        c = torch.empty((T, N), dtype=torch.float32, device=x.device)
    sc = _op_scratch(x.device, st.cuda_stream)
    rc = lib.ss_op_gemm_bf16(_ptr(x), _ptr(w), _ptr(c), T, N, K, _ptr(sc), sc.numel(), st.cuda_stream)
    if rc != SS_OK:
        raise ShuntStageError(rc, "ss_op_gemm_bf16")
    return c


OP_GEMM_STATIC_MAX_T = 128  # SS_OP_GEMM_STATIC_MAX_T


def op_gemm_bf16_static(x: torch.Tensor, w: torch.Tensor, out: torch.Tensor, stream=None) -> torch.Tensor:
    """ss_op_gemm_bf16_static: out[T,N] fp32 = x[T,K] bf16 @ w[N,K]^T bf16 with the library's own static scratch.  The
    caller passes the output too, so that nothing at all is allocated by the call (T <= OP_GEMM_STATIC_MAX_T)."""
    lib = load_library()
    T, K = x.shape
    N = w.shape[0]
    assert out.shape == (T, N) and out.dtype == torch.float32
    st = _op_stream(stream)
    rc = lib.ss_op_gemm_bf16_static(_ptr(x), _ptr(w), _ptr(out), T, N, K, st.cuda_stream)
    if rc != SS_OK:
        raise ShuntStageError(rc, "ss_op_gemm_bf16_static")
    return out


def op_gemm_swiglu_bf16(x: torch.Tensor, wg: torch.Tensor, wu: torch.Tensor, stream=None) -> torch.Tensor:
    lib = load_library()
    T, K = x.shape
    F = wg.shape[0]
    st = _op_stream(stream)
    with torch.cuda.stream(st):
        a = torch.empty((T, F), dtype=torch.bfloat16, device=x.device)
    sc = _op_scratch(x.device, st.cuda_stream)
    rc = lib.ss_op_gemm_swiglu_bf16(_ptr(x), _ptr(wg), _ptr(wu), _ptr(a), T, F, K, _ptr(sc), sc.numel(),
                                    st.cuda_stream)
    if rc != SS_OK:
        raise ShuntStageError(rc, "ss_op_gemm_swiglu_bf16")
    return a


class PagePool:
    """ss_pool_*: the stand-alone host page allocator (argument marshalling only)."""

    def __init__(self, num_pages: int):
        self.lib = load_library()
        h = C.c_void_p()
        rc = self.lib.ss_pool_create(C.byref(h), num_pages)
        if rc != SS_OK:
            raise ShuntStageError(rc, "ss_pool_create")
        self.h = h

    def num_pages(self) -> int:
        return self.lib.ss_pool_num_pages(self.h)

    def num_free(self) -> int:
        return self.lib.ss_pool_num_free(self.h)

    def alloc(self, n: int):
        """returns (rc, list of ids)"""
        buf = (C.c_int32 * max(n, 1))()
        rc = self.lib.ss_pool_alloc(self.h, n, buf)
        return rc, (list(buf[:n]) if rc == SS_OK else [])

    def free(self, ids) -> int:
        buf = (C.c_int32 * max(len(ids), 1))(*ids)
        return self.lib.ss_pool_free(self.h, len(ids), buf)

    def destroy(self):
        if self.h:
            self.lib.ss_pool_destroy(self.h)
            self.h = None
