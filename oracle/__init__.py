"""CPU oracle of one ShuntServe pipeline stage — TEST INFRASTRUCTURE, not product.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  It shares no code with ``paper_2606_18600_b200`` (the CUDA path) and never imports it.

``stage_oracle.c`` holds the arithmetic (one C file, written from the paper: see its header).  This module only
compiles it with gcc (``build()``), loads it with ctypes and marshals numpy arrays.  Two builds of the same
source: ``f32`` (the oracle proper; north_star fixes "plain fp32") and ``f64`` (all arithmetic in double; exists
to bound the fp32 build's own rounding error, pin P13).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading
from dataclasses import dataclass
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "stage_oracle.c"
_LOCK = threading.Lock()
_LIBS: dict[str, C.CDLL] = {}


def _lib_path(prec: str) -> Path:
    return _HERE / f"libstage_oracle_{prec}.so"


def build(force: bool = False) -> None:
    """Compile both builds of the oracle with gcc (portable x86-64-v3 code: AVX2 + FMA, no -ffast-math)."""
    for prec, defs in (("f32", []), ("f64", ["-DSO_F64"])):
        out = _lib_path(prec)
        if not force and out.exists() and out.stat().st_mtime >= _SRC.stat().st_mtime:
            continue
        cmd = ["gcc", "-O3", "-march=x86-64-v3", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-fno-fast-math",
               *defs, str(_SRC), "-o", str(out), "-lm"]
        subprocess.run(cmd, check=True)


def _load(prec: str) -> C.CDLL:
    with _LOCK:
        if prec not in _LIBS:
            build()
            _LIBS[prec] = C.CDLL(str(_lib_path(prec)))
        return _LIBS[prec]


class _Dims(C.Structure):
    _fields_ = [("hidden", C.c_int32), ("n_q", C.c_int32), ("n_kv", C.c_int32), ("d", C.c_int32),
                ("ffn", C.c_int32), ("vocab", C.c_int32), ("eps", C.c_float), ("theta", C.c_float),
                ("qk_norm", C.c_int32), ("rounding", C.c_int32)]


class _Taps(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("h1", "q", "attn", "x1", "a")]


@dataclass
class OracleDims:
    hidden: int
    n_q: int
    n_kv: int
    d: int
    ffn: int
    vocab: int = 0
    eps: float = 1e-5
    theta: float = 5e5
    qk_norm: int = 0
    rounding: int = 0  # 0 = R0 (plain), 1 = R1 (bf16 at materialisation points)

    def c(self) -> _Dims:
        return _Dims(self.hidden, self.n_q, self.n_kv, self.d, self.ffn, self.vocab, self.eps, self.theta,
                     self.qk_norm, self.rounding)


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _u16(a):
    """bf16 bit patterns: accept uint16/int16 numpy arrays, C-contiguous."""
    if a is None:
        return None
    a = np.ascontiguousarray(a)
    assert a.dtype in (np.uint16, np.int16), a.dtype
    return a.view(np.uint16)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


class Oracle:
    """numpy front-end.  ``real`` is np.float32 (prec='f32') or np.float64 (prec='f64')."""

    def __init__(self, prec: str = "f32"):
        assert prec in ("f32", "f64")
        self.prec = prec
        self.lib = _load(prec)
        self.real = np.float32 if prec == "f32" else np.float64
        self.lib.so_real_bytes.restype = C.c_int
        assert self.lib.so_real_bytes() == np.dtype(self.real).itemsize
        self.lib.so_f32_to_bf16.restype = C.c_uint16
        self.lib.so_f32_to_bf16.argtypes = [C.c_float]
        self.lib.so_bf16_to_f32.restype = C.c_float
        self.lib.so_bf16_to_f32.argtypes = [C.c_uint16]
        self.lib.so_layer.restype = C.c_int
        self.lib.so_swiglu.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_int]

    # -- helpers ------------------------------------------------------------------------------------------
    def _r(self, a):
        return np.ascontiguousarray(a, dtype=self.real)

    def threads(self) -> int:
        return len(os.sched_getaffinity(0))

    # -- element ops --------------------------------------------------------------------------------------
    def f32_to_bf16(self, f: float) -> int:
        return int(self.lib.so_f32_to_bf16(C.c_float(f)))

    def bf16_to_f32(self, b: int) -> float:
        return float(self.lib.so_bf16_to_f32(C.c_uint16(b)))

    def rmsnorm(self, x, w_bf16, eps, round_out=0):
        x = self._r(x)
        T, n = x.shape
        out = np.empty_like(x)
        self.lib.so_rmsnorm(_p(x), _p(_u16(w_bf16)), _p(out), C.c_int(T), C.c_int(n), C.c_float(eps),
                            C.c_int(round_out))
        return out

    def matmul(self, x, w_bf16):
        """x [T,K] real, w [N,K] bf16 bits -> [T,N] real."""
        x = self._r(x)
        w = _u16(w_bf16)
        T, K = x.shape
        N = w.shape[0]
        assert w.shape[1] == K
        out = np.empty((T, N), dtype=self.real)
        self.lib.so_matmul(_p(x), _p(w), _p(out), C.c_int(T), C.c_int(N), C.c_int(K), C.c_int(N))
        return out

    def head_rmsnorm(self, u, g_bf16, eps):
        u = self._r(u).copy()
        T, nh, d = u.shape
        self.lib.so_head_rmsnorm(_p(u), _p(_u16(g_bf16)), C.c_int(T), C.c_int(nh), C.c_int(d), C.c_float(eps))
        return u

    def rope(self, u, pos, theta, inv_freq=None):
        u = self._r(u).copy()
        T, nh, d = u.shape
        pos = _i32(pos)
        inv = None if inv_freq is None else np.ascontiguousarray(inv_freq, dtype=np.float32)
        self.lib.so_rope(_p(u), _p(pos), C.c_int(T), C.c_int(nh), C.c_int(d), C.c_float(theta), _p(inv))
        return u

    def swiglu(self, g, u, round_out=0):
        g = self._r(g)
        u = self._r(u)
        a = np.empty_like(g)
        self.lib.so_swiglu(_p(g), _p(u), _p(a), g.size, round_out)
        return a

    def kv_append(self, k, v, kpool, vpool, cu_q, ctx_before, bt):
        """k, v [T,n_kv,d] real; kpool/vpool [pages,n_kv,16,d] uint16, modified in place."""
        k = self._r(k)
        v = self._r(v)
        T, n_kv, d = k.shape
        cu_q, ctx_before, bt = _i32(cu_q), _i32(ctx_before), _i32(bt)
        assert kpool.dtype == np.uint16 and kpool.flags.c_contiguous
        assert vpool.dtype == np.uint16 and vpool.flags.c_contiguous
        self.lib.so_kv_append(_p(k), _p(v), _p(kpool), _p(vpool), C.c_int(len(ctx_before)), _p(cu_q),
                              _p(ctx_before), _p(bt), C.c_int(bt.shape[1]), C.c_int(n_kv), C.c_int(d))

    def attention(self, q, kpool, vpool, cu_q, ctx_before, bt, round_out=0):
        """q [T,n_q,d] real; pools [pages,n_kv,16,d] uint16 -> [T,n_q,d] real."""
        q = self._r(q)
        T, n_q, d = q.shape
        n_kv = kpool.shape[1]
        cu_q, ctx_before, bt = _i32(cu_q), _i32(ctx_before), _i32(bt)
        out = np.empty_like(q)
        self.lib.so_attention(_p(q), _p(kpool), _p(vpool), _p(out), C.c_int(len(ctx_before)), _p(cu_q),
                              _p(ctx_before), _p(bt), C.c_int(bt.shape[1]), C.c_int(n_q), C.c_int(n_kv),
                              C.c_int(d), C.c_int(round_out))
        return out

    def attention_weights(self, qv, kpool, bt_row, p, hk):
        qv = self._r(qv)
        n_kv, d = kpool.shape[1], kpool.shape[3]
        w = np.empty(p + 1, dtype=self.real)
        bt_row = _i32(bt_row)
        self.lib.so_attention_weights(_p(qv), _p(kpool), _p(bt_row), C.c_int(p), C.c_int(hk), C.c_int(n_kv),
                                      C.c_int(d), _p(w))
        return w

    def embed(self, emb_bf16, ids, H):
        ids = _i32(ids)
        x = np.empty((len(ids), H), dtype=self.real)
        self.lib.so_embed(_p(_u16(emb_bf16)), _p(ids), _p(x), C.c_int(len(ids)), C.c_int(H))
        return x

    # -- whole layer / stage ------------------------------------------------------------------------------
    def layer(self, dims: OracleDims, w: dict, kpool, vpool, cu_q, ctx_before, bt, x, inv_freq=None,
              taps: bool = False):
        """One decoder layer.  ``w``: dict of bf16-bit arrays (ln1,wq,wk,wv,q_norm,k_norm,wo,ln2,w_gate,w_up,
        w_down).  ``x`` [T,H] real is updated IN PLACE.  Returns a dict of taps if requested."""
        assert x.dtype == self.real and x.flags.c_contiguous
        cu_q, ctx_before, bt = _i32(cu_q), _i32(ctx_before), _i32(bt)
        T = int(cu_q[-1])
        assert x.shape == (T, dims.hidden)
        cd = dims.c()
        tp = None
        out = {}
        if taps:
            Hq = dims.n_q * dims.d
            out = {"h1": np.empty((T, dims.hidden), self.real), "q": np.empty((T, Hq), self.real),
                   "attn": np.empty((T, Hq), self.real), "x1": np.empty((T, dims.hidden), self.real),
                   "a": np.empty((T, dims.ffn), self.real)}
            tp = _Taps(*[out[n].ctypes.data for n in ("h1", "q", "attn", "x1", "a")])
        inv = None if inv_freq is None else np.ascontiguousarray(inv_freq, dtype=np.float32)
        ws = {k: _u16(v) for k, v in w.items()}
        rc = self.lib.so_layer(C.byref(cd), _p(ws["ln1"]), _p(ws["wq"]), _p(ws["wk"]), _p(ws["wv"]),
                               _p(ws.get("q_norm")), _p(ws.get("k_norm")), _p(ws["wo"]), _p(ws["ln2"]),
                               _p(ws["w_gate"]), _p(ws["w_up"]), _p(ws["w_down"]), _p(kpool), _p(vpool),
                               C.c_int(len(ctx_before)), _p(cu_q), _p(ctx_before), _p(bt),
                               C.c_int(bt.shape[1]), _p(inv), _p(x), C.byref(tp) if tp is not None else None)
        if rc != 0:
            raise MemoryError("so_layer: allocation failed")
        return out

    def logits(self, dims: OracleDims, y, final_norm, lm_head):
        y = self._r(y)
        n = y.shape[0]
        logits = np.empty((n, dims.vocab), dtype=self.real)
        am = np.empty(n, dtype=np.int32)
        margin = np.empty(n, dtype=self.real)
        cd = dims.c()
        self.lib.so_logits(C.byref(cd), _p(y), _p(_u16(final_norm)), _p(_u16(lm_head)), C.c_int(n), _p(logits),
                           _p(am), _p(margin))
        return logits, am, margin

    def stage(self, dims: OracleDims, layers: list, kv_pool, cu_q, ctx_before, bt, x_in_bf16=None,
              token_ids=None, embed=None, inv_freq=None, taps: bool = False):
        """Whole stage.  ``kv_pool`` uint16 [L,2,pages,n_kv,16,d] modified in place.  Input: bf16 bits [T,H]
        or token ids + embed.  Returns (y [T,H] real, list of per-layer taps)."""
        if token_ids is not None:
            x = self.embed(embed, token_ids, dims.hidden)
        else:
            xb = _u16(x_in_bf16)
            x = (xb.astype(np.uint32) << 16).view(np.float32).astype(self.real)
        x = np.ascontiguousarray(x)
        all_taps = []
        for li, w in enumerate(layers):
            t = self.layer(dims, w, kv_pool[li, 0], kv_pool[li, 1], cu_q, ctx_before, bt, x, inv_freq, taps)
            if taps:
                t["out"] = x.copy()
            all_taps.append(t)
        return x, all_taps
