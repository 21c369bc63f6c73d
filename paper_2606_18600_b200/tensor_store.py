"""Shared Tensor Store: weights and KV-cache space owned by one process, attached zero-copy by engine processes.

PAPER.md:271-275 (Section 5.2, Figure 7): ShuntServe keeps "model weight tensors and KV cache space" in a separate
per-node process and shares them with the inference engine "through CUDA IPC handles", so that a replacement engine can
be initialised beside the serving one without a second copy of either ("concurrent initialization").  PAPER.md:283:
weights travel as "individual binary files in a custom raw binary format" that hold "only the actual partition data".

This module is the thin Python side of `ss_store_*` (include/shuntstage.h): it lays tensors out in ONE device arena,
publishes a JSON-serialisable manifest {handle, bytes, tensors: name -> dtype/shape/offset}, and on the engine side maps
the arena and hands out torch views that `binding.Stage` borrows (weights, KV pool).  No arithmetic lives here.

    store process                         engine process (any number, coexisting)
    -------------                         ---------------------------------------
    st = TensorStore(layout)              att = attach(manifest)
    st.put(name, cpu_tensor) ...          layers, edge, kv = stage_tensors(att, L)
    send(st.manifest())                   stage = binding.Stage(dims, l0, l1, layers, edge, kv_pool=kv)
    ... keep alive ...                    ... stage.destroy(); att.close()
    st.close()
"""
from __future__ import annotations

import ctypes as C
import json
from pathlib import Path

import numpy as np
import torch

from . import binding

ALIGN = 256  # every tensor starts on a 256-byte boundary of the arena (TMA needs 16; the GEMM scratch 256)
_DTYPES = {"bfloat16": torch.bfloat16, "float32": torch.float32, "int32": torch.int32, "uint8": torch.uint8}
_LAYER_NAMES = [n for n, _ in binding.ss_layer_weights._fields_]
_EDGE_NAMES = ["embed", "final_norm", "lm_head"]


def _nbytes(dtype: str, shape) -> int:
    return int(np.prod(shape, dtype=np.int64)) * torch.empty((), dtype=_DTYPES[dtype]).element_size()


def plan_layout(entries: dict) -> tuple[dict, int]:
    """entries: name -> (dtype name, shape).  Returns ({name: {dtype, shape, offset, bytes}}, arena bytes): tensors in
    insertion order, each offset rounded up to ALIGN.  Pure host arithmetic (CPU-testable)."""
    out, off = {}, 0
    for name, (dtype, shape) in entries.items():
        if dtype not in _DTYPES:
            raise ValueError(f"{name}: unsupported dtype {dtype}")
        off = (off + ALIGN - 1) // ALIGN * ALIGN
        nb = _nbytes(dtype, shape)
        out[name] = {"dtype": dtype, "shape": [int(s) for s in shape], "offset": off, "bytes": nb}
        off += nb
    return out, max(off, ALIGN)


def _dtype_name(t: torch.Tensor) -> str:
    return str(t.dtype).replace("torch.", "")


def stage_entries(layers: list, edge: dict | None, kv_pool_elems: int) -> dict:
    """Layout entries of a stage: 'layers.<i>.<name>' for every present weight, the edge tensors, then 'kv_pool'."""
    ent = {}
    for i, w in enumerate(layers):
        for n in _LAYER_NAMES:
            if w.get(n) is not None:
                ent[f"layers.{i}.{n}"] = (_dtype_name(w[n]), tuple(w[n].shape))
    for n in _EDGE_NAMES:
        if edge and edge.get(n) is not None:
            ent[n] = (_dtype_name(edge[n]), tuple(edge[n].shape))
    ent["kv_pool"] = ("bfloat16", (int(kv_pool_elems),))
    return ent


# ---- raw binary shards: one file per tensor holding exactly the partition's bytes + a manifest ----
def save_shards(directory, tensors: dict) -> None:
    d = Path(directory)
    d.mkdir(parents=True, exist_ok=True)
    meta = {}
    for name, t in tensors.items():
        t = t.detach().cpu().contiguous()  # a slice is stored as its own bytes, not as its parent storage
        raw = t.view(torch.uint8).numpy() if t.numel() else np.zeros(0, np.uint8)
        raw.tofile(d / (name + ".bin"))
        meta[name] = {"dtype": _dtype_name(t), "shape": list(t.shape), "bytes": int(raw.size)}
    (d / "manifest.json").write_text(json.dumps(meta, indent=1))


def load_shards(directory, names=None) -> dict:
    """Read the named tensors (default: all) back as CPU tensors; only the requested files are touched."""
    d = Path(directory)
    meta = json.loads((d / "manifest.json").read_text())
    out = {}
    for name in (names if names is not None else meta):
        m = meta[name]
        raw = np.fromfile(d / (name + ".bin"), dtype=np.uint8)
        if raw.size != m["bytes"]:
            raise IOError(f"{name}: {raw.size} bytes on disk, manifest says {m['bytes']}")
        if raw.size == 0:
            out[name] = torch.empty(m["shape"], dtype=_DTYPES[m["dtype"]])
            continue
        out[name] = torch.from_numpy(raw).view(_DTYPES[m["dtype"]]).view(m["shape"])
    return out


# ---- device side -----------------------------------------------------------------------------------------------
class _Arena:
    """Exposes a raw device range to torch through __cuda_array_interface__ (zero-copy view, no ownership)."""

    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def _views(base_ptr: int, nbytes: int, tensors: dict, device) -> tuple[torch.Tensor, dict]:
    arena = torch.as_tensor(_Arena(base_ptr, nbytes), device=device)
    assert arena.data_ptr() == base_ptr, "torch copied the arena instead of viewing it"
    out = {}
    for name, m in tensors.items():
        out[name] = arena[m["offset"]:m["offset"] + m["bytes"]].view(_DTYPES[m["dtype"]]).view(m["shape"])
    return arena, out


def _check(rc: int, where: str) -> None:
    if rc != binding.SS_OK:
        raise binding.ShuntStageError(rc, where)


class TensorStore:
    """Owner side: one cudaMalloc arena laid out by plan_layout(); lives in the store process."""

    def __init__(self, entries: dict, device="cuda:0"):
        if not torch.cuda.is_available():
            raise RuntimeError("the tensor store needs a CUDA device; there is no CPU path")
        self.lib = binding.load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        torch.cuda.init()
        self.layout, self.nbytes = plan_layout(entries)
        p = C.c_void_p()
        _check(self.lib.ss_store_alloc(C.byref(p), self.nbytes), "ss_store_alloc")
        self.ptr = p.value
        self._arena, self.tensors = _views(self.ptr, self.nbytes, self.layout, self.device)

    def put(self, name: str, t: torch.Tensor) -> None:
        """Upload a CPU tensor's bytes into its slot (shape and dtype must match the layout)."""
        m = self.layout[name]
        t = t.detach().cpu().contiguous()
        if _dtype_name(t) != m["dtype"] or list(t.shape) != m["shape"]:
            raise ValueError(f"{name}: got {_dtype_name(t)}{list(t.shape)}, layout has {m['dtype']}{m['shape']}")
        _check(self.lib.ss_store_upload(self.ptr + m["offset"], t.data_ptr(), m["bytes"]), "ss_store_upload")

    def manifest(self) -> dict:
        h = (C.c_ubyte * 64)()
        _check(self.lib.ss_store_export(self.ptr, h), "ss_store_export")
        return {"handle": bytes(h).hex(), "bytes": self.nbytes, "device": self.device.index or 0,
                "tensors": self.layout}

    def close(self) -> None:
        if self.ptr:
            self.tensors, self._arena = {}, None
            torch.cuda.synchronize(self.device)
            _check(self.lib.ss_store_free(self.ptr), "ss_store_free")
            self.ptr = None


class Attachment:
    """Engine side: the store's arena mapped into this process; `.tensors[name]` are borrowed views."""

    def __init__(self, manifest: dict):
        if not torch.cuda.is_available():
            raise RuntimeError("attaching to a tensor store needs a CUDA device; there is no CPU path")
        self.lib = binding.load_library()
        self.device = torch.device(f"cuda:{manifest['device']}")
        torch.cuda.set_device(self.device)
        torch.cuda.init()
        h = (C.c_ubyte * 64).from_buffer_copy(bytes.fromhex(manifest["handle"]))
        p = C.c_void_p()
        _check(self.lib.ss_store_attach(h, C.byref(p)), "ss_store_attach")
        self.ptr, self.nbytes = p.value, manifest["bytes"]
        self._arena, self.tensors = _views(self.ptr, self.nbytes, manifest["tensors"], self.device)

    def close(self) -> None:
        if self.ptr:
            self.tensors, self._arena = {}, None
            torch.cuda.synchronize(self.device)
            _check(self.lib.ss_store_detach(self.ptr), "ss_store_detach")
            self.ptr = None


def attach(manifest: dict) -> Attachment:
    return Attachment(manifest)


def stage_tensors(att, n_layers: int) -> tuple[list, dict | None, torch.Tensor]:
    """(layers, edge, kv_pool) in the form binding.Stage takes, out of a store's or an attachment's `.tensors`."""
    t = att.tensors
    layers = [{n: t.get(f"layers.{i}.{n}") for n in _LAYER_NAMES} for i in range(n_layers)]
    edge = {n: t[n] for n in _EDGE_NAMES if n in t} or None
    return layers, edge, t["kv_pool"]
