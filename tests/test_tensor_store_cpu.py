"""Host-side logic of the Shared Tensor Store: arena layout and the raw binary shard format.
No GPU: the ss_store_* calls are only probed for their argument checks."""
import ctypes as C
import json

import numpy as np
import pytest
import torch

from paper_2606_18600_b200 import binding, synth, tensor_store as ts


def test_layout_is_aligned_ordered_and_disjoint():
    L = synth.TINY.n_layers
    layers = [synth.layer_weights(synth.TINY, l, 0) for l in range(L)]
    ent = ts.stage_entries(layers, synth.edge_weights(synth.TINY, 0), 12345)
    lay, total = ts.plan_layout(ent)
    assert list(lay)[-1] == "kv_pool" and lay["kv_pool"]["bytes"] == 2 * 12345
    end = 0
    for name, m in lay.items():
        assert m["offset"] % ts.ALIGN == 0 and m["offset"] >= end, name
        assert m["offset"] - end < ts.ALIGN          # no gap beyond the alignment padding
        end = m["offset"] + m["bytes"]
    assert total == end
    w = layers[0]["wq"]
    assert lay["layers.0.wq"]["bytes"] == w.numel() * 2 and lay["layers.0.wq"]["shape"] == list(w.shape)
    # Llama-style layers have no QK-norm gains: absent tensors get no slot
    assert "layers.0.q_norm" not in lay and "layers.1.w_down" in lay
    json.dumps(lay)                                   # the manifest must be JSON-serialisable
    with pytest.raises(ValueError):
        ts.plan_layout({"x": ("float64", (4,))})


def test_raw_shards_hold_only_the_partition_bytes(tmp_path):
    """torch.save of a slice keeps the parent's storage; the raw format stores the slice alone."""
    full = synth.randn_bf16((64, 256), 0.02, torch.Generator().manual_seed(1))
    part = full[16:32]                                # a row partition, as TP / layer sharding produces
    idx = torch.arange(10, dtype=torch.int32)
    ts.save_shards(tmp_path, {"w.part": part, "idx": idx, "empty": torch.empty(0, dtype=torch.float32)})
    assert (tmp_path / "w.part.bin").stat().st_size == 16 * 256 * 2
    assert (tmp_path / "idx.bin").stat().st_size == 40 and (tmp_path / "empty.bin").stat().st_size == 0
    back = ts.load_shards(tmp_path)
    assert back["w.part"].dtype == torch.bfloat16 and torch.equal(back["w.part"], part)
    assert torch.equal(back["idx"], idx) and back["empty"].numel() == 0
    only = ts.load_shards(tmp_path, ["idx"])
    assert list(only) == ["idx"]
    # the file is the tensor's bytes and nothing else
    raw = np.fromfile(tmp_path / "w.part.bin", dtype=np.uint16)
    assert np.array_equal(raw, synth.bits(part.contiguous()).reshape(-1))
    (tmp_path / "idx.bin").write_bytes(b"\0" * 39)
    with pytest.raises(IOError):
        ts.load_shards(tmp_path, ["idx"])


def test_store_calls_reject_null_arguments_before_touching_cuda():
    lib = binding.load_library()
    p = C.c_void_p()
    h = (C.c_ubyte * 64)()
    assert lib.ss_store_alloc(None, 16) == -1 and lib.ss_store_alloc(C.byref(p), 0) == -1
    assert lib.ss_store_free(None) == -1 and lib.ss_store_detach(None) == -1
    assert lib.ss_store_export(None, h) == -1 and lib.ss_store_export(1024, None) == -1
    assert lib.ss_store_attach(None, C.byref(p)) == -1 and lib.ss_store_attach(h, None) == -1
    assert lib.ss_store_upload(None, h, 4) == -1 and lib.ss_store_upload(1024, None, 4) == -1
