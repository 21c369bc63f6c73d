"""ctypes binding of libshuntplace.so (include/shuntplace.h): ShuntServe's performance estimator and partitioned model
placement optimizer (paper section 4).  Argument marshalling only."""
from __future__ import annotations

import ctypes as C

from . import build as _build

SP_MAX_STAGES = 64
EXPORTS = ["sp_stage_latency", "sp_max_batch", "sp_evaluate", "sp_optimize", "sp_wrr_create", "sp_wrr_destroy",
           "sp_wrr_next", "sp_wrr_set_weight"]


class sp_model(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("hidden", "hq", "hkv", "ffn", "vocab", "n_layers", "elem_bytes")]


class sp_instance(C.Structure):
    _fields_ = [("flops", C.c_double), ("mem_bw", C.c_double), ("mem_bytes", C.c_double), ("n_gpus", C.c_int32),
                ("alpha_intra", C.c_double), ("beta_intra", C.c_double), ("cost", C.c_double)]


class sp_opts(C.Structure):
    _fields_ = [("s_in", C.c_double), ("s_out", C.c_double), ("alpha_inter", C.c_double), ("beta_inter", C.c_double),
                ("act_bytes", C.c_double), ("gamma", C.c_double), ("slo", C.c_double), ("beam", C.c_int32),
                ("max_stages", C.c_int32), ("max_batch", C.c_int32)]


class sp_placement(C.Structure):
    _fields_ = [("n_stages", C.c_int32), ("inst", C.c_int32 * SP_MAX_STAGES), ("layers", C.c_int32 * SP_MAX_STAGES),
                ("batch", C.c_int32), ("prefill_s", C.c_double), ("decode_s", C.c_double), ("rps", C.c_double),
                ("cost", C.c_double), ("score", C.c_double)]


_LIB = None


def load_library() -> C.CDLL:
    global _LIB
    if _LIB is None:
        path = _build.build_placement()
        lib = C.CDLL(str(path))
        lib.sp_stage_latency.restype = C.c_double
        lib.sp_stage_latency.argtypes = [C.POINTER(sp_model), C.POINTER(sp_instance), C.POINTER(sp_opts), C.c_int,
                                         C.c_int, C.c_int, C.c_int, C.c_int]
        lib.sp_max_batch.argtypes = [C.POINTER(sp_model), C.POINTER(sp_instance), C.POINTER(sp_opts), C.c_int,
                                     C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        lib.sp_evaluate.argtypes = [C.POINTER(sp_model), C.POINTER(sp_instance), C.c_int, C.POINTER(sp_opts),
                                    C.POINTER(sp_placement)]
        lib.sp_optimize.argtypes = [C.POINTER(sp_model), C.POINTER(sp_instance), C.c_int, C.POINTER(C.c_int32),
                                    C.POINTER(sp_opts), C.POINTER(sp_placement)]
        lib.sp_wrr_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.POINTER(C.c_double)]
        lib.sp_wrr_destroy.argtypes = [C.c_void_p]
        lib.sp_wrr_next.argtypes = [C.c_void_p]
        lib.sp_wrr_set_weight.argtypes = [C.c_void_p, C.c_int, C.c_double]
        _LIB = lib
    return _LIB


def _types(types):
    arr = (sp_instance * len(types))(*types)
    return arr


def stage_latency(model, inst, opts, layers, B, phase, is_last, has_next) -> float:
    return load_library().sp_stage_latency(C.byref(model), C.byref(inst), C.byref(opts), layers, B, phase,
                                           int(is_last), int(has_next))


def evaluate(model, types, opts, inst_ids, layers) -> sp_placement:
    p = sp_placement()
    p.n_stages = len(inst_ids)
    for i, (t, l) in enumerate(zip(inst_ids, layers)):
        p.inst[i], p.layers[i] = t, l
    rc = load_library().sp_evaluate(C.byref(model), _types(types), len(types), C.byref(opts), C.byref(p))
    if rc != 0:
        raise ValueError("sp_evaluate: bad input")
    return p


def optimize(model, types, opts, avail=None):
    """returns (rc, sp_placement): rc 0 = found, 1 = nothing fits"""
    p = sp_placement()
    av = None if avail is None else (C.c_int32 * len(avail))(*avail)
    rc = load_library().sp_optimize(C.byref(model), _types(types), len(types), av, C.byref(opts), C.byref(p))
    if rc < 0:
        raise ValueError("sp_optimize: bad input")
    return rc, p


class Dispatcher:
    """sp_wrr_*: smooth weighted round-robin over pipelines, weights = their throughputs."""

    def __init__(self, weights):
        self.lib = load_library()
        self.h = C.c_void_p()
        arr = (C.c_double * max(len(weights), 1))(*[float(w) for w in weights])
        if self.lib.sp_wrr_create(C.byref(self.h), len(weights), arr) != 0:
            raise ValueError("sp_wrr_create: bad input")

    def next(self) -> int:
        return self.lib.sp_wrr_next(self.h)

    def set_weight(self, i: int, w: float) -> None:
        if self.lib.sp_wrr_set_weight(self.h, i, float(w)) != 0:
            raise ValueError("sp_wrr_set_weight: bad input")

    def close(self) -> None:
        if self.h:
            self.lib.sp_wrr_destroy(self.h)
            self.h = C.c_void_p()
