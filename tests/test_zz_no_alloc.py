"""ss_op_gemm_bf16_static (include/shuntstage.h): the op-level GEMM for callers that may not allocate device memory.
Its stream-K fix-up scratch is a fixed __device__ array inside the library, shared by every call.  Checked against the
existing path (ss_op_gemm_bf16 with caller-owned scratch) on two calls in a row, the second of a different shape so
that what the first left in the array matters.  Collected last on purpose (the suite runs with pytest -x); passes
alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

from paper_2606_18600_b200 import synth


def _operands(T, N, K, seed):
    g = torch.Generator().manual_seed(seed)
    return synth.randn_bf16((T, K), 1.0, g).cuda(), synth.randn_bf16((N, K), 0.05, g).cuda()


@pytest.mark.gpu
def test_static_scratch_gemm_matches_existing_path_on_two_calls_in_a_row():
    from paper_2606_18600_b200 import binding
    # decode shapes: every SM busy, each row tile cut across several CTAs (the fix-up slots and flags are all in use);
    # then a small ragged one that reuses a corner of the array the first call filled
    shapes = [(128, 8192, 8192), (37, 1000, 4104), (128, 8192, 8192)]
    outs = [torch.full((T, N), float("nan"), dtype=torch.float32, device="cuda") for T, N, _ in shapes]
    ops = [_operands(T, N, K, 5 + i) for i, (T, N, K) in enumerate(shapes)]
    # set-up call (the header asks for one outside any capture): the first use on a device looks up the array's address
    # and makes the driver load the library's modules, which is when the array itself takes its 16 MiB
    xs, ws = _operands(8, 128, 64, 1)
    binding.op_gemm_bf16_static(xs, ws, torch.empty((8, 128), dtype=torch.float32, device="cuda"))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # back to back on one stream, no synchronisation in between: the calls are ordered by the stream, not by the host
    for (x, w), out in zip(ops, outs):
        binding.op_gemm_bf16_static(x, w, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0  # the calls took no device memory
    for (T, N, K), (x, w), got in zip(shapes, ops, outs):
        want = binding.op_gemm_bf16(x, w)  # existing path: caller-owned scratch
        torch.cuda.synchronize()
        g, r = got.cpu().numpy(), want.cpu().numpy()
        assert np.isfinite(g).all()
        # the tolerance of test_op_gemm_vs_oracle ...
        assert np.abs(g - r).max() <= 2e-5 * np.abs(r).max() * np.sqrt(K / 64) + 1e-6
        # ... and, the kernel and the launch plan being the same, the same bits
        assert torch.equal(got, want)


@pytest.mark.gpu
def test_static_scratch_gemm_rejects_sizes_beyond_its_maximum():
    from paper_2606_18600_b200 import binding
    x, w = _operands(binding.OP_GEMM_STATIC_MAX_T + 1, 256, 512, 3)
    out = torch.zeros((x.shape[0], 256), dtype=torch.float32, device="cuda")
    with pytest.raises(binding.ShuntStageError) as ei:
        binding.op_gemm_bf16_static(x, w, out)
    assert ei.value.code == -3  # SS_ERR_CAPACITY
    assert b"SS_OP_GEMM_STATIC_MAX_T" in binding.load_library().ss_last_cuda_error()
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0  # refused, not clipped: nothing was launched


@pytest.mark.gpu
def test_static_scratch_gemm_can_be_captured_in_a_cuda_graph():
    """The use the entry point exists for: after one set-up call outside the capture, two calls are recorded into a CUDA
    graph (a memset node and a kernel node each, nothing allocated) and the replay gives the existing path's bits."""
    from paper_2606_18600_b200 import binding
    (x1, w1), (x2, w2) = _operands(64, 8192, 8192, 21), _operands(128, 5120, 8192, 22)
    o1 = torch.zeros((64, 8192), dtype=torch.float32, device="cuda")
    o2 = torch.zeros((128, 5120), dtype=torch.float32, device="cuda")
    xs, ws = _operands(8, 128, 64, 1)
    binding.op_gemm_bf16_static(xs, ws, torch.empty((8, 128), dtype=torch.float32, device="cuda"))  # set-up call
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        graph.capture_begin()
        binding.op_gemm_bf16_static(x1, w1, o1, stream=side)
        binding.op_gemm_bf16_static(x2, w2, o2, stream=side)
        graph.capture_end()
    torch.cuda.synchronize()
    assert float(o1.abs().max()) == 0.0 and float(o2.abs().max()) == 0.0  # captured, not run
    for _ in range(2):
        o1.fill_(float("nan"))
        o2.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(o1, binding.op_gemm_bf16(x1, w1)) and torch.equal(o2, binding.op_gemm_bf16(x2, w2))
