"""fcp_attn_bwd_static (include/fcp.h section 4): the backward on the library's own static device
workspace, for callers that cannot call cudaMalloc, against the existing fcp_attn_bwd on a
caller-provided workspace.  Both run the same kernels on the same schedule, so dk / dv (fixed
summation order) must be bit-identical and dq (L2 reductions, order varies) within the tolerances
of the parity tests.  Several calls in a row, on different shapes, share the one workspace: each
must be independent of what the previous one left there.

This file is collected last on purpose (the run uses `pytest -x`)."""
import math

import numpy as np
import pytest

import fcp_inputs
import gpu_util as U

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


# d, N, rank, Hq, Hkv, D, dk / dv in fp32
CALLS = [
    ([700, 500, 400, 192], 2, 0, 4, 2, 128, False),
    ([1000, 37, 1, 1, 1, 260, 100], 4, 1, 6, 2, 64, True),     # smaller, other kernel variant
    ([700, 500, 400, 192], 2, 0, 4, 2, 128, False),            # the first one again
    ([129, 127, 65, 63], 1, 0, 4, 1, 128, True),
]


def _existing_path(fcp, torch, d, N, r, Hq, Hkv, D, dkv_f32, seed):
    Q, K, V, dO = fcp_inputs.make_tensors(sum(d), Hq, Hkv, D, seed, device="cuda")
    plan = fcp.Plan(d, N)
    g = U.run_rank_gpu(fcp, plan, r, Q, K, V, dO, 1.0 / math.sqrt(D), dkv_f32=dkv_f32)
    return plan, g


def test_static_workspace_backward_matches_existing_path(fcp, torch):
    for i, (d, N, r, Hq, Hkv, D, dkv_f32) in enumerate(CALLS):
        scale = 1.0 / math.sqrt(D)
        plan, g = _existing_path(fcp, torch, d, N, r, Hq, Hkv, D, dkv_f32, seed=20 + i)
        # a schedule of its own that was never uploaded: the entry point brings its lists itself
        sched = plan.sched(r, Hq, Hkv, D)
        assert sched.workspace is None and sched.workspace_size() <= fcp.STATIC_WORKSPACE_BYTES
        # outputs are the caller's; pre-filled so that an unwritten element shows
        dq = torch.full_like(g["dq"], float("nan"))
        dk = torch.full_like(g["dk"], float("nan"))
        dv = torch.full_like(g["dv"], float("nan"))
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        held_before = torch.cuda.memory_allocated()
        sched.attn_bwd_static(g["q"], g["k"], g["v"], g["o"], g["lse"], g["do"], scale, dq, dk, dv)
        torch.cuda.synchronize()
        assert sched.workspace is None
        assert torch.cuda.memory_allocated() == held_before
        if i >= 2:          # every kernel variant of this call has been loaded by an earlier one
            assert torch.cuda.mem_get_info()[0] >= free_before, "the call took device memory"
        tag = "call %d" % i
        assert torch.equal(dk, g["dk"]), tag + ": dk differs from fcp_attn_bwd"
        assert torch.equal(dv, g["dv"]), tag + ": dv differs from fcp_attn_bwd"
        U.check(tag + " dq", U.to_f64(dq), U.to_f64(g["dq"]))
        ref = g["dq"].float()
        assert float((dq.float() - ref).abs().max()) <= 2e-3 * max(1.0, float(ref.abs().max()))


def test_static_workspace_rejects_what_does_not_fit(fcp, torch):
    Hq, Hkv, D, n = 8, 2, 128, 20000              # fp32 dq accumulator alone: 82 MB > 32 MiB
    sched = fcp.Sched.create([0, n], [0], [0], [0, n], Hq, Hkv, D)
    assert sched.workspace_size() > fcp.STATIC_WORKSPACE_BYTES
    q = torch.zeros((n, Hq, D), dtype=torch.bfloat16, device="cuda")
    k = torch.zeros((n, Hkv, D), dtype=torch.bfloat16, device="cuda")
    lse = torch.zeros((Hq, n), dtype=torch.float32, device="cuda")
    dq, dk, dv = torch.ones_like(q), torch.ones_like(k), torch.ones_like(k)
    with pytest.raises(fcp.FcpError) as e:
        sched.attn_bwd_static(q, k, k, q, lse, q, 1.0, dq, dk, dv)
    assert e.value.status == fcp.TOO_LARGE and "FCP_STATIC_WORKSPACE_BYTES" in str(e.value)
    torch.cuda.synchronize()
    assert bool((dq == 1).all()) and bool((dk == 1).all()) and bool((dv == 1).all())   # untouched


def test_static_workspace_wants_no_caller_workspace(fcp, torch):
    """args->workspace must be NULL: a caller that has a workspace uses fcp_attn_bwd."""
    import ctypes as C
    from paper_2606_08476_b200 import binding as B
    sched = fcp.Sched.create([0, 64], [0], [0], [0, 64], 2, 1, 64)
    t = torch.zeros((64, 2, 64), dtype=torch.bfloat16, device="cuda")
    a = B._AttnArgs(sched._h, t.data_ptr(), t.data_ptr(), t.data_ptr(), t.data_ptr(), t.data_ptr(),
                    t.data_ptr(), 1.0, 0, None, None, None, None, 0)
    st = B._lib().fcp_attn_bwd_static(C.byref(a), t.data_ptr(), t.data_ptr(), t.data_ptr(),
                                      t.data_ptr())
    assert st == -1       # FCP_INVALID_ARG
