"""ringx_attn_fwd_static: the forward for callers that cannot allocate device memory.

Who that is: code that runs inside a process whose allocator already owns the whole GPU (a cudaMalloc there fails),
a thread that has to launch work while another thread captures a CUDA graph in global mode (cudaMalloc is forbidden
there), a latency-bound loop that cannot take the device-wide synchronisation of cudaMalloc / cudaFree, or a small C or
Fortran driver with inputs and outputs but no workspace management.  For them the scratch of the KV-chunk passes is a
fixed 32 MiB array inside libringx, and the entry point takes inputs and outputs only.

What is checked here: on two calls in a row (different shapes, so the second one finds the first one's leftovers in the
shared array) the results agree with ringx_attn_fwd on a caller-allocated workspace within the tolerances of
tests/test_gpu_parity.py, and with the fp64 oracle; a repeat of the same calls does not lower the free device memory;
a problem beyond the 32 MiB limit is refused with RINGX_ERR_WORKSPACE_TOO_SMALL and the outputs untouched.

The file name sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides no other test.
"""
import ctypes
import math

import numpy as np
import pytest
import torch

from oracle import attention as orc
from paper_2507_16697_b200 import workloads as wl

# tests/test_gpu_parity.py's bars (BASELINE.json north_star + the scale-free one)
TOL_BF16_O_REL_V = 1e-2
TOL_BF16_O_RELF = 1e-2
TOL_LSE = 1e-3
RINGX_ERR_WORKSPACE_TOO_SMALL = 5


@pytest.fixture(scope="module")
def rx():
    from paper_2507_16697_b200 import ringx
    from paper_2507_16697_b200.build import build_library
    build_library()
    ringx.lib()
    return ringx


def test_limit_is_refused_before_any_cuda_call(rx):
    """Host-only: C3's shape needs a 1 GiB accumulator, far beyond the 32 MiB array; the refusal comes from the size check,
    which runs before the library touches the device (so this passes on a box without a GPU), and nothing is dereferenced."""
    L = rx.lib()
    fake = ctypes.c_void_p(4096)      # non-null, aligned, never read: the call is refused first
    assert L.ringx_attn_fwd_workspace_bytes(1, 8, 262144, 128, 32768, rx.RINGX_BF16) > rx.RINGX_STATIC_SCRATCH_BYTES
    st = L.ringx_attn_fwd_static(fake, fake, fake, fake, fake, 1, 8, 262144, 128, 32768, 128 ** -0.5, rx.RINGX_BF16, None)
    assert st == RINGX_ERR_WORKSPACE_TOO_SMALL
    assert L.ringx_attn_fwd_static(None, fake, fake, fake, fake, 1, 1, 256, 64, 128, 0.125, rx.RINGX_BF16, None) == 1


def _agree(o_s, lse_s, o_e, lse_e, o_ref, lse_ref, v64):
    """static entry vs existing entry, and each against the oracle, at test_gpu_parity.py's tolerances"""
    os_, oe = o_s.float().cpu().double().numpy(), o_e.float().cpu().double().numpy()
    ls, le = lse_s.cpu().double().numpy(), lse_e.cpu().double().numpy()
    assert np.isfinite(os_).all() and np.isfinite(ls).all()
    vmax = np.abs(v64).max()
    assert np.abs(os_ - oe).max() <= TOL_BF16_O_REL_V * vmax
    assert np.linalg.norm(os_ - oe) <= TOL_BF16_O_RELF * np.linalg.norm(oe)
    assert np.abs(ls - le).max() <= TOL_LSE
    assert np.abs(os_ - o_ref).max() <= TOL_BF16_O_REL_V * vmax
    assert np.linalg.norm(os_ - o_ref) <= TOL_BF16_O_RELF * np.linalg.norm(o_ref)
    assert np.abs(ls - lse_ref).max() <= TOL_LSE


# B, H, N, d, kv_chunk: the first fills 4.2 MB of the array over 4 passes; the second (ragged length, other head width,
# 4 passes with a short last one) then runs on top of what the first left there
CALLS = [(1, 2, 2048, 128, 512), (2, 2, 1000, 64, 256)]


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_workspace_path_and_allocate_nothing(rx):
    assert torch.cuda.is_available(), "GPU tests need a B200"
    cases = []
    for i, (B, H, N, d, chunk) in enumerate(CALLS):
        q, k, v = (wl.make_tensor((B, H, N, d), w, seed=41 + i, dtype="bf16") for w in "qkv")
        scale = 1.0 / math.sqrt(d)
        assert 0 < rx.ringx_attn_fwd_workspace_bytes(B, H, N, d, chunk, torch.bfloat16) <= rx.RINGX_STATIC_SCRATCH_BYTES
        o_ref, lse_ref = orc.attention_fwd_bhnd(wl.to_f64_numpy(q), wl.to_f64_numpy(k), wl.to_f64_numpy(v), scale)
        qc, kc, vc = q.cuda(), k.cuda(), v.cuda()
        o_e, lse_e = rx.ringx_attn_fwd(qc, kc, vc, chunk, scale)          # the existing path, caller-allocated workspace
        o_s = torch.full_like(qc, 7.0)                                      # outputs are the caller's, allocated up front
        lse_s = torch.full((B, H, N), 7.0, dtype=torch.float32, device="cuda")
        cases.append((qc, kc, vc, chunk, scale, o_s, lse_s, o_e, lse_e, o_ref, lse_ref, wl.to_f64_numpy(v)))
    torch.cuda.synchronize()

    # the two calls, back to back on one stream (calls that share the array must not overlap)
    for qc, kc, vc, chunk, scale, o_s, lse_s, *_ in cases:
        rx.ringx_attn_fwd_static(qc, kc, vc, chunk, scale, o=o_s, lse=lse_s)
    torch.cuda.synchronize()
    for qc, kc, vc, chunk, scale, o_s, lse_s, o_e, lse_e, o_ref, lse_ref, v64 in cases:
        _agree(o_s, lse_s, o_e, lse_e, o_ref, lse_ref, v64)

    # the same two calls again (every module and kernel is loaded by now): the free device memory must not drop
    free_before, _ = torch.cuda.mem_get_info()
    for qc, kc, vc, chunk, scale, o_s, lse_s, *_ in cases:
        o_s.fill_(7.0)
        lse_s.fill_(7.0)
        rx.ringx_attn_fwd_static(qc, kc, vc, chunk, scale, o=o_s, lse=lse_s)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, (free_before, free_after)
    for qc, kc, vc, chunk, scale, o_s, lse_s, o_e, lse_e, o_ref, lse_ref, v64 in cases:
        _agree(o_s, lse_s, o_e, lse_e, o_ref, lse_ref, v64)

    # beyond the limit: refused before anything is enqueued, outputs untouched
    B, H, N, d = 1, 8, 8192, 128
    big = torch.zeros((B, H, N, d), dtype=torch.bfloat16, device="cuda")
    o_big = torch.full_like(big, 7.0)
    lse_big = torch.full((B, H, N), 7.0, dtype=torch.float32, device="cuda")
    assert rx.ringx_attn_fwd_workspace_bytes(B, H, N, d, 1024, torch.bfloat16) > rx.RINGX_STATIC_SCRATCH_BYTES
    with pytest.raises(rx.RingxError) as ei:
        rx.ringx_attn_fwd_static(big, big, big, 1024, d ** -0.5, o=o_big, lse=lse_big)
    assert ei.value.status == RINGX_ERR_WORKSPACE_TOO_SMALL
    torch.cuda.synchronize()
    assert (o_big == 7.0).all() and (lse_big == 7.0).all()
