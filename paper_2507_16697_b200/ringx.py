"""Thin ctypes binding over libringx.so -- same names as include/ringx.h, argument marshalling only.

Every step of the path runs in the library's CUDA kernels; this file allocates outputs/workspace with
torch (device memory and streams are what PyTorch is used for here) and passes raw pointers.  There
is no CPU fallback: a missing library or a non-CUDA tensor raises.
"""
from __future__ import annotations

import ctypes
import os

import torch

from .build import LIB_PATH

RINGX_F32, RINGX_BF16 = 0, 1
_DTYPES = {torch.float32: RINGX_F32, torch.bfloat16: RINGX_BF16}
_lib = None


class RingxError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().ringx_status_string(status).decode()
        super().__init__(f"{where}: {msg} (ringx_status {status})")


def lib() -> ctypes.CDLL:
    """Load libringx.so (built in-tree by `python -m paper_2507_16697_b200.build`).  Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2507_16697_b200.build` "
            "(there is no CPU or PyTorch fallback for the RingX hot path)")
    L = ctypes.CDLL(LIB_PATH)
    c_p, c_i, c_f, c_sz, c_ll = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_size_t, ctypes.c_longlong
    L.ringx_attn_fwd.argtypes = [c_p] * 5 + [c_i] * 5 + [c_f, c_i, c_p, c_sz, c_p]
    L.ringx_attn_fwd.restype = c_i
    L.ringx_attn_fwd_static.argtypes = [c_p] * 5 + [c_i] * 5 + [c_f, c_i, c_p]
    L.ringx_attn_fwd_static.restype = c_i
    L.ringx_attn_fwd_host.argtypes = [c_p] * 5 + [c_i] * 5 + [c_f, c_i, c_p, c_sz, c_p]
    L.ringx_attn_fwd_host.restype = c_i
    L.ringx_attn_bwd.argtypes = [c_p] * 9 + [c_i] * 5 + [c_f, c_i, c_p, c_sz, c_p]
    L.ringx_attn_bwd.restype = c_i
    L.ringx_attn_fwd_mla.argtypes = [c_p] * 5 + [c_i] * 6 + [c_f, c_i, c_p, c_sz, c_p]
    L.ringx_attn_fwd_mla.restype = c_i
    L.ringx_attn_fwd_mla_workspace_bytes.argtypes = [c_i] * 6
    L.ringx_attn_fwd_mla_workspace_bytes.restype = c_sz
    L.ringx_attn_bwd_mla.argtypes = [c_p] * 9 + [c_i] * 6 + [c_f, c_i, c_p, c_sz, c_p]
    L.ringx_attn_bwd_mla.restype = c_i
    L.ringx_attn_bwd_mla_workspace_bytes.argtypes = [c_i] * 6
    L.ringx_attn_bwd_mla_workspace_bytes.restype = c_sz
    L.ringx_attn_chunk_fwd_mla.argtypes = [c_p] * 7 + [c_i] * 6 + [c_f, c_i, c_i, c_p]
    L.ringx_attn_chunk_fwd_mla.restype = c_i
    L.ringx_attn_bwd_partial_mla.argtypes = [c_p] * 9 + [c_i] * 6 + [c_f, c_i, c_i, c_i, c_p, c_sz, c_p]
    L.ringx_attn_bwd_partial_mla.restype = c_i
    L.ringx_attn_bwd_partial_mla_workspace_bytes.argtypes = [c_i] * 3
    L.ringx_attn_bwd_partial_mla_workspace_bytes.restype = c_sz
    L.ringx_dq_finalize_mla.argtypes = [c_p, c_p, c_i, c_i, c_i, c_i, c_p]
    L.ringx_dq_finalize_mla.restype = c_i
    L.ringx_lse_merge.argtypes = [c_p] * 6 + [c_ll, c_i, c_i, c_i, c_p]
    L.ringx_lse_merge.restype = c_i
    L.ringx_attn_chunk_fwd.argtypes = [c_p] * 5 + [c_i] * 5 + [c_f, c_i, c_p]
    L.ringx_attn_chunk_fwd.restype = c_i
    L.ringx_attn_fwd_bwd_host.argtypes = [c_p] * 9 + [c_i] * 5 + [c_f, c_i, c_p, c_sz, c_p]
    L.ringx_attn_fwd_bwd_host.restype = c_i
    L.ringx_attn_chunk_fwd_fold.argtypes = [c_p] * 7 + [c_i] * 5 + [c_f, c_i, c_p]
    L.ringx_attn_chunk_fwd_fold.restype = c_i
    L.ringx_attn_chunk_fwd_ex.argtypes = [c_p] * 7 + [c_i] * 5 + [c_f, c_i, c_i, c_p, c_sz, c_p]
    L.ringx_attn_chunk_fwd_ex.restype = c_i
    L.ringx_attn_chunk_fwd_ex_workspace_bytes.argtypes = [c_i] * 6
    L.ringx_attn_chunk_fwd_ex_workspace_bytes.restype = c_sz
    L.ringx_attn_fwd_gqa.argtypes = [c_p] * 5 + [c_i] * 6 + [c_f, c_i, c_p, c_sz, c_p]
    L.ringx_attn_fwd_gqa.restype = c_i
    L.ringx_attn_bwd_gqa.argtypes = [c_p] * 9 + [c_i] * 6 + [c_f, c_i, c_p, c_sz, c_p]
    L.ringx_attn_bwd_gqa.restype = c_i
    L.ringx_attn_bwd_partial.argtypes = [c_p] * 9 + [c_i] * 5 + [c_f, c_i, c_p, c_sz, c_p]
    L.ringx_attn_bwd_partial.restype = c_i
    L.ringx_attn_bwd_partial_ex.argtypes = [c_p] * 9 + [c_i] * 5 + [c_f, c_i, c_i, c_i, c_p, c_sz, c_p]
    L.ringx_attn_bwd_partial_ex.restype = c_i
    L.ringx_attn_bwd_partial_workspace_bytes.argtypes = [c_i] * 4
    L.ringx_attn_bwd_partial_workspace_bytes.restype = c_sz
    L.ringx_dq_finalize.argtypes = [c_p, c_p, c_ll, c_p]
    L.ringx_dq_finalize.restype = c_i
    L.ringx_eq5_scale.argtypes = [c_p] * 5 + [c_ll, c_i, c_p]
    L.ringx_eq5_scale.restype = c_i
    L.ringx_eq5_finalize.argtypes = [c_p] * 5 + [c_ll, c_i, c_i, c_p]
    L.ringx_eq5_finalize.restype = c_i
    L.ringx_out_proj_bwd.argtypes = [c_p] * 5 + [c_i] * 4 + [c_p]
    L.ringx_out_proj_bwd.restype = c_i
    L.ringx_qkv_proj_bwd.argtypes = [c_p] * 7 + [c_i] * 4 + [c_p]
    L.ringx_qkv_proj_bwd.restype = c_i
    L.ringx_attn_block_bwd.argtypes = [c_p] * 8 + [c_i] * 5 + [c_f, c_p, c_sz, c_p]
    L.ringx_attn_block_bwd.restype = c_i
    L.ringx_attn_block_bwd_workspace_bytes.argtypes = [c_i] * 5
    L.ringx_attn_block_bwd_workspace_bytes.restype = c_sz
    L.ringx_fidelity_tokens.argtypes = [c_p, c_p] + [c_i] * 12 + [c_f, c_i, c_p]
    L.ringx_fidelity_tokens.restype = c_i
    L.ringx_qkv_proj.argtypes = [c_p] * 5 + [c_i] * 4 + [c_p]
    L.ringx_qkv_proj.restype = c_i
    L.ringx_out_proj.argtypes = [c_p] * 3 + [c_i] * 4 + [c_p]
    L.ringx_out_proj.restype = c_i
    L.ringx_attn_block_fwd.argtypes = [c_p] * 4 + [c_i] * 5 + [c_f, c_p, c_sz, c_p]
    L.ringx_attn_block_fwd.restype = c_i
    L.ringx_attn_block_fwd_workspace_bytes.argtypes = [c_i] * 5
    L.ringx_attn_block_fwd_workspace_bytes.restype = c_sz
    for name in ("ringx_attn_fwd_workspace_bytes", "ringx_attn_bwd_workspace_bytes",
                 "ringx_attn_fwd_host_workspace_bytes", "ringx_attn_fwd_bwd_host_workspace_bytes"):
        getattr(L, name).argtypes = [c_i] * 6
        getattr(L, name).restype = c_sz
    L.ringx_set_deterministic.argtypes = [c_i]
    L.ringx_set_deterministic.restype = c_i
    L.ringx_get_deterministic.argtypes = []
    L.ringx_get_deterministic.restype = c_i
    L.ringx_last_launch_count.argtypes = []
    L.ringx_last_launch_count.restype = c_i
    L.ringx_profile_enable.argtypes = [c_i]
    L.ringx_profile_enable.restype = c_i
    L.ringx_profile_read.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(c_i)]
    L.ringx_profile_read.restype = c_i
    L.ringx_status_string.argtypes = [c_i]
    L.ringx_status_string.restype = ctypes.c_char_p
    L.ringx_version.argtypes = []
    L.ringx_version.restype = c_i
    _lib = L
    return L


def _check(status: int, where: str):
    if status != 0:
        raise RingxError(status, where)


def _dev(t: torch.Tensor, name: str) -> int:
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous [B,H,N,d]")
    return t.data_ptr()


def _expect(t: torch.Tensor, shape, name: str, dtype=None):
    """The C ABI takes ONE set of sizes for all its tensors: a tensor of another shape would be read or written out of
    bounds, so the binding refuses it (argument marshalling, no arithmetic)."""
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name} has shape {tuple(t.shape)}, expected {tuple(shape)}")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"{name} has dtype {t.dtype}, expected {dtype}")


def _expect_workspace(workspace: torch.Tensor, need: int, name: str):
    if workspace.numel() * workspace.element_size() < need:
        raise ValueError(f"{name}: workspace holds {workspace.numel() * workspace.element_size()} bytes, "
                         f"the size query asks for {need}")


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _workspace(nbytes: int, device) -> torch.Tensor | None:
    return torch.empty(nbytes, dtype=torch.uint8, device=device) if nbytes else None


def ringx_attn_fwd_workspace_bytes(B, H, N, d, kv_chunk, dtype) -> int:
    return lib().ringx_attn_fwd_workspace_bytes(B, H, N, d, kv_chunk, _DTYPES[dtype])


def ringx_attn_bwd_workspace_bytes(B, H, N, d, kv_chunk, dtype) -> int:
    return lib().ringx_attn_bwd_workspace_bytes(B, H, N, d, kv_chunk, _DTYPES[dtype])


def ringx_attn_fwd_host_workspace_bytes(B, H, N, d, kv_chunk, dtype) -> int:
    return lib().ringx_attn_fwd_host_workspace_bytes(B, H, N, d, kv_chunk, _DTYPES[dtype])


def ringx_attn_fwd(q, k, v, kv_chunk: int, scale: float, o=None, lse=None, workspace=None):
    """O, LSE = chunked attention of q,k,v [B,H,N,d] (include/ringx.h: ringx_attn_fwd)."""
    B, H, N, d = q.shape
    dt = _DTYPES[q.dtype]
    if o is None:
        o = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((B, H, N), dtype=torch.float32, device=q.device)
    for t, nm in ((k, "k"), (v, "v"), (o, "o")):
        _expect(t, q.shape, nm, q.dtype)
    _expect(lse, (B, H, N), "lse", torch.float32)
    need = lib().ringx_attn_fwd_workspace_bytes(B, H, N, d, kv_chunk, dt)
    if workspace is None:
        workspace = _workspace(need, q.device)
    ws_ptr = workspace.data_ptr() if workspace is not None else None
    ws_len = workspace.numel() * workspace.element_size() if workspace is not None else 0
    st = lib().ringx_attn_fwd(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o, "o"), _dev(lse, "lse"),
                              B, H, N, d, kv_chunk, scale, dt, ws_ptr, ws_len, _stream())
    _check(st, "ringx_attn_fwd")
    return o, lse


RINGX_STATIC_SCRATCH_BYTES = 32 << 20     # include/ringx.h


def ringx_attn_fwd_static(q, k, v, kv_chunk: int, scale: float, o=None, lse=None):
    """ringx_attn_fwd for callers that cannot supply a device workspace (include/ringx.h: ringx_attn_fwd_static): the
    scratch of the chunk passes is a fixed 32 MiB array inside libringx, so the call allocates no device memory -- pass
    `o` and `lse` and this wrapper allocates nothing either (without them it creates the two outputs, nothing else).
    Problems whose ringx_attn_fwd workspace would exceed RINGX_STATIC_SCRATCH_BYTES raise RingxError
    (RINGX_ERR_WORKSPACE_TOO_SMALL).  All calls on one GPU share the array: do not let two of them overlap."""
    B, H, N, d = q.shape
    if o is None:
        o = torch.empty_like(q)
    if lse is None:
        lse = torch.empty((B, H, N), dtype=torch.float32, device=q.device)
    for t, nm in ((k, "k"), (v, "v"), (o, "o")):
        _expect(t, q.shape, nm, q.dtype)
    _expect(lse, (B, H, N), "lse", torch.float32)
    st = lib().ringx_attn_fwd_static(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o, "o"), _dev(lse, "lse"),
                                     B, H, N, d, kv_chunk, scale, _DTYPES[q.dtype], _stream())
    _check(st, "ringx_attn_fwd_static")
    return o, lse


def _check_mla_shapes(q, k, v, same_len=True):
    """q [B,H,Nq,192], k [B,H,Nk,192], v [B,H,Nk,128]: the C ABI takes one (B, H) for all three, so they must agree."""
    if q.dim() != 4 or k.dim() != 4 or v.dim() != 4 or q.shape[:2] != k.shape[:2] or k.shape[:3] != v.shape[:3] \
            or q.shape[3] != k.shape[3] or (same_len and q.shape[2] != k.shape[2]):
        raise ValueError(f"MLA shapes do not match: q {tuple(q.shape)}, k {tuple(k.shape)}, v {tuple(v.shape)}")


def ringx_attn_fwd_mla_workspace_bytes(B, H, N, d_qk, d_v, kv_chunk) -> int:
    return lib().ringx_attn_fwd_mla_workspace_bytes(B, H, N, d_qk, d_v, kv_chunk)


def ringx_attn_fwd_mla(q, k, v, kv_chunk: int, scale: float, o=None, lse=None, workspace=None):
    """O, LSE for multi-head latent attention shapes: q, k [B,H,N,192], v [B,H,N,128] bf16 (include/ringx.h:
    ringx_attn_fwd_mla)."""
    _check_mla_shapes(q, k, v)
    B, H, N, d_qk = q.shape
    d_v = v.shape[3]
    if o is None:
        o = torch.empty((B, H, N, d_v), dtype=q.dtype, device=q.device)
    if lse is None:
        lse = torch.empty((B, H, N), dtype=torch.float32, device=q.device)
    _expect(o, (B, H, N, d_v), "o", q.dtype)
    _expect(lse, (B, H, N), "lse", torch.float32)
    need = lib().ringx_attn_fwd_mla_workspace_bytes(B, H, N, d_qk, d_v, kv_chunk)
    if workspace is None:
        workspace = _workspace(need, q.device)
    st = lib().ringx_attn_fwd_mla(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o, "o"), _dev(lse, "lse"), B, H, N, d_qk, d_v,
                                  kv_chunk, scale, _DTYPES[q.dtype], workspace.data_ptr() if workspace is not None else None,
                                  workspace.numel() if workspace is not None else 0, _stream())
    _check(st, "ringx_attn_fwd_mla")
    return o, lse


def ringx_attn_bwd_mla_workspace_bytes(B, H, N, d_qk, d_v, kv_chunk) -> int:
    return lib().ringx_attn_bwd_mla_workspace_bytes(B, H, N, d_qk, d_v, kv_chunk)


def ringx_attn_bwd_mla(q, k, v, o, lse, dO, kv_chunk: int, scale: float, dq=None, dk=None, dv=None, workspace=None):
    """(dq, dk, dv) for multi-head latent attention shapes: q, k [B,H,N,192], v, o, dO [B,H,N,128] bf16 (include/ringx.h:
    ringx_attn_bwd_mla)."""
    _check_mla_shapes(q, k, v)
    B, H, N, d_qk = q.shape
    d_v = v.shape[3]
    dq = torch.empty_like(q) if dq is None else dq
    dk = torch.empty_like(k) if dk is None else dk
    dv = torch.empty_like(v) if dv is None else dv
    for t, nm in ((o, "o"), (dO, "dO"), (dv, "dv")):
        _expect(t, v.shape, nm, q.dtype)
    for t, nm in ((dq, "dq"), (dk, "dk")):
        _expect(t, q.shape, nm, q.dtype)
    _expect(lse, (B, H, N), "lse", torch.float32)
    need = lib().ringx_attn_bwd_mla_workspace_bytes(B, H, N, d_qk, d_v, kv_chunk)
    if workspace is None:
        workspace = _workspace(max(need, 256), q.device)
    st = lib().ringx_attn_bwd_mla(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o, "o"), _dev(lse, "lse"), _dev(dO, "dO"),
                                  _dev(dq, "dq"), _dev(dk, "dk"), _dev(dv, "dv"), B, H, N, d_qk, d_v, kv_chunk, scale,
                                  _DTYPES[q.dtype], workspace.data_ptr(), workspace.numel(), _stream())
    _check(st, "ringx_attn_bwd_mla")
    return dq, dk, dv


def ringx_attn_chunk_fwd_mla(q, k, v, scale: float, o_acc=None, lse_acc=None, final: bool = False):
    """One pass of the MLA widths in general form (include/ringx.h: ringx_attn_chunk_fwd_mla): q [B,H,Nq,192] against
    k [B,H,Nk,192], v [B,H,Nk,128].  No accumulator: (loc_out fp32, loc_lse), or (o bf16, lse) when final.  With
    (o_acc, lse_acc): folds this pass in -- in place, or, when final, into a new (o bf16, lse)."""
    _check_mla_shapes(q, k, v, same_len=False)
    B, H, Nq, d_qk = q.shape
    Nk, d_v = k.shape[2], v.shape[3]
    if (o_acc is None) != (lse_acc is None):
        raise ValueError("o_acc and lse_acc go together")
    if final:
        o_out = torch.empty((B, H, Nq, d_v), dtype=torch.bfloat16, device=q.device)
        lse_out = torch.empty((B, H, Nq), dtype=torch.float32, device=q.device)
    elif o_acc is not None:
        o_out, lse_out = o_acc, lse_acc
    else:
        o_out = torch.empty((B, H, Nq, d_v), dtype=torch.float32, device=q.device)
        lse_out = torch.empty((B, H, Nq), dtype=torch.float32, device=q.device)
    st = lib().ringx_attn_chunk_fwd_mla(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"),
                                        _dev(o_acc, "o_acc") if o_acc is not None else None,
                                        _dev(lse_acc, "lse_acc") if lse_acc is not None else None,
                                        _dev(o_out, "o_out"), _dev(lse_out, "lse_out"), B, H, Nq, Nk, d_qk, d_v, scale,
                                        _DTYPES[q.dtype], _DTYPES[o_out.dtype], _stream())
    _check(st, "ringx_attn_chunk_fwd_mla")
    return o_out, lse_out


def ringx_attn_bwd_partial_mla_workspace_bytes(B, H, Nq) -> int:
    return lib().ringx_attn_bwd_partial_mla_workspace_bytes(B, H, Nq)


def ringx_attn_bwd_partial_mla(q, k, v, o, lse, dO, scale: float, dq_acc_t, dk, dv, workspace, prepared: bool = False):
    """The per-device backward step for the MLA widths (include/ringx.h: ringx_attn_bwd_partial_mla).  dq_acc_t holds the
    fp32 dQ accumulator TRANSPOSED, [B,H,192,Nq] (any tensor of B*H*Nq*192 floats: it is opaque until
    ringx_dq_finalize_mla); dk, dv bf16 or float32 shares.  Every buffer is the caller's; returns (dq_acc_t, dk, dv)."""
    _check_mla_shapes(q, k, v, same_len=False)
    B, H, Nq, d_qk = q.shape
    Nk, d_v = k.shape[2], v.shape[3]
    if dk.dtype != dv.dtype:
        raise ValueError("dk and dv must have the same dtype")
    if dq_acc_t.dtype != torch.float32 or dq_acc_t.numel() != q.numel():
        raise ValueError("dq_acc_t must hold B*H*Nq*d_qk floats")
    _expect(o, (B, H, Nq, d_v), "o", q.dtype)
    _expect(dO, (B, H, Nq, d_v), "dO", q.dtype)
    _expect(lse, (B, H, Nq), "lse", torch.float32)
    _expect(dk, (B, H, Nk, d_qk), "dk")
    _expect(dv, (B, H, Nk, d_v), "dv")
    _expect_workspace(workspace, lib().ringx_attn_bwd_partial_mla_workspace_bytes(B, H, Nq), "ringx_attn_bwd_partial_mla")
    st = lib().ringx_attn_bwd_partial_mla(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o, "o"), _dev(lse, "lse"),
                                          _dev(dO, "dO"), _dev(dq_acc_t, "dq_acc_t"), _dev(dk, "dk"), _dev(dv, "dv"),
                                          B, H, Nq, Nk, d_qk, d_v, scale, _DTYPES[q.dtype], _DTYPES[dk.dtype],
                                          1 if prepared else 0, workspace.data_ptr(),
                                          workspace.numel() * workspace.element_size(), _stream())
    _check(st, "ringx_attn_bwd_partial_mla")
    return dq_acc_t, dk, dv


def ringx_dq_finalize_mla(dq_acc_t, B, H, Nq, d_qk=192, dq=None):
    """dq [B,H,Nq,192] bf16 from the transposed fp32 accumulator (include/ringx.h: ringx_dq_finalize_mla)."""
    if dq is None:
        dq = torch.empty((B, H, Nq, d_qk), dtype=torch.bfloat16, device=dq_acc_t.device)
    _check(lib().ringx_dq_finalize_mla(_dev(dq_acc_t, "dq_acc_t"), _dev(dq, "dq"), B, H, Nq, d_qk, _stream()),
           "ringx_dq_finalize_mla")
    return dq


def ringx_attn_chunk_fwd(q, k, v, scale: float):
    """(loc_out fp32, loc_lse) of q [B,H,Nq,d] against the keys k,v [B,H,Nk,d] (one chunk pass)."""
    B, H, Nq, d = q.shape
    Nk = k.shape[2]
    loc_out = torch.empty((B, H, Nq, d), dtype=torch.float32, device=q.device)
    loc_lse = torch.empty((B, H, Nq), dtype=torch.float32, device=q.device)
    st = lib().ringx_attn_chunk_fwd(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(loc_out, "loc_out"),
                                    _dev(loc_lse, "loc_lse"), B, H, Nq, Nk, d, scale, _DTYPES[q.dtype], _stream())
    _check(st, "ringx_attn_chunk_fwd")
    return loc_out, loc_lse


def ringx_attn_chunk_fwd_ex_workspace_bytes(B, H, Nq, Nk, d, dtype) -> int:
    return lib().ringx_attn_chunk_fwd_ex_workspace_bytes(B, H, Nq, Nk, d, _DTYPES[dtype])


def ringx_attn_chunk_fwd_ex(q, k, v, scale: float, o_acc=None, lse_acc=None, final: bool = False, workspace=None):
    """One pass in its general form, with split-KV when the pass cannot fill the GPU (include/ringx.h:
    ringx_attn_chunk_fwd_ex).  No accumulator: returns (loc_out fp32, loc_lse), or (o bf16, lse) when final.  With
    (o_acc, lse_acc): folds this pass in -- in place (returns them) or, when final, into a new (o bf16, lse)."""
    B, H, Nq, d = q.shape
    Nk = k.shape[2]
    if (o_acc is None) != (lse_acc is None):
        raise ValueError("o_acc and lse_acc go together")
    if final:
        o_out = torch.empty((B, H, Nq, d), dtype=torch.bfloat16, device=q.device)
        lse_out = torch.empty((B, H, Nq), dtype=torch.float32, device=q.device)
    elif o_acc is not None:
        o_out, lse_out = o_acc, lse_acc
    else:
        o_out = torch.empty((B, H, Nq, d), dtype=torch.float32, device=q.device)
        lse_out = torch.empty((B, H, Nq), dtype=torch.float32, device=q.device)
    need = lib().ringx_attn_chunk_fwd_ex_workspace_bytes(B, H, Nq, Nk, d, _DTYPES[q.dtype])
    if workspace is None and need:
        workspace = _workspace(need, q.device)
    st = lib().ringx_attn_chunk_fwd_ex(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"),
                                       _dev(o_acc, "o_acc") if o_acc is not None else None,
                                       _dev(lse_acc, "lse_acc") if lse_acc is not None else None,
                                       _dev(o_out, "o_out"), _dev(lse_out, "lse_out"), B, H, Nq, Nk, d, scale,
                                       _DTYPES[q.dtype], _DTYPES[o_out.dtype],
                                       workspace.data_ptr() if workspace is not None else None,
                                       workspace.numel() if workspace is not None else 0, _stream())
    _check(st, "ringx_attn_chunk_fwd_ex")
    return o_out, lse_out


def ringx_lse_merge(o_a, lse_a, o_b, lse_b, out_dtype=None, inplace: bool = False):
    """Two-operand Eq. 5 on [..., d] partials (include/ringx.h: ringx_lse_merge)."""
    d = o_a.shape[-1]
    rows = o_a.numel() // d if d else 0
    out_dtype = o_a.dtype if out_dtype is None else out_dtype
    if inplace:
        if out_dtype != o_a.dtype:
            raise ValueError("in-place merge keeps the dtype of operand a")
        o_out, lse_out = o_a, lse_a
    else:
        o_out = torch.empty(o_a.shape, dtype=out_dtype, device=o_a.device)
        lse_out = torch.empty_like(lse_a)
    st = lib().ringx_lse_merge(_dev(o_a, "o_a"), _dev(lse_a, "lse_a"), _dev(o_b, "o_b"), _dev(lse_b, "lse_b"),
                               _dev(o_out, "o_out"), _dev(lse_out, "lse_out"), rows, d, _DTYPES[o_a.dtype],
                               _DTYPES[out_dtype], _stream())
    _check(st, "ringx_lse_merge")
    return o_out, lse_out


def ringx_attn_bwd(q, k, v, o, lse, dO, kv_chunk: int, scale: float, workspace=None, dq=None, dk=None, dv=None):
    """dQ, dK, dV (bf16) from the saved (o, lse) of ringx_attn_fwd (include/ringx.h: ringx_attn_bwd)."""
    B, H, N, d = q.shape
    dt = _DTYPES[q.dtype]
    dq = torch.empty_like(q) if dq is None else dq
    dk = torch.empty_like(k) if dk is None else dk
    dv = torch.empty_like(v) if dv is None else dv
    for t, nm in ((k, "k"), (v, "v"), (o, "o"), (dO, "dO"), (dq, "dq"), (dk, "dk"), (dv, "dv")):
        _expect(t, q.shape, nm, q.dtype)
    _expect(lse, (B, H, N), "lse", torch.float32)
    need = lib().ringx_attn_bwd_workspace_bytes(B, H, N, d, kv_chunk, dt)
    if workspace is None:
        workspace = _workspace(max(need, 256), q.device)
    st = lib().ringx_attn_bwd(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o, "o"), _dev(lse, "lse"),
                              _dev(dO, "dO"), _dev(dq, "dq"), _dev(dk, "dk"), _dev(dv, "dv"),
                              B, H, N, d, kv_chunk, scale, dt, workspace.data_ptr(),
                              workspace.numel() * workspace.element_size(), _stream())
    _check(st, "ringx_attn_bwd")
    return dq, dk, dv


def ringx_attn_fwd_host(q_host, k_host, v_host, kv_chunk: int, scale: float, o_host=None, lse_host=None,
                        workspace=None, device="cuda"):
    """End-to-end entry with HOST tensors (pinned recommended): H2D, forward, D2H, synchronise."""
    B, H, N, d = q_host.shape
    dt = _DTYPES[q_host.dtype]
    for t in (q_host, k_host, v_host):
        if t.is_cuda or not t.is_contiguous():
            raise ValueError("ringx_attn_fwd_host takes contiguous HOST tensors")
    if o_host is None:
        o_host = torch.empty_like(q_host).pin_memory()
    if lse_host is None:
        lse_host = torch.empty((B, H, N), dtype=torch.float32).pin_memory()
    need = lib().ringx_attn_fwd_host_workspace_bytes(B, H, N, d, kv_chunk, dt)
    if workspace is None:
        workspace = _workspace(need, device)
    with torch.cuda.device(workspace.device):
        st = lib().ringx_attn_fwd_host(q_host.data_ptr(), k_host.data_ptr(), v_host.data_ptr(), o_host.data_ptr(),
                                       lse_host.data_ptr(), B, H, N, d, kv_chunk, scale, dt, workspace.data_ptr(),
                                       workspace.numel(), _stream())
    _check(st, "ringx_attn_fwd_host")
    return o_host, lse_host


def ringx_attn_fwd_bwd_host_workspace_bytes(B, H, N, d, kv_chunk, dtype) -> int:
    return lib().ringx_attn_fwd_bwd_host_workspace_bytes(B, H, N, d, kv_chunk, _DTYPES[dtype])


def ringx_attn_fwd_bwd_host(q_host, k_host, v_host, dO_host, kv_chunk: int, scale: float, outs=None, workspace=None,
                            device="cuda"):
    """End-to-end forward+backward with HOST tensors: returns (o, lse, dq, dk, dv) host tensors."""
    B, H, N, d = q_host.shape
    dt = _DTYPES[q_host.dtype]
    for t in (q_host, k_host, v_host, dO_host):
        if t.is_cuda or not t.is_contiguous():
            raise ValueError("ringx_attn_fwd_bwd_host takes contiguous HOST tensors")
    if outs is None:
        outs = (torch.empty_like(q_host).pin_memory(), torch.empty((B, H, N), dtype=torch.float32).pin_memory(),
                torch.empty_like(q_host).pin_memory(), torch.empty_like(q_host).pin_memory(),
                torch.empty_like(q_host).pin_memory())
    o_host, lse_host, dq_host, dk_host, dv_host = outs
    need = lib().ringx_attn_fwd_bwd_host_workspace_bytes(B, H, N, d, kv_chunk, dt)
    if workspace is None:
        workspace = _workspace(need, device)
    with torch.cuda.device(workspace.device):
        st = lib().ringx_attn_fwd_bwd_host(q_host.data_ptr(), k_host.data_ptr(), v_host.data_ptr(), dO_host.data_ptr(),
                                           o_host.data_ptr(), lse_host.data_ptr(), dq_host.data_ptr(),
                                           dk_host.data_ptr(), dv_host.data_ptr(), B, H, N, d, kv_chunk, scale, dt,
                                           workspace.data_ptr(), workspace.numel(), _stream())
    _check(st, "ringx_attn_fwd_bwd_host")
    return outs


def ringx_set_deterministic(on: bool) -> None:
    """Bit-reproducible dQ, process-wide (include/ringx.h: ringx_set_deterministic)."""
    _check(lib().ringx_set_deterministic(1 if on else 0), "ringx_set_deterministic")


def ringx_get_deterministic() -> bool:
    return bool(lib().ringx_get_deterministic())


def ringx_last_launch_count() -> int:
    return lib().ringx_last_launch_count()


PROFILE_KINDS = ("attn_fwd", "merge", "attn_bwd", "bwd_aux", "tokeniser", "proj")


def ringx_profile_enable(on: bool) -> None:
    _check(lib().ringx_profile_enable(1 if on else 0), "ringx_profile_enable")


def ringx_profile_read() -> dict:
    """{kind: (total_ms, launches)} of the launches recorded since the last read (synchronises)."""
    ms = (ctypes.c_double * len(PROFILE_KINDS))()
    n = (ctypes.c_int * len(PROFILE_KINDS))()
    _check(lib().ringx_profile_read(ms, n), "ringx_profile_read")
    return {k: (ms[i], n[i]) for i, k in enumerate(PROFILE_KINDS)}


def ringx_version() -> int:
    return lib().ringx_version()


def ringx_qkv_proj(x, w_qkv, H: int, q=None, k=None, v=None):
    """[q|k|v] = x W_qkv^T in the head-split layout (include/ringx.h: ringx_qkv_proj).  x [B,S,h], w_qkv [3h,h]."""
    B, S, h = x.shape
    d = h // H
    if x.dtype != torch.bfloat16 or w_qkv.dtype != torch.bfloat16 or tuple(w_qkv.shape) != (3 * h, h) or d * H != h:
        raise ValueError("x [B,S,h] and w_qkv [3h,h] must be bfloat16 with h = H*d")
    q, k, v = (torch.empty((B, H, S, d), dtype=torch.bfloat16, device=x.device) if t is None else t for t in (q, k, v))
    _check(lib().ringx_qkv_proj(_dev(x, "x"), _dev(w_qkv, "w_qkv"), _dev(q, "q"), _dev(k, "k"), _dev(v, "v"), B, S, H, d,
                                _stream()), "ringx_qkv_proj")
    return q, k, v


def ringx_out_proj(o, w_o, y=None):
    """y = merge_heads(o) W_o^T (include/ringx.h: ringx_out_proj).  o [B,H,S,d], w_o [h,h] -> y [B,S,h]."""
    B, H, S, d = o.shape
    h = H * d
    if o.dtype != torch.bfloat16 or w_o.dtype != torch.bfloat16 or tuple(w_o.shape) != (h, h):
        raise ValueError("o [B,H,S,d] and w_o [h,h] must be bfloat16")
    y = torch.empty((B, S, h), dtype=torch.bfloat16, device=o.device) if y is None else y
    _check(lib().ringx_out_proj(_dev(o, "o"), _dev(w_o, "w_o"), _dev(y, "y"), B, S, H, d, _stream()), "ringx_out_proj")
    return y


def ringx_out_proj_bwd(dy, o, w_o):
    """(dO bf16 [B,H,S,d], dW_o fp32 [h,h]) (include/ringx.h: ringx_out_proj_bwd)."""
    B, H, S, d = o.shape
    h = H * d
    d_o = torch.empty_like(o)
    dw = torch.empty((h, h), dtype=torch.float32, device=o.device)
    _check(lib().ringx_out_proj_bwd(_dev(dy, "dy"), _dev(o, "o"), _dev(w_o, "w_o"), _dev(d_o, "d_o"), _dev(dw, "dw_o"),
                                    B, S, H, d, _stream()), "ringx_out_proj_bwd")
    return d_o, dw


def ringx_qkv_proj_bwd(dq, dk, dv, x, w_qkv):
    """(dX bf16 [B,S,h], dW_qkv fp32 [3h,h]) (include/ringx.h: ringx_qkv_proj_bwd)."""
    B, H, S, d = dq.shape
    h = H * d
    dx = torch.empty_like(x)
    dw = torch.empty((3 * h, h), dtype=torch.float32, device=x.device)
    _check(lib().ringx_qkv_proj_bwd(_dev(dq, "dq"), _dev(dk, "dk"), _dev(dv, "dv"), _dev(x, "x"), _dev(w_qkv, "w_qkv"),
                                    _dev(dx, "dx"), _dev(dw, "dw_qkv"), B, S, H, d, _stream()), "ringx_qkv_proj_bwd")
    return dx, dw


def ringx_attn_block_bwd_workspace_bytes(B, S, H, d, kv_chunk) -> int:
    return lib().ringx_attn_block_bwd_workspace_bytes(B, S, H, d, kv_chunk)


def ringx_attn_block_bwd(x, w_qkv, w_o, dy, fwd_workspace, H: int, kv_chunk: int, scale: float, workspace=None):
    """(dX bf16, dW_qkv fp32, dW_o fp32) of the attention block; `fwd_workspace` is the workspace tensor the matching
    ringx_attn_block_fwd call used (include/ringx.h: ringx_attn_block_bwd)."""
    B, S, h = x.shape
    d = h // H
    dx = torch.empty_like(x)
    dw_qkv = torch.empty((3 * h, h), dtype=torch.float32, device=x.device)
    dw_o = torch.empty((h, h), dtype=torch.float32, device=x.device)
    need = lib().ringx_attn_block_bwd_workspace_bytes(B, S, H, d, kv_chunk)
    if workspace is None:
        workspace = _workspace(max(need, 256), x.device)
    st = lib().ringx_attn_block_bwd(_dev(x, "x"), _dev(w_qkv, "w_qkv"), _dev(w_o, "w_o"), _dev(dy, "dy"),
                                    _dev(fwd_workspace, "fwd_workspace"), _dev(dx, "dx"), _dev(dw_qkv, "dw_qkv"),
                                    _dev(dw_o, "dw_o"), B, S, H, d, kv_chunk, scale, workspace.data_ptr(),
                                    workspace.numel(), _stream())
    _check(st, "ringx_attn_block_bwd")
    return dx, dw_qkv, dw_o


def ringx_attn_block_fwd_workspace_bytes(B, S, H, d, kv_chunk) -> int:
    return lib().ringx_attn_block_fwd_workspace_bytes(B, S, H, d, kv_chunk)


def ringx_attn_block_fwd(x, w_qkv, w_o, H: int, kv_chunk: int, scale: float, y=None, workspace=None):
    """The attention block of Table II (include/ringx.h: ringx_attn_block_fwd).  x [B,S,h] -> y [B,S,h]."""
    B, S, h = x.shape
    d = h // H
    if any(t.dtype != torch.bfloat16 for t in (x, w_qkv, w_o)) or tuple(w_qkv.shape) != (3 * h, h) or \
            tuple(w_o.shape) != (h, h) or d * H != h:
        raise ValueError("x [B,S,h], w_qkv [3h,h], w_o [h,h] must be bfloat16 with h = H*d")
    y = torch.empty_like(x) if y is None else y
    need = lib().ringx_attn_block_fwd_workspace_bytes(B, S, H, d, kv_chunk)
    if workspace is None:
        workspace = _workspace(max(need, 256), x.device)
    st = lib().ringx_attn_block_fwd(_dev(x, "x"), _dev(w_qkv, "w_qkv"), _dev(w_o, "w_o"), _dev(y, "y"), B, S, H, d,
                                    kv_chunk, scale, workspace.data_ptr(), workspace.numel(), _stream())
    _check(st, "ringx_attn_block_fwd")
    return y


def ringx_fidelity_tokens(y, origin, size, k: int, sigma: float = 0.0, out_dtype=torch.float32, tokens=None):
    """One fidelity mode F_k(C(Y)) of the Turbulence-Transformer tokeniser (include/ringx.h: ringx_fidelity_tokens).
    y [M,D,H,W,4] fp32; origin (z0,y0,x0); size (Dc,Hc,Wc).  Returns tokens [M,Dc/k,Hc/k,Wc/k,4] of out_dtype."""
    M, D, H, W, C = y.shape
    if y.dtype != torch.float32:
        raise ValueError("y must be float32")
    (z0, y0, x0), (Dc, Hc, Wc) = origin, size
    if tokens is None:
        tokens = torch.empty((M, max(Dc // max(k, 1), 0), max(Hc // max(k, 1), 0), max(Wc // max(k, 1), 0), C),
                             dtype=out_dtype, device=y.device)
    st = lib().ringx_fidelity_tokens(_dev(y, "y"), _dev(tokens, "tokens"), M, D, H, W, C, z0, y0, x0, Dc, Hc, Wc, k,
                                     float(sigma), _DTYPES[tokens.dtype], _stream())
    _check(st, "ringx_fidelity_tokens")
    return tokens


def _expect_bwd_partial(q, k, v, o, lse, dO, dq_acc, dk, dv):
    """Shapes of one per-device backward step: q, o, dO [B,H,Nq,d]; k, v, dk, dv [B,H,Nk,d]; lse [B,H,Nq]; dq_acc B*H*Nq*d
    floats.  The kernel writes dk, dv with the sizes of k: a slice of another length would be written out of bounds."""
    B, H, Nq, d = q.shape
    Nk = k.shape[2]
    _expect(k, (B, H, Nk, d), "k", q.dtype)
    _expect(v, (B, H, Nk, d), "v", q.dtype)
    _expect(o, q.shape, "o", q.dtype)
    _expect(dO, q.shape, "dO", q.dtype)
    _expect(lse, (B, H, Nq), "lse", torch.float32)
    _expect(dk, (B, H, Nk, d), "dk")
    _expect(dv, (B, H, Nk, d), "dv", dk.dtype)
    if dq_acc.dtype != torch.float32 or dq_acc.numel() != q.numel():
        raise ValueError(f"dq_acc must hold B*H*Nq*d = {q.numel()} floats, got {dq_acc.numel()} of {dq_acc.dtype}")


def ringx_attn_bwd_partial(q, k, v, o, lse, dO, scale: float, dq_acc=None, dk=None, dv=None, workspace=None):
    """Per-device backward step (include/ringx.h: ringx_attn_bwd_partial): q,o,dO [B,H,Nq,d], k,v [B,H,Nk,d].
    Adds these keys' contribution to dq_acc (fp32, allocated and zeroed when None); returns (dq_acc, dk, dv)."""
    B, H, Nq, d = q.shape
    Nk = k.shape[2]
    if dq_acc is None:
        dq_acc = torch.zeros((B, H, Nq, d), dtype=torch.float32, device=q.device)
    dk = torch.empty_like(k) if dk is None else dk
    dv = torch.empty_like(v) if dv is None else dv
    _expect_bwd_partial(q, k, v, o, lse, dO, dq_acc, dk, dv)
    need = lib().ringx_attn_bwd_partial_workspace_bytes(B, H, Nq, d)
    if workspace is None:
        workspace = _workspace(max(need, 256), q.device)
    _expect_workspace(workspace, need, "ringx_attn_bwd_partial")
    st = lib().ringx_attn_bwd_partial(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o, "o"), _dev(lse, "lse"),
                                      _dev(dO, "dO"), _dev(dq_acc, "dq_acc"), _dev(dk, "dk"), _dev(dv, "dv"),
                                      B, H, Nq, Nk, d, scale, _DTYPES[q.dtype], workspace.data_ptr(),
                                      workspace.numel() * workspace.element_size(), _stream())
    _check(st, "ringx_attn_bwd_partial")
    return dq_acc, dk, dv


def ringx_attn_bwd_partial_ex(q, k, v, o, lse, dO, scale: float, dq_acc, dk, dv, workspace, prepared: bool = False):
    """The per-device backward step in its general form (include/ringx.h: ringx_attn_bwd_partial_ex): dk, dv may be
    float32 (this device's unrounded share of a cross-device sum); `prepared` reuses the D / lse2 that an earlier step of the
    same backward left in `workspace`.  Every buffer is the caller's; returns (dq_acc, dk, dv)."""
    B, H, Nq, d = q.shape
    Nk = k.shape[2]
    if dk.dtype != dv.dtype:
        raise ValueError("dk and dv must have the same dtype")
    _expect_bwd_partial(q, k, v, o, lse, dO, dq_acc, dk, dv)
    _expect_workspace(workspace, lib().ringx_attn_bwd_partial_workspace_bytes(B, H, Nq, d), "ringx_attn_bwd_partial_ex")
    st = lib().ringx_attn_bwd_partial_ex(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o, "o"), _dev(lse, "lse"),
                                         _dev(dO, "dO"), _dev(dq_acc, "dq_acc"), _dev(dk, "dk"), _dev(dv, "dv"),
                                         B, H, Nq, Nk, d, scale, _DTYPES[q.dtype], _DTYPES[dk.dtype], 1 if prepared else 0,
                                         workspace.data_ptr(), workspace.numel() * workspace.element_size(), _stream())
    _check(st, "ringx_attn_bwd_partial_ex")
    return dq_acc, dk, dv


def ringx_dq_finalize(dq_acc, dq=None):
    """bf16 cast of the fp32 dQ accumulator (include/ringx.h: ringx_dq_finalize)."""
    if dq is None:
        dq = torch.empty(dq_acc.shape, dtype=torch.bfloat16, device=dq_acc.device)
    _check(lib().ringx_dq_finalize(_dev(dq_acc, "dq_acc"), _dev(dq, "dq"), dq_acc.numel(), _stream()),
           "ringx_dq_finalize")
    return dq


def ringx_eq5_scale(loc_out, loc_lse, lse_max, inplace: bool = False):
    """(num, den) of one operand of the N-operand Eq. 5 (include/ringx.h: ringx_eq5_scale)."""
    d = loc_out.shape[-1]
    rows = loc_out.numel() // d
    num = loc_out if inplace else torch.empty_like(loc_out)
    den = torch.empty_like(loc_lse)
    _check(lib().ringx_eq5_scale(_dev(loc_out, "loc_out"), _dev(loc_lse, "loc_lse"), _dev(lse_max, "lse_max"),
                                 _dev(num, "num"), _dev(den, "den"), rows, d, _stream()), "ringx_eq5_scale")
    return num, den


def ringx_eq5_finalize(num, den, lse_max, out_dtype=torch.float32):
    """o = num/den, lse = lse_max + log(den) (include/ringx.h: ringx_eq5_finalize)."""
    d = num.shape[-1]
    rows = num.numel() // d
    o = torch.empty(num.shape, dtype=out_dtype, device=num.device)
    lse = torch.empty_like(den)
    _check(lib().ringx_eq5_finalize(_dev(num, "num"), _dev(den, "den"), _dev(lse_max, "lse_max"), _dev(o, "o"),
                                    _dev(lse, "lse"), rows, d, _DTYPES[out_dtype], _stream()), "ringx_eq5_finalize")
    return o, lse


def ringx_attn_bwd_partial_workspace_bytes(B, H, Nq, d) -> int:
    return lib().ringx_attn_bwd_partial_workspace_bytes(B, H, Nq, d)


def ringx_attn_fwd_gqa(q, k, v, kv_chunk: int, scale: float, o=None, lse=None, workspace=None):
    """Grouped-query forward: q [B,Hq,N,d], k,v [B,Hkv,N,d] (include/ringx.h: ringx_attn_fwd_gqa)."""
    B, Hq, N, d = q.shape
    Hkv = k.shape[1]
    dt = _DTYPES[q.dtype]
    o = torch.empty_like(q) if o is None else o
    lse = torch.empty((B, Hq, N), dtype=torch.float32, device=q.device) if lse is None else lse
    _expect(k, (B, Hkv, N, d), "k", q.dtype)
    _expect(v, (B, Hkv, N, d), "v", q.dtype)
    _expect(o, q.shape, "o", q.dtype)
    _expect(lse, (B, Hq, N), "lse", torch.float32)
    need = lib().ringx_attn_fwd_workspace_bytes(B, Hq, N, d, kv_chunk, dt)
    if workspace is None:
        workspace = _workspace(need, q.device)
    ws_ptr = workspace.data_ptr() if workspace is not None else None
    ws_len = workspace.numel() * workspace.element_size() if workspace is not None else 0
    st = lib().ringx_attn_fwd_gqa(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o, "o"), _dev(lse, "lse"),
                                  B, Hq, Hkv, N, d, kv_chunk, scale, dt, ws_ptr, ws_len, _stream())
    _check(st, "ringx_attn_fwd_gqa")
    return o, lse


def ringx_attn_bwd_gqa(q, k, v, o, lse, dO, kv_chunk: int, scale: float, workspace=None):
    """Grouped-query backward: dq [B,Hq,N,d], dk, dv [B,Hkv,N,d] (include/ringx.h: ringx_attn_bwd_gqa)."""
    B, Hq, N, d = q.shape
    Hkv = k.shape[1]
    dt = _DTYPES[q.dtype]
    dq, dk, dv = torch.empty_like(q), torch.empty_like(k), torch.empty_like(v)
    _expect(k, (B, Hkv, N, d), "k", q.dtype)
    _expect(v, (B, Hkv, N, d), "v", q.dtype)
    for t, nm in ((o, "o"), (dO, "dO")):
        _expect(t, q.shape, nm, q.dtype)
    _expect(lse, (B, Hq, N), "lse", torch.float32)
    need = lib().ringx_attn_bwd_workspace_bytes(B, Hq, N, d, kv_chunk, dt)
    if workspace is None:
        workspace = _workspace(max(need, 256), q.device)
    st = lib().ringx_attn_bwd_gqa(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o, "o"), _dev(lse, "lse"),
                                  _dev(dO, "dO"), _dev(dq, "dq"), _dev(dk, "dk"), _dev(dv, "dv"),
                                  B, Hq, Hkv, N, d, kv_chunk, scale, dt, workspace.data_ptr(),
                                  workspace.numel() * workspace.element_size(), _stream())
    _check(st, "ringx_attn_bwd_gqa")
    return dq, dk, dv


def ringx_attn_chunk_fwd_fold(q, k, v, o_acc, lse_acc, scale: float, final: bool = False):
    """One chunk pass folded into the running fp32 (o_acc, lse_acc) by Eq. 5 inside the kernel (include/ringx.h:
    ringx_attn_chunk_fwd_fold).  final=False: in place, returns (o_acc, lse_acc); final=True: returns the folded
    result as (o bf16, lse), the accumulators untouched."""
    B, H, Nq, d = q.shape
    Nk = k.shape[2]
    o_f = lse_f = None
    if final:
        o_f = torch.empty((B, H, Nq, d), dtype=q.dtype, device=q.device)
        lse_f = torch.empty((B, H, Nq), dtype=torch.float32, device=q.device)
    st = lib().ringx_attn_chunk_fwd_fold(_dev(q, "q"), _dev(k, "k"), _dev(v, "v"), _dev(o_acc, "o_acc"),
                                         _dev(lse_acc, "lse_acc"), _dev(o_f, "o_final") if final else None,
                                         _dev(lse_f, "lse_final") if final else None, B, H, Nq, Nk, d, scale,
                                         _DTYPES[q.dtype], _stream())
    _check(st, "ringx_attn_chunk_fwd_fold")
    return (o_f, lse_f) if final else (o_acc, lse_acc)
