"""CPU-side checks of the boundary: libringx.so builds (nvcc cross-compiles), loads, and exports every
symbol include/ringx.h declares; host-only entry points (workspace queries, status strings, argument
validation that happens before any CUDA call) behave as the header says.  No compute call is made."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ringx.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2507_16697_b200.build import build_library
    from paper_2507_16697_b200 import ringx
    build_library()
    return ringx.lib()


def declared_symbols():
    text = open(HEADER).read()
    return sorted(set(re.findall(r"RINGX_API\s+[\w\s\*]+?\b(ringx_\w+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    syms = declared_symbols()
    for name in ("ringx_attn_fwd", "ringx_attn_bwd", "ringx_lse_merge"):
        assert name in syms
    assert len(syms) >= 10


def test_every_declared_symbol_is_exported(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in ringx.h but not exported by libringx.so"


def test_no_torch_or_cxx_types_cross_the_boundary():
    text = open(HEADER).read()
    assert "torch" not in text.lower() and "std::" not in text and "at::" not in text
    # the header must compile as plain C
    r = subprocess.run(["gcc", "-std=c99", "-fsyntax-only", "-x", "c", HEADER], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr


def test_binding_has_the_same_names():
    from paper_2507_16697_b200 import ringx
    for name in declared_symbols():
        if name in ("ringx_status_string",):
            continue
        assert hasattr(ringx, name), f"python binding lacks {name}"


def test_version_and_status_strings(lib):
    assert lib.ringx_version() >= 100
    seen = set()
    for st in range(0, 8):
        s = lib.ringx_status_string(st).decode()
        assert s and s != "unknown status"
        seen.add(s)
    assert len(seen) == 8
    assert lib.ringx_status_string(99).decode() == "unknown status"


def test_workspace_queries_are_host_only(lib):
    align = lambda n: (n + 255) // 256 * 256
    f = lib.ringx_attn_fwd_workspace_bytes
    # single pass needs no workspace; multi-pass bf16 needs the running fp32 accumulator [R,d] + [R]
    # (Eq. 5 is folded in the chunk kernel's epilogue: no separate partial buffer)
    assert f(1, 1, 1024, 64, 1024, 1) == 0
    R, d = 2 * 4 * 1024, 128
    assert f(2, 4, 1024, d, 256, 1) == R * d * 4 + R * 4
    assert f(2, 4, 1024, d, 256, 0) == R * d * 4 + R * 4          # f32 accumulates in the caller's o
    # unsupported shapes report 0 (and the compute entry points reject them)
    assert f(1, 1, 1000, 64, 250, 1) == 0
    assert f(1, 1, 1024, 96, 256, 1) == 0
    assert f(1, 1, 1024, 64, 1152, 1) == 0                        # kv_chunk longer than the sequence rounded up to a tile
    assert f(1, 1, 1024, 64, 384, 0) == 0                         # fp32: N % kv_chunk != 0
    # bf16 takes any sequence length and a short last chunk: the running accumulator for the rows that exist
    assert f(1, 1, 1024, 64, 384, 1) == 1024 * 64 * 4 + 1024 * 4
    assert f(1, 1, 1000, 64, 256, 1) == 1000 * 64 * 4 + align(1000 * 4)
    assert f(1, 1, 100, 128, 128, 1) == 0                         # one (ragged) pass
    b = lib.ringx_attn_bwd_workspace_bytes
    # D, lse2, the dQ accumulator (fp32, or int32 fixed point in deterministic mode), the per-row fixed-point scales
    # and the two K/V maxima per head
    assert b(2, 4, 1024, 64, 256, 1) == 3 * R * 4 + R * 64 * 4 + 256
    assert b(2, 4, 1024, 64, 256, 0) == 0                         # backward is bf16 only
    h = lib.ringx_attn_fwd_host_workspace_bytes
    assert h(2, 4, 1024, d, 256, 1) == 4 * R * d * 2 + R * 4 + f(2, 4, 1024, d, 256, 1)


def test_argument_validation_happens_before_any_cuda_call(lib):
    """NULL pointers, bad dtypes and bad shapes are rejected on the host (works on a box with no GPU)."""
    buf = ctypes.create_string_buffer(4096)
    p = ctypes.cast(buf, ctypes.c_void_p).value
    p = (p + 255) // 256 * 256
    assert lib.ringx_attn_fwd(None, p, p, p, p, 1, 1, 256, 64, 256, 0.125, 1, None, 0, None) == 1      # NULL_PTR
    assert lib.ringx_attn_fwd(p, p, p, p, p, 1, 1, 256, 64, 256, 0.125, 7, None, 0, None) == 3         # BAD_DTYPE
    assert lib.ringx_attn_fwd(p, p, p, p, p, 1, 1, 250, 64, 250, 0.125, 1, None, 0, None) == 2         # BAD_SHAPE
    assert lib.ringx_attn_fwd(p, p, p, p, p, 1, 1, 256, 64, 256, 0.0, 1, None, 0, None) == 2           # scale <= 0
    assert lib.ringx_attn_fwd(p, p, p, p, p, 1, 1, 256, 64, 256, float("nan"), 1, None, 0, None) == 2
    assert lib.ringx_attn_fwd(p + 4, p, p, p, p, 1, 1, 256, 64, 256, 0.125, 1, None, 0, None) == 4     # MISALIGNED
    assert lib.ringx_attn_fwd(p, p, p, p, p, 1, 1, 512, 64, 256, 0.125, 1, None, 0, None) == 1         # ws NULL
    assert lib.ringx_attn_fwd(p, p, p, p, p, 1, 1, 512, 64, 256, 0.125, 1, p, 16, None) == 5           # ws small
    assert lib.ringx_lse_merge(p, p, p, p, p, p, -1, 64, 0, 0, None) == 2
    assert lib.ringx_lse_merge(p, p, p, p, p, p, 8, 60, 0, 0, None) == 2
    assert lib.ringx_lse_merge(p, p, p, p, p, p, 8, 64, 0, 5, None) == 3
    assert lib.ringx_lse_merge(None, None, None, None, None, None, 0, 64, 0, 0, None) == 0             # rows=0 no-op
    assert lib.ringx_attn_bwd(p, p, p, p, p, p, p, p, p, 1, 1, 256, 64, 256, 0.125, 0, p, 1 << 20, None) == 3
    assert lib.ringx_attn_chunk_fwd(p, p, p, p, p, 1, 1, 256, 100, 64, 0.125, 0, None) == 2   # fp32: Nk % 128
    assert lib.ringx_attn_chunk_fwd(p, p, p, p, p, 1, 1, 256, 0, 64, 0.125, 1, None) == 2
    # the MLA dQ finalize takes what ringx_attn_bwd_partial_mla can have produced: Nq % 128 == 0 (not 64)
    assert lib.ringx_dq_finalize_mla(p, p, 1, 1, 192, 192, None) == 2
    assert lib.ringx_dq_finalize_mla(p, p, 1, 1, 64, 192, None) == 2
    assert lib.ringx_dq_finalize_mla(p, p, 1, 1, 256, 128, None) == 2


def test_product_fails_loudly_without_the_library(monkeypatch, tmp_path):
    from paper_2507_16697_b200 import ringx
    monkeypatch.setattr(ringx, "_lib", None)
    monkeypatch.setattr(ringx, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU or PyTorch fallback"):
        ringx.lib()


def test_product_rejects_cpu_tensors(lib):
    import torch
    from paper_2507_16697_b200 import ringx
    q = torch.zeros(1, 1, 256, 64, dtype=torch.bfloat16)
    with pytest.raises(ValueError, match="CUDA tensor"):
        ringx.ringx_attn_fwd(q, q, q, 256, 0.125, o=torch.empty_like(q), lse=torch.empty(1, 1, 256))


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2507_16697_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2507_16697_b200" not in re.sub(r'"""[\s\S]*?"""', "", text), f


def test_binding_refuses_tensors_whose_shapes_disagree():
    """The C ABI takes one set of sizes for all tensors of a call; the binding must refuse a tensor of another shape or
    dtype BEFORE the call (it would be read or written out of bounds).  Needs no GPU: the check precedes the device check."""
    import pytest
    import torch
    from paper_2507_16697_b200 import ringx
    q = torch.zeros(1, 2, 256, 64, dtype=torch.bfloat16)
    with pytest.raises(ValueError, match="k has shape"):
        ringx.ringx_attn_fwd(q, q[:, :1], q, 256, 0.125)
    with pytest.raises(ValueError, match="dO has shape"):
        ringx.ringx_attn_bwd(q, q, q, q, torch.zeros(1, 2, 256), q[:, :, :128], 256, 0.125)
    with pytest.raises(ValueError, match="lse has dtype"):
        ringx.ringx_attn_bwd(q, q, q, q, torch.zeros(1, 2, 256, dtype=torch.float64), q, 256, 0.125)
    qm, vm = torch.zeros(1, 2, 256, 192, dtype=torch.bfloat16), torch.zeros(1, 1, 256, 128, dtype=torch.bfloat16)
    with pytest.raises(ValueError, match="MLA shapes"):
        ringx.ringx_attn_fwd_mla(qm, qm, vm, 256, 0.1)
    # the per-device backward steps (what ringx_dist hands slices to): keys of another length than dk / dv, a gradient
    # accumulator of another size, a workspace smaller than the size query
    kk = torch.zeros(1, 2, 384, 64, dtype=torch.bfloat16)
    lse = torch.zeros(1, 2, 256)
    acc = torch.zeros(1, 2, 256, 64)
    ws = torch.zeros(1 << 16, dtype=torch.uint8)
    with pytest.raises(ValueError, match="dk has shape"):
        ringx.ringx_attn_bwd_partial_ex(q, kk, kk, q, lse, q, 0.125, acc, kk[:, :, :256], kk, ws)
    with pytest.raises(ValueError, match="v has shape"):
        ringx.ringx_attn_bwd_partial_ex(q, kk, kk[:, :, :128], q, lse, q, 0.125, acc, kk, kk, ws)
    with pytest.raises(ValueError, match="dq_acc"):
        ringx.ringx_attn_bwd_partial_ex(q, kk, kk, q, lse, q, 0.125, acc[:, :1], kk, kk, ws)
    with pytest.raises(ValueError, match="lse has shape"):
        ringx.ringx_attn_bwd_partial(q, kk, kk, q, lse[:, :, :128], q, 0.125, dq_acc=acc)
    with pytest.raises(ValueError, match="workspace"):
        ringx.ringx_attn_bwd_partial_ex(q, kk, kk, q, lse, q, 0.125, acc, kk, kk, ws[:64])
    km, vv = torch.zeros(1, 2, 384, 192, dtype=torch.bfloat16), torch.zeros(1, 2, 384, 128, dtype=torch.bfloat16)
    om = torch.zeros(1, 2, 256, 128, dtype=torch.bfloat16)
    acc_t = torch.zeros(1, 2, 192, 256)
    with pytest.raises(ValueError, match="dv has shape"):
        ringx.ringx_attn_bwd_partial_mla(qm, km, vv, om, lse, om, 0.1, acc_t, km, vv[:, :, :256], ws)
    with pytest.raises(ValueError, match="o has shape"):
        ringx.ringx_attn_bwd_partial_mla(qm, km, vv, om[:, :, :128], lse, om, 0.1, acc_t, km, vv, ws)
    with pytest.raises(ValueError, match="workspace"):
        ringx.ringx_attn_bwd_partial_mla(qm, km, vv, om, lse, om, 0.1, acc_t, km, vv, ws[:64])
