"""The C ABI used from plain C: tests/c_abi/ringx_c1.c is compiled with gcc against include/ringx.h and linked against
libringx.so + libcudart -- no Python, no PyTorch in the process that computes (the property include/ringx.h promises;
SURVEY.md §7 step 2).  It runs BASELINE.json configs[0] (C1) through ringx_attn_fwd and through ringx_attn_chunk_fwd +
ringx_lse_merge (Eq. 5) and compares with tests/golden/c1_expected.txt, values the fp64 oracle wrote
(tests/golden/make_c1_golden.py).  Compiling and linking is a CPU test; running needs the GPU."""
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "c_abi", "ringx_c1.c")
GOLDEN = os.path.join(ROOT, "tests", "golden", "c1_expected.txt")
SRC_RAGGED = os.path.join(ROOT, "tests", "c_abi", "ringx_bf16_ragged.c")
GOLDEN_RAGGED = os.path.join(ROOT, "tests", "golden", "bf16_ragged_expected.txt")
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def build_program(tmp_path, src=SRC):
    from paper_2507_16697_b200.build import build_library, PKG_DIR
    build_library()
    exe = str(tmp_path / os.path.splitext(os.path.basename(src))[0])
    cmd = ["gcc", "-std=c99", "-O1", "-Wall", "-Werror", src, "-I", os.path.join(ROOT, "include"),
           "-I", os.path.join(CUDA_HOME, "include"), "-L", PKG_DIR, "-lringx", "-L", os.path.join(CUDA_HOME, "lib64"),
           "-lcudart", "-lm", f"-Wl,-rpath,{PKG_DIR}", f"-Wl,-rpath,{os.path.join(CUDA_HOME, 'lib64')}", "-o", exe]
    r = subprocess.run(cmd, capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    return exe


def test_c_program_compiles_and_links_against_the_library(tmp_path):
    exe = build_program(tmp_path)
    # nothing of Python or torch is linked in
    r = subprocess.run(["ldd", exe], capture_output=True, text=True)
    libs = [line.split()[0] for line in r.stdout.splitlines() if line.strip()]        # sonames, not install paths
    assert any(x.startswith("libringx.so") for x in libs) and any(x.startswith("libcudart") for x in libs), libs
    assert not any("python" in x.lower() or "torch" in x.lower() or "c10" in x.lower() for x in libs), libs


def test_golden_file_is_what_the_committed_script_writes(tmp_path):
    """The stored expected values are reproducible from oracle/ alone."""
    from oracle import attention as orc
    from paper_2507_16697_b200 import workloads as wl
    cfg = wl.CONFIGS["C1"]
    q, k, v = wl.make_qkv(cfg)
    o, lse = orc.attention_fwd(wl.to_f64_numpy(q[0, 0]), wl.to_f64_numpy(k[0, 0]), wl.to_f64_numpy(v[0, 0]), cfg.scale)
    n = 0
    for line in open(GOLDEN):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] == "lse":
            assert abs(lse[int(f[1])] - float(f[2])) <= 1e-13
        else:
            assert f[0] == "o" and abs(o[int(f[1]), int(f[2])] - float(f[3])) <= 1e-13
        n += 1
    assert n >= 1000


@pytest.mark.gpu
def test_c_program_runs_C1_without_python_in_the_process(tmp_path):
    from paper_2507_16697_b200 import workloads as wl
    exe = build_program(tmp_path)
    cfg = wl.CONFIGS["C1"]
    q, k, v = wl.make_qkv(cfg)
    inputs = tmp_path / "c1_inputs.bin"
    with open(inputs, "wb") as f:
        for t in (q, k, v):
            f.write(np.ascontiguousarray(t.numpy(), dtype="<f4").tobytes())
    r = subprocess.run([exe, str(inputs), GOLDEN], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "RINGX_C1_OK" in r.stdout, (r.stdout, r.stderr)
    sys.stdout.write(r.stdout)


# ---- the bf16 forward AND backward of a ragged sequence (N = 333) from plain C: tests/c_abi/ringx_bf16_ragged.c
def _ragged_golden_module():
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_bf16_ragged_golden",
                                                  os.path.join(ROOT, "tests", "golden", "make_bf16_ragged_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_ragged_c_program_compiles_and_links(tmp_path):
    exe = build_program(tmp_path, SRC_RAGGED)
    libs = [line.split()[0] for line in subprocess.run(["ldd", exe], capture_output=True, text=True).stdout.splitlines() if line.strip()]
    assert any(x.startswith("libringx.so") for x in libs)
    assert not any("python" in x.lower() or "torch" in x.lower() or "c10" in x.lower() for x in libs), libs


def test_ragged_golden_file_is_what_the_committed_script_writes():
    """The stored expected values are reproducible from oracle/ alone (to the 10 digits the file keeps)."""
    want = _ragged_golden_module().expected()
    got = [line.split() for line in open(GOLDEN_RAGGED) if line.strip() and not line.startswith("#")]
    assert len(got) == len(want) >= 6000
    for (name, idx, val), f in zip(want, got):
        assert f[0] == name and int(f[1]) == idx and abs(float(f[2]) - val) <= 1e-9 * max(1.0, abs(val))


@pytest.mark.gpu
def test_ragged_c_program_runs_forward_and_backward_without_python_in_the_process(tmp_path):
    exe = build_program(tmp_path, SRC_RAGGED)
    inputs = tmp_path / "ragged_inputs.bin"
    with open(inputs, "wb") as f:
        for t in _ragged_golden_module().inputs():          # q, k, v, dO as raw bf16
            f.write(t.contiguous().view(__import__("torch").int16).numpy().astype("<i2").tobytes())
    r = subprocess.run([exe, str(inputs), GOLDEN_RAGGED], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "RINGX_BF16_RAGGED_OK" in r.stdout, (r.stdout, r.stderr)
    sys.stdout.write(r.stdout)
