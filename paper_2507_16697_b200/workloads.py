"""Seeded synthetic inputs for the RingX hot path (shared by the tests, the oracle side and bench.py).

This module holds NONE of the method's arithmetic: it only draws numbers.  Both the CUDA path and
the fp64 oracle are fed the *same bits* produced here (the oracle gets them widened exactly to
fp64), so it is the one module the two sides have in common.

Recipe (BASELINE.json `configs`): tensors are `[B,H,N,d]`, d fastest; values are
iid N(0,1) drawn by a counter-based generator -- SplitMix64 of (seed, tensor_id, element index)
-> two 24-bit uniforms -> Box-Muller in fp32 -> optional gain (x3 for Q,K of the peaked config C5)
-> rounded to bf16 RN-even for the bf16 configs.  The paper's own workloads (JHTDB forced HIT and
stratified Taylor-Green fields pushed through the trained Matey model)
are not available; these inputs take the paper's *shapes* (3-D voxel grids flattened to 10^4-10^6
tokens, Table III) and stand in for them.
"""
from __future__ import annotations

import dataclasses
import math

import torch

_MASK64 = (1 << 64) - 1


def _s64(x: int) -> int:
    """Python int (mod 2^64) -> the signed 64-bit value torch.int64 holds."""
    x &= _MASK64
    return x - (1 << 64) if x >= (1 << 63) else x


def _lshr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical right shift of an int64 tensor."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def _splitmix64(z: torch.Tensor) -> torch.Tensor:
    z = z + _s64(0x9E3779B97F4A7C15)
    z = (z ^ _lshr(z, 30)) * _s64(0xBF58476D1CE4E5B9)
    z = (z ^ _lshr(z, 27)) * _s64(0x94D049BB133111EB)
    return z ^ _lshr(z, 31)


def normal_f32(numel: int, seed: int, tensor_id: int, device="cpu", chunk: int = 1 << 24) -> torch.Tensor:
    """`numel` iid N(0,1) fp32 values, a pure function of (seed, tensor_id, element index)."""
    out = torch.empty(numel, dtype=torch.float32, device=device)
    key = _s64((seed * 0x100000001B3) ^ (tensor_id * 0xD6E8FEB86659FD93))
    for lo in range(0, numel, chunk):
        hi = min(numel, lo + chunk)
        idx = torch.arange(lo, hi, dtype=torch.int64, device=device)
        z = _splitmix64(_splitmix64(idx ^ key) + key)
        u1 = ((_lshr(z, 40) & 0xFFFFFF).to(torch.float32) + 1.0) * (1.0 / 16777216.0)  # (0,1]
        u2 = (z & 0xFFFFFF).to(torch.float32) * (1.0 / 16777216.0)                      # [0,1)
        out[lo:hi] = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)
    return out


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json config (SURVEY.md §8 shorthand C1..C5)."""
    name: str
    dtype: str          # "f32" | "bf16"
    B: int
    H: int
    N: int
    d: int
    kv_chunk: int
    qk_gain: float = 1.0
    backward: bool = False
    seed: int = 0
    note: str = ""

    @property
    def scale(self) -> float:
        return 1.0 / math.sqrt(self.d)

    @property
    def fwd_flops(self) -> float:      # PAPER.md:188-189 (Table II): 2bS^2h + 2bS^2h
        return 4.0 * self.B * self.H * self.N * self.N * self.d

    @property
    def bwd_flops(self) -> float:      # five 2*N^2*d GEMMs
        return 10.0 * self.B * self.H * self.N * self.N * self.d


CONFIGS = {
    "C1": Config("C1", "f32", 1, 1, 1024, 64, 256, seed=20250717, note="fp32 single head, 4 chunks of 256"),
    "C2": Config("C2", "bf16", 1, 16, 32768, 64, 4096, seed=20250718, note="32^3 voxel grid, x-fastest"),
    "C3": Config("C3", "bf16", 1, 8, 262144, 128, 32768, seed=20250719, note="64^3 voxel tokens"),
    "C4": Config("C4", "bf16", 2, 16, 65536, 64, 8192, backward=True, seed=20250720, note="fwd+bwd"),
    "C5": Config("C5", "bf16", 1, 4, 1048576, 128, 65536, qk_gain=3.0, seed=20250721, note="peaked softmax"),
}

TENSOR_IDS = {"q": 0, "k": 1, "v": 2, "do": 3, "x": 4, "w_qkv": 5, "w_o": 6}


def make_block_inputs(B: int, S: int, H: int, d: int, seed: int = 20250723, device="cpu"):
    """Inputs of the attention block of Table II: x [B,S,h] ~ N(0,1); W_qkv [3h,h], W_o [h,h] ~
    N(0, 1/h) (so that q, k, v come out ~ N(0,1), the distribution of the BASELINE.json configs); all bf16."""
    h = H * d
    x = make_tensor((B, S, h), "x", seed=seed, device=device)
    w_qkv = make_tensor((3 * h, h), "w_qkv", seed=seed, gain=h ** -0.5, device=device)
    w_o = make_tensor((h, h), "w_o", seed=seed, gain=h ** -0.5, device=device)
    return x, w_qkv, w_o


def make_tensor(cfg_or_shape, which: str, seed: int | None = None, dtype: str | None = None,
                gain: float | None = None, device="cpu") -> torch.Tensor:
    """One of q/k/v/do as a contiguous `[B,H,N,d]` tensor (torch.float32 or torch.bfloat16)."""
    if isinstance(cfg_or_shape, Config):
        cfg = cfg_or_shape
        shape = (cfg.B, cfg.H, cfg.N, cfg.d)
        seed = cfg.seed if seed is None else seed
        dtype = cfg.dtype if dtype is None else dtype
        if gain is None:
            gain = cfg.qk_gain if which in ("q", "k") else 1.0
    else:
        shape = tuple(cfg_or_shape)
        seed = 0 if seed is None else seed
        dtype = "bf16" if dtype is None else dtype
        gain = 1.0 if gain is None else gain
    numel = math.prod(shape)
    x = normal_f32(numel, seed, TENSOR_IDS[which], device=device)
    if gain != 1.0:
        x = x * gain
    x = x.view(shape)
    if dtype == "bf16":
        return x.to(torch.bfloat16)          # RN-even
    if dtype == "f32":
        return x
    raise ValueError(f"unknown dtype {dtype!r}")


def make_qkv(cfg_or_shape, with_do: bool = False, device="cpu", **kw):
    names = ("q", "k", "v") + (("do",) if with_do else ())
    return tuple(make_tensor(cfg_or_shape, n, device=device, **kw) for n in names)


def to_f64_numpy(t: torch.Tensor):
    """Exact widening of the bits the GPU sees to the fp64 numpy array the oracle takes."""
    return t.detach().to("cpu").to(torch.float64).numpy()


def voxel_token_index(x: int, y: int, z: int, G: int) -> int:
    """Token order of the grid configs: x fastest.  Metadata only -- non-causal
    attention with no positional term is permutation-equivariant, which the tests use."""
    return x + G * (y + G * z)


# ------------------------------------------------------------------------------------------------
# Synthetic turbulence-like state for the tokeniser (Y in R^{D x H x W x 4} = V_x, V_y, V_z, P).
# The paper's fields (JHTDB forced HIT 1024^3; stratified Taylor-Green, Table VI) are not available;
# this stand-in has their *shape and layout* and a value structure with both large scales and grid-scale noise:
# per variable, `n_modes` seeded Fourier modes with integer wave vectors |kappa| <= 8 and amplitude ~ |kappa|^(-5/6)
# (a Kolmogorov-like E(kappa) ~ kappa^(-5/3)), plus 0.25 * iid N(0,1) from the counter-based generator.
# No arithmetic of the method (no filtering, no cropping) happens here.
# ------------------------------------------------------------------------------------------------
FIELD_TENSOR_ID = 8


def make_field(M: int, D: int, H: int, W: int, seed: int = 20250722, n_modes: int = 6, device="cpu") -> torch.Tensor:
    """Y [M, D, H, W, 4] fp32, channels fastest; a pure function of (seed, shape)."""
    C = 4
    out = torch.empty((M, D, H, W, C), dtype=torch.float32, device=device)
    par = normal_f32(M * C * n_modes * 5, seed, FIELD_TENSOR_ID + 1).view(M, C, n_modes, 5)
    z = torch.arange(D, dtype=torch.float32, device=device).view(D, 1, 1) / D
    y = torch.arange(H, dtype=torch.float32, device=device).view(1, H, 1) / H
    x = torch.arange(W, dtype=torch.float32, device=device).view(1, 1, W) / W
    for m in range(M):
        noise = normal_f32(D * H * W * C, seed + 1 + m, FIELD_TENSOR_ID, device=device).view(D, H, W, C)
        for c in range(C):
            f = 0.25 * noise[..., c]
            for j in range(n_modes):
                kz, ky, kx = (int(round(float(v) * 3.0)) for v in par[m, c, j, :3])
                kz, ky, kx = (max(-8, min(8, v)) for v in (kz, ky, kx))
                kk = max(1.0, math.sqrt(kz * kz + ky * ky + kx * kx))
                phase = float(par[m, c, j, 3]) * math.pi
                f = f + (kk ** (-5.0 / 6.0)) * torch.sin((2.0 * math.pi) * (kz * z + ky * y + kx * x) + phase)
            out[m, ..., c] = f
    return out
