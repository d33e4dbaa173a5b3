"""Seeded synthetic inputs for the Spense FP8 GLU-MLP path (shared by the oracle tests, the GPU
tests and bench.py).

This module holds NONE of the method's arithmetic: it only draws random tensors and prepares
them the way the paper's pipeline would hand them to the runtime (FP8 models,
MLP pruned).  It imports neither ``oracle/`` nor the CUDA package.  The FP8 casts are torch's own
library casts (``Tensor.to(torch.float8_e4m3fn)`` after an explicit clamp), a third party to both
sides.  Magnitude 2:4 pruning stands in for SparseGPT (out of scope: needs calibration data).

Recipe:
* weights fp32 ~ N(0, 0.02^2), three independent matrices gate/up [I, H], down [H, I];
* dense set D: I_d = round(p*I/128)*128 indices drawn uniformly without replacement (seeded);
  perm = stable partition (non-dense ascending, then dense ascending);
* in PERMUTED order, rows < I_s of gate/up are 2:4-magnitude-pruned along H and columns < I_s of
  down along the (permuted) intermediate dim: keep the 2 largest |w| of every 4, ties -> lower index;
* per-tensor scale amax/448, cast to E4M3;
* activations fp32 ~ N(0,1), ``n_outlier`` seeded channels x20, per-token scale amax/448, E4M3.

Everything runs on ``device`` (CPU for parity cases, CUDA for bench layers that no oracle sees).
"""
from __future__ import annotations

import dataclasses

import torch

E4M3_MAX = 448.0

# BASELINE.json configs (shapes only; M and p are swept by the callers)
SHAPES = {
    "tiny": dict(H=256, I=1024),            # configs[0]
    "qwen3_32b": dict(H=5120, I=25600),     # configs[1], [3], [4]
    "seed_oss_36b": dict(H=5120, I=27648),  # configs[2]
}


def dense_count(I: int, p: float, align: int = 128) -> int:
    return int(round(p * I / align)) * align


@dataclasses.dataclass
class Layer:
    H: int
    I: int
    I_dense: int
    wgate: torch.Tensor    # uint8 [I, H]  E4M3 bytes, ORIGINAL index order
    wup: torch.Tensor      # uint8 [I, H]
    wdown: torch.Tensor    # uint8 [H, I]
    w_scale: tuple         # (s_gate, s_up, s_down) python floats (fp32 values)
    perm: torch.Tensor     # int32 [I]  perm[new] = old
    dense_idx: torch.Tensor  # int64 [I_dense] sorted


def _to_e4m3_bytes(x: torch.Tensor) -> torch.Tensor:
    return torch.clamp(x, -E4M3_MAX, E4M3_MAX).to(torch.float8_e4m3fn).view(torch.uint8)


def _prune_2_4_lastdim(w: torch.Tensor) -> torch.Tensor:
    """Keep the 2 largest |w| of every 4 consecutive along the last dim (ties -> lower index)."""
    shp = w.shape
    a = w.abs().reshape(-1, 4)
    keep = torch.empty_like(a, dtype=torch.bool)
    for i in range(4):
        beats = torch.zeros(a.shape[0], dtype=torch.int32, device=w.device)
        for j in range(4):
            if j == i:
                continue
            if j < i:
                beats += (a[:, j] >= a[:, i]).to(torch.int32)
            else:
                beats += (a[:, j] > a[:, i]).to(torch.int32)
        keep[:, i] = beats < 2
    return (w.reshape(-1, 4) * keep).reshape(shp)


def _quant_tensor(w: torch.Tensor):
    amax = w.abs().max().to(torch.float32)
    s = (amax / E4M3_MAX) if float(amax) > 0 else torch.tensor(1.0, device=w.device)
    s = s.to(torch.float32)
    return _to_e4m3_bytes(w / s), float(s)


def make_layer(H: int, I: int, p: float, seed: int, device="cpu", I_dense: int | None = None,
               prune: bool = True, all_2_4: bool = False) -> Layer:
    """One synthetic Spense layer.  ``all_2_4`` prunes the dense region too (used by the
    dense-fraction-invariance test: the same weights are then valid at any I_dense)."""
    dev = torch.device(device)
    g = torch.Generator(device=dev).manual_seed(int(seed))
    I_d = dense_count(I, p) if I_dense is None else int(I_dense)
    I_s = I - I_d
    order = torch.randperm(I, generator=g, device=dev)
    dense_idx = torch.sort(order[:I_d]).values
    is_dense = torch.zeros(I, dtype=torch.bool, device=dev)
    is_dense[dense_idx] = True
    idx = torch.arange(I, device=dev)
    perm = torch.cat([idx[~is_dense], idx[is_dense]])

    out = []
    for name in ("gate", "up"):
        w = torch.randn(I, H, generator=g, device=dev, dtype=torch.float32) * 0.02
        if prune:
            wp = w[perm]
            n = I if all_2_4 else I_s
            if n:
                wp[:n] = _prune_2_4_lastdim(wp[:n])
            w = torch.empty_like(wp)
            w[perm] = wp
            del wp
        out.append(_quant_tensor(w))
        del w
    w = torch.randn(H, I, generator=g, device=dev, dtype=torch.float32) * 0.02
    if prune:
        wp = w[:, perm]
        n = I if all_2_4 else I_s
        if n:
            wp[:, :n] = _prune_2_4_lastdim(wp[:, :n].contiguous())
        w = torch.empty_like(wp)
        w[:, perm] = wp
        del wp
    out.append(_quant_tensor(w))
    del w
    return Layer(H=H, I=I, I_dense=I_d, wgate=out[0][0], wup=out[1][0], wdown=out[2][0],
                 w_scale=(out[0][1], out[1][1], out[2][1]), perm=perm.to(torch.int32),
                 dense_idx=dense_idx)


@dataclasses.dataclass
class Linear:
    N: int
    K: int
    n_dense: int
    split: str             # "out": rows split (perm over N); "in": columns split (perm over K)
    w: torch.Tensor        # uint8 [N, K] E4M3 bytes, ORIGINAL order
    w_scale: float
    perm: torch.Tensor     # int32, perm[new] = old


def linear_dense_count(N: int, K: int, p: float, split: str) -> int:
    """dense rows / columns: a multiple of 128; the out-split keeps its sparse row count a multiple of 256 (one MMA tile)"""
    if split == "out":
        return N - int(round((1.0 - p) * N / 256)) * 256
    return dense_count(K, p)


def make_linear(N: int, K: int, p: float, split: str, seed: int, device="cpu", n_dense: int | None = None) -> Linear:
    """One synthetic Spense linear (same recipe as make_layer, one matrix): W ~ N(0, 0.02^2) [N, K]; a seeded dense set of
    rows (split "out") or columns (split "in"), perm = stable partition; in PERMUTED order the sparse region is
    magnitude-2:4 pruned along K; per-tensor scale amax/448, E4M3."""
    dev = torch.device(device)
    g = torch.Generator(device=dev).manual_seed(int(seed))
    n = N if split == "out" else K
    n_d = linear_dense_count(N, K, p, split) if n_dense is None else int(n_dense)
    n_s = n - n_d
    order = torch.randperm(n, generator=g, device=dev)
    is_dense = torch.zeros(n, dtype=torch.bool, device=dev)
    is_dense[order[:n_d]] = True
    idx = torch.arange(n, device=dev)
    perm = torch.cat([idx[~is_dense], idx[is_dense]])
    w = torch.randn(N, K, generator=g, device=dev, dtype=torch.float32) * 0.02
    if n_s:
        if split == "out":
            wp = w[perm]
            wp[:n_s] = _prune_2_4_lastdim(wp[:n_s])
            w = torch.empty_like(wp)
            w[perm] = wp
        else:
            wp = w[:, perm]
            wp[:, :n_s] = _prune_2_4_lastdim(wp[:, :n_s].contiguous())
            w = torch.empty_like(wp)
            w[:, perm] = wp
    wb, sc = _quant_tensor(w)
    return Linear(N=N, K=K, n_dense=n_d, split=split, w=wb, w_scale=sc, perm=perm.to(torch.int32))


def make_activations(M: int, H: int, seed: int, device="cpu", n_outlier: int | None = None):
    """x uint8 [M, H] E4M3 bytes, s_x fp32 [M] (per-token amax/448)."""
    dev = torch.device(device)
    g = torch.Generator(device=dev).manual_seed(int(seed) + 7919)
    x = torch.randn(M, H, generator=g, device=dev, dtype=torch.float32)
    if n_outlier is None:
        n_outlier = 4 if H <= 1024 else int(round(0.001 * H))
    ch = torch.randperm(H, generator=g, device=dev)[:n_outlier]
    x[:, ch] *= 20.0
    amax = x.abs().amax(dim=1)
    s = torch.where(amax > 0, amax / E4M3_MAX, torch.ones_like(amax)).to(torch.float32)
    return _to_e4m3_bytes(x / s[:, None]), s


def make_small_int_case(H: int, I: int, I_dense: int, M: int, seed: int):
    """Exactness case: E4M3 bytes whose values are small integers (|v| <= 3) so that every
    partial sum is an integer below 2^24 -- any summation order gives the same fp32 result.
    Sparse region 2:4 by construction (2 random positions per group non-zero)."""
    g = torch.Generator().manual_seed(int(seed))
    codes = torch.tensor([0x00, 0x38, 0x40, 0x44, 0xB8, 0xC0, 0xC4], dtype=torch.uint8)  # 0, +-1, +-2, +-3

    def rnd(shape):
        return codes[torch.randint(0, len(codes), shape, generator=g)]

    def mask24(rows, cols):
        r = torch.rand(rows, cols // 4, 4, generator=g)
        keep = r.argsort(dim=2).argsort(dim=2) < 2
        return keep.reshape(rows, cols)

    I_s = I - I_dense
    wg, wu = rnd((I, H)), rnd((I, H))
    wd = rnd((H, I))
    if I_s:
        wg[:I_s] *= mask24(I_s, H)
        wu[:I_s] *= mask24(I_s, H)
        wd[:, :I_s] *= mask24(H, I_s)
    x = rnd((M, H))
    return wg, wu, wd, x
