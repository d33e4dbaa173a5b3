"""-m gpu: parity at BASELINE.json's FULL size (configs[1]: Qwen3-32B-shaped layer, H=5120, I=25600,
p=25 %) in the launch configuration bench.py times: spense_mlp captured in a CUDA graph, bf16 output,
the next layer named as L2 prefetch hint, replayed several times.

The oracle finishes the whole layer in about half a minute on the host cores, so every element is
compared, not a sample: pack bit-exact (canonical arrays), h within tol_glu, y within tol_gemm against
the oracle fed the GPU's own Hq bytes, Hq = E4M3(h_gpu / s_h) bit for bit."""
import numpy as np
import pytest
import torch

import spense_inputs as si
from oracle import spense_oracle as o
from tests.gpu_common import assert_down_parity, assert_gate_up_parity, cuda

pytestmark = pytest.mark.gpu

H, I, P = 5120, 25600, 0.25


@pytest.fixture(scope="module")
def sp():
    from paper_2606_10445_b200 import build, spense
    build.build()
    assert torch.cuda.is_available()
    return spense


@pytest.fixture(scope="module")
def layer(sp):
    """One full-size layer: generated on the host (the oracle needs the bytes), packed on the GPU."""
    L = si.make_layer(H, I, P, seed=2000)
    canon = o.pack_canonical(L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(), L.perm.numpy(), L.I_dense)
    wg, wu, wd = o.unpack_canonical(canon)
    pk = sp.spense_pack(cuda(L.wgate), cuda(L.wup), cuda(L.wdown), L.w_scale, cuda(L.perm), L.I_dense, want_canon=True)
    torch.cuda.synchronize()
    return dict(L=L, canon=canon, wg=wg, wu=wu, wd=wd, pk=pk)


def test_full_size_pack_bit_exact(sp, layer):
    assert layer["L"].I_dense == 6400
    for k, ref in layer["canon"].items():
        got = layer["pk"].canon[k].cpu().numpy()
        assert got.shape == ref.shape and np.array_equal(got, ref), k


@pytest.mark.parametrize("M", [1, 64, 128])
def test_full_size_mlp_parity_in_bench_launch_configuration(sp, layer, M):
    L, pk = layer["L"], layer["pk"]
    x, s_x = si.make_activations(M, H, 1000 + M)
    r1 = o.gate_up(x.numpy(), s_x.numpy(), layer["wg"], layer["wu"], L.w_scale[0], L.w_scale[1], 1.0)
    s_h = o.requant_scale_from_h(r1["h"])
    r = o.gate_up(x.numpy(), s_x.numpy(), layer["wg"], layer["wu"], L.w_scale[0], L.w_scale[1], s_h)
    ws = sp.spense_workspace(pk, max(M, 256))
    xd, sxd, shd = cuda(x), cuda(s_x), cuda(torch.from_numpy(s_h))

    # eager, fp32 output, with the fp32 dump of h
    h = torch.full((M, I), float("nan"), dtype=torch.float32, device="cuda")
    hq = sp.spense_gate_up(pk, xd, sxd, shd, ws, h_f32=h)
    y32 = sp.spense_down(pk, hq, shd, ws)
    torch.cuda.synchronize()
    h_gpu, hq_gpu = h.cpu().numpy(), hq.cpu().numpy()
    assert not np.isnan(h_gpu).any()
    frac = assert_gate_up_parity(r, h_gpu, hq_gpu, s_h, f"gate_up M={M}")
    assert frac < 5e-3
    assert_down_parity(y32.cpu().numpy(), hq_gpu, s_h, layer["wd"], L.w_scale[2], f"down M={M}")

    # bench.py's launch: CUDA graph of 2 x spense_mlp (bf16 out, next-layer hint), replayed
    hq2 = torch.empty(M, I, dtype=torch.uint8, device="cuda")
    y16 = torch.empty(M, H, dtype=torch.bfloat16, device="cuda")

    def step():
        for _ in range(2):
            sp.spense_mlp(pk, xd, sxd, shd, ws, hq_scratch=hq2, y=y16, next_layer=pk)

    step()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            step()
    torch.cuda.current_stream().wait_stream(s)
    for _ in range(3):
        y16.zero_()
        hq2.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(hq2, hq), "graph replay: Hq differs from the eager launch"
        assert torch.equal(y16, y32.to(torch.bfloat16)), "graph replay: bf16 y is not the RNE rounding of the fp32 y"


@pytest.mark.parametrize("M", [256, 2048])
def test_full_size_many_tokens_sampled_rows(sp, layer, M):
    """BASELINE.json configs[1] at M=256 and configs[4] (prefill-shaped, M=2048): ONE launch per GEMM over
    128-token blocks.  Token rows are independent, so the oracle computes a sample of them one by one (first and
    last row of blocks, a ragged spread in between) and every column of those rows is compared."""
    L, pk = layer["L"], layer["pk"]
    x, s_x = si.make_activations(M, H, 3000 + M)
    rows = np.unique(np.concatenate([[0, 1, 127, 128, 129, 255, M - 129, M - 128, M - 1],
                                     np.random.default_rng(M).integers(0, M, 23)])).astype(np.int64)
    xs, sxs = x.numpy()[rows], s_x.numpy()[rows]
    r1 = o.gate_up(xs, sxs, layer["wg"], layer["wu"], L.w_scale[0], L.w_scale[1], 1.0)
    s_h = np.full(M, 0.05, np.float32)
    s_h[rows] = o.requant_scale_from_h(r1["h"])
    r = o.gate_up(xs, sxs, layer["wg"], layer["wu"], L.w_scale[0], L.w_scale[1], s_h[rows])
    ws = sp.spense_workspace(pk, M)
    xd, sxd, shd = cuda(x), cuda(s_x), cuda(torch.from_numpy(s_h))
    h = torch.full((M, I), float("nan"), dtype=torch.float32, device="cuda")
    hq = sp.spense_gate_up(pk, xd, sxd, shd, ws, h_f32=h)
    y = sp.spense_down(pk, hq, shd, ws)
    y2 = sp.spense_mlp(pk, xd, sxd, shd, ws)
    torch.cuda.synchronize()
    assert not torch.isnan(h).any()
    h_s, hq_s, y_s = h.cpu().numpy()[rows], hq.cpu().numpy()[rows], y.cpu().numpy()[rows]
    frac = assert_gate_up_parity(r, h_s, hq_s, s_h[rows], f"gate_up M={M} sampled rows")
    assert frac < 5e-3
    assert_down_parity(y_s, hq_s, s_h[rows], layer["wd"], L.w_scale[2], f"down M={M} sampled rows")
    assert torch.equal(y, y2)
    # every row: Hq is the E4M3 cast of the kernel's own h (the decision is taken in fp32 on both sides)
    own = o.e4m3_encode((h.cpu().numpy() / s_h[:, None]).astype(np.float32))
    assert np.array_equal(own, hq.cpu().numpy())
