"""-m gpu: stand-alone Spense linears (spense_pack_linear, spense_linear_out_split / _in_split; SURVEY.md 8f NEXT-3,
PAPER.md:123-125) through the C ABI against the CPU oracle: pack bit-exact (canonical arrays and the blob body), GEMM
within |gpu - oracle| <= 2e-3 * sum|a*w| + 1e-5 per element on the fp32 output."""
import numpy as np
import pytest
import torch

import spense_inputs as si
from oracle import spense_oracle as o
from tests import blob_layout
from tests.gpu_common import cuda

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    from paper_2606_10445_b200 import build, spense
    build.build()
    assert torch.cuda.is_available()
    return spense


def _split_id(sp, split):
    return sp.SPENSE_SPLIT_OUT if split == "out" else sp.SPENSE_SPLIT_IN


# N, K, p, split, M: several tiles and spans, ragged K (K % 256 == 128), a dense half tile, both degenerate splits,
# one token block (down to 16 token columns) and several side by side
LINEAR_CASES = [
    (1024, 256, 0.25, "out", 8),
    (1024, 256, 0.25, "in", 8),
    (1024, 384, 0.0, "out", 33),      # all sparse, K % 256 == 128
    (1024, 384, 1.0, "out", 33),      # all dense == the baseline kernel
    (640, 1152, 0.2, "out", 64),      # 512 sparse rows + a dense half tile (128 rows)
    (384, 1024, 0.25, "in", 64),      # N % 256 == 128: half row tile
    (384, 1024, 0.0, "in", 5),
    (384, 1024, 1.0, "in", 100),
    (4096, 1024, 0.25, "out", 16),    # enough stages for many spans and split-K partials
    (1024, 4096, 0.25, "in", 16),
    (4096, 1024, 0.25, "out", 128),   # one full-width token block
    (1024, 4096, 0.25, "in", 200),
    (2048, 512, 0.5, "out", 300),     # two token blocks
    (512, 2048, 0.5, "in", 513),      # three token blocks, ragged last one
]


@pytest.mark.parametrize("N,K,p,split,M", LINEAR_CASES)
def test_linear_pack_and_gemm_parity(sp, N, K, p, split, M):
    L = si.make_linear(N, K, p, split, seed=3000 + N + K + M)
    c = o.pack_linear_canonical(L.w.numpy(), L.perm.numpy(), L.n_dense, split)
    pk = sp.spense_pack_linear(cuda(L.w), L.w_scale, cuda(L.perm), L.n_dense, _split_id(sp, split), want_canon=True)
    torch.cuda.synchronize()
    for k in ("perm", "sp_val", "sp_meta", "dn"):
        assert np.array_equal(pk.canon[k].cpu().numpy(), c[k]), f"canonical array {k} differs from the oracle"
    body = pk.blob.cpu().numpy()[blob_layout.HEADER:]
    assert np.array_equal(body, blob_layout.expected_linear_body(c, N, K, L.n_dense, split)), "blob body (P3 re-tile) differs"

    x, s_x = si.make_activations(M, K, seed=3000 + M)
    ws = sp.spense_linear_workspace(pk, M)
    y = sp.spense_linear(pk, cuda(x), cuda(s_x), ws)
    y2 = sp.spense_linear(pk, cuda(x), cuda(s_x), ws)
    torch.cuda.synchronize()
    assert sp.spense_device_status() == "SPENSE_OK"
    r = o.linear(x.numpy(), s_x.numpy(), o.unpack_linear_canonical(c), L.w_scale)
    err = np.abs(y.cpu().numpy().astype(np.float64) - r["y"])
    tol = o.tol_gemm(r["absY"])
    assert (err <= tol).all(), f"{(err > tol).sum()} of {err.size} outputs out of tolerance, worst {err.max():.3e}"
    assert torch.equal(y, y2)                                    # fixed-order split-K fix-up: bitwise repeatable
    yb = sp.spense_linear(pk, cuda(x), cuda(s_x), ws, dtype=torch.bfloat16)
    torch.cuda.synchronize()
    assert torch.equal(yb, y.to(torch.bfloat16))                 # bf16 output = RNE of the fp32 output
    # a scalar activation scale (sx_stride 0)
    one = torch.full((1,), 0.5, device="cuda")
    y1 = sp.spense_linear(pk, cuda(x), one, ws)
    torch.cuda.synchronize()
    r1 = o.linear(x.numpy(), np.float32(0.5), o.unpack_linear_canonical(c), L.w_scale)
    assert (np.abs(y1.cpu().numpy().astype(np.float64) - r1["y"]) <= o.tol_gemm(r1["absY"])).all()


@pytest.mark.parametrize("split", ["out", "in"])
def test_linear_one_hot_and_small_integer_exact(sp, split):
    """one-hot activations return a weight column exactly; small-integer operands give sums below 2^24, so the fp32
    result must equal the oracle bit for bit whatever the summation order (SURVEY.md 8c GEMM pins iii, iv)."""
    N, K, M = 512, 512, 24
    n_dense = 256 if split == "out" else 128
    wg, _, wd, x = si.make_small_int_case(K, N, n_dense, M, seed=77) if split == "out" else si.make_small_int_case(N, K, n_dense, M, seed=78)
    w = wg if split == "out" else wd                             # [N, K], sparse region first (identity perm), 2:4 by construction
    c = o.pack_linear_canonical(w.numpy(), None, n_dense, split)
    pk = sp.spense_pack_linear(cuda(w), 1.0, None, n_dense, _split_id(sp, split))
    ws = sp.spense_linear_workspace(pk, M)
    xs = x.clone()
    xs[0] = 0
    xs[0, 5] = 0x38                                              # one-hot row: y[0] = column 5 of W
    one = torch.ones(1, device="cuda")
    y = sp.spense_linear(pk, cuda(xs), one, ws)
    torch.cuda.synchronize()
    r = o.linear(xs.numpy(), np.float32(1.0), o.unpack_linear_canonical(c), 1.0)
    assert np.array_equal(y.cpu().numpy().astype(np.float64), r["y"])
    assert np.array_equal(y[0].cpu().numpy().astype(np.float64), o.e4m3_decode(o.unpack_linear_canonical(c)[:, 5]))


def test_linear_pack_error_paths(sp):
    L = si.make_linear(512, 256, 0.5, "out", seed=5)
    w = L.w.clone()
    pw = L.perm.long()
    w[pw[3], 8:12] = torch.tensor([0x38, 0x38, 0x38, 0], dtype=torch.uint8)      # sparse row 3, group 2: three non-zeros
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_pack_linear(cuda(w), L.w_scale, cuda(L.perm), L.n_dense, sp.SPENSE_SPLIT_OUT)
    assert e.value.code == "SPENSE_ERR_NOT_2_4" and e.value.where[:3] == (0, 3, 2)
    with pytest.raises(o.SpenseOracleError) as eo:
        o.pack_linear_canonical(w.numpy(), L.perm.numpy(), L.n_dense, "out")
    assert eo.value.where[:3] == e.value.where[:3]
    bad = L.perm.clone()
    bad[0] = bad[1]
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_pack_linear(cuda(L.w), L.w_scale, cuda(bad), L.n_dense, sp.SPENSE_SPLIT_OUT)
    assert e.value.code == "SPENSE_ERR_BAD_PERM"
    # a blob of the wrong kind is refused on the device
    pk = sp.spense_pack_linear(cuda(L.w), L.w_scale, cuda(L.perm), L.n_dense, sp.SPENSE_SPLIT_OUT)
    wrong = sp.PackedLinear(512, 256, 256, sp.SPENSE_SPLIT_IN, pk.blob)
    x, s_x = si.make_activations(4, 256, seed=1)
    ws = sp.spense_linear_workspace(pk, 4)
    sp.spense_linear(wrong, cuda(x), cuda(s_x), ws)
    torch.cuda.synchronize()
    assert sp.spense_device_status(clear=True) == "SPENSE_ERR_BAD_BLOB"
    assert sp.spense_device_status() == "SPENSE_OK"


def test_linear_full_size_qwen_projections(sp):
    """The three projections of the Qwen3-32B-shaped layer as stand-alone linears at M = 64 (sampled rows of the oracle)."""
    M = 64
    rng = np.random.default_rng(0)
    for (N, K, split) in ((25600, 5120, "out"), (5120, 25600, "in")):
        L = si.make_linear(N, K, 0.25, split, seed=9000 + N, device="cuda")
        pk = sp.spense_pack_linear(L.w, L.w_scale, L.perm, L.n_dense, _split_id(sp, split))
        x, s_x = si.make_activations(M, K, seed=9000 + M)
        ws = sp.spense_linear_workspace(pk, M)
        y = sp.spense_linear(pk, cuda(x), cuda(s_x), ws)
        torch.cuda.synchronize()
        w = L.w.cpu().numpy()
        perm = L.perm.cpu().numpy().astype(np.int64)
        rows = np.sort(rng.choice(N, 512, replace=False))        # output features (permuted order for the out-split)
        if split == "out":
            wr = w[perm[rows]]
        else:
            wr = w[rows][:, perm]
        wr = np.where((wr & 0x7F) == 0, 0, wr)
        r = o.linear(x.numpy(), s_x.numpy(), wr, L.w_scale)
        err = np.abs(y[:, torch.from_numpy(rows).cuda()].cpu().numpy().astype(np.float64) - r["y"])
        assert (err <= o.tol_gemm(r["absY"])).all(), f"{split}: worst {err.max():.3e}"
