"""-m gpu: spense_gate_up / spense_down / spense_mlp through the C ABI against the CPU oracle.

Bar (BASELINE.json north_star): |gpu - oracle| <= 2e-3 * sum|a*w| + 1e-5 per element, measured
before FP8 re-quantisation (on the fp32 dump of h and on the fp32 y)."""
import numpy as np
import pytest
import torch

import spense_inputs as si
from oracle import spense_oracle as o
from tests.gpu_common import HQ_MISMATCH_BOUND, Case, assert_down_parity, assert_gate_up_parity, cuda

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    from paper_2606_10445_b200 import build, spense
    build.build()
    assert torch.cuda.is_available()
    return spense


def run_gate_up(sp, c, pk, s_h, ws=None):
    ws = ws if ws is not None else sp.spense_workspace(pk, c.M)
    h = torch.full((c.M, c.I), float("nan"), dtype=torch.float32, device="cuda")
    hq = sp.spense_gate_up(pk, cuda(c.x), cuda(c.s_x), cuda(torch.as_tensor(s_h, dtype=torch.float32).reshape(-1)), ws, h_f32=h)
    torch.cuda.synchronize()
    return h.cpu().numpy(), hq.cpu().numpy()


# H, I, p, I_dense, M  -- Tiny is BASELINE.json configs[0]; the rest span several tiles, ragged tails,
# every padding case and both degenerate splits
GEMM_CASES = [
    (256, 1024, 0.25, None, 8),
    (256, 1024, 1.0, None, 8),      # all dense  == the baseline kernel
    (256, 1024, 0.0, None, 8),      # all sparse
    (256, 1024, 0.25, None, 1),
    (256, 1024, 0.25, None, 33),
    (256, 1024, 0.25, None, 64),
    (256, 1024, 0.25, None, 100),
    (256, 1024, 0.25, None, 128),
    (256, 1024, 0.25, None, 200),   # one block of 208 token columns
    (384, 640, None, 128, 16),      # H % 256 == 128
    (128, 384, None, 0, 5),         # I_s % 256 == 128, single half down tile
    (640, 896, None, 384, 48),
    (1024, 4096, 0.25, None, 64),   # enough stages for many spans / split-K partials
    (256, 1024, 0.25, None, 80),    # token columns not a multiple of 32
    (1024, 4096, 0.25, None, 96),
    (1024, 4096, 0.25, None, 112),  # 7 x 16 token columns
    (256, 1024, 0.25, None, 240),   # the widest double-buffered token tile
    (1024, 4096, 0.25, None, 241),  # 241..256 tokens: one 256-column tile, single accumulator buffer, ragged
    (256, 1024, 0.25, None, 256),   # the same, full
    (1024, 4096, 0.25, None, 257),  # gate_up: two blocks of 144 columns; down: three of 96
    (1024, 4096, 0.25, None, 300),  # gate_up two blocks of 160, down three of 112 (ragged last one)
    (640, 896, None, 384, 513),     # three blocks of 176, the last one ragged
]


@pytest.mark.parametrize("H,I,p,I_d,M", GEMM_CASES)
def test_gate_up_down_mlp_parity(sp, H, I, p, I_d, M):
    c = Case(H, I, p if p is not None else 0.0, M, seed=1000 + H + I + M, I_dense=I_d)
    pk = c.pack_gpu(sp)
    s_h = c.default_s_h()
    r = c.oracle_gate_up(s_h)
    ws = sp.spense_workspace(pk, M)
    h_gpu, hq_gpu = run_gate_up(sp, c, pk, s_h, ws)
    assert not np.isnan(h_gpu).any()
    frac = assert_gate_up_parity(r, h_gpu, hq_gpu, s_h, "gate_up")
    assert frac < HQ_MISMATCH_BOUND, f"too many Hq bytes differ from the oracle: {frac}"
    # down, fed the GPU's own Hq bytes (strict tolerance)
    sh_dev = cuda(torch.from_numpy(s_h))
    y = sp.spense_down(pk, cuda(torch.from_numpy(hq_gpu)), sh_dev, ws)
    torch.cuda.synchronize()
    assert_down_parity(y.cpu().numpy(), hq_gpu, s_h, c.wd, c.L.w_scale[2], "down")
    # chained spense_mlp == gate_up followed by down, bit for bit; and repeated runs are bitwise identical
    y2 = sp.spense_mlp(pk, cuda(c.x), cuda(c.s_x), sh_dev, ws)
    y3 = sp.spense_mlp(pk, cuda(c.x), cuda(c.s_x), sh_dev, ws)
    torch.cuda.synchronize()
    assert torch.equal(y, y2) and torch.equal(y2, y3)
    # bf16 output = RNE rounding of the fp32 output
    yb = sp.spense_mlp(pk, cuda(c.x), cuda(c.s_x), sh_dev, ws, dtype=torch.bfloat16)
    torch.cuda.synchronize()
    assert torch.equal(yb, y.to(torch.bfloat16))
    # workspace control words: every launch advanced the epoch and left the finished-CTA count at zero
    ctrl = ws[:8].view(torch.int32).cpu()
    assert int(ctrl[0]) > 0 and int(ctrl[1]) == 0


def _random_cases(n, seed):
    """seeded random shapes: H, I multiples of 128, any dense count (multiple of 128), any token count up to 300 -- spans of a
    single stage, tiles shared by three and more spans, half tiles, every token-column padding"""
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(n):
        H = 128 * int(rng.integers(1, 9))
        I = 128 * int(rng.integers(1, 17))
        I_d = 128 * int(rng.integers(0, I // 128 + 1))
        M = int(rng.choice([1, 2, 7, 15, 16, 17, 31, 33, 63, 65, 97, 113, 129, 191, 239, 241, 255, 257, 299]))
        out.append((H, I, I_d, M))
    return out


@pytest.mark.parametrize("H,I,I_d,M", _random_cases(24, seed=20261105))
def test_random_shapes_parity(sp, H, I, I_d, M):
    c = Case(H, I, 0.0, M, seed=4000 + H + 3 * I + 7 * I_d + M, I_dense=I_d)
    pk = c.pack_gpu(sp)
    s_h = c.default_s_h()
    r = c.oracle_gate_up(s_h)
    ws = sp.spense_workspace(pk, M)
    h_gpu, hq_gpu = run_gate_up(sp, c, pk, s_h, ws)
    frac = assert_gate_up_parity(r, h_gpu, hq_gpu, s_h, f"random {H}x{I} I_d={I_d} M={M}")
    assert frac < max(HQ_MISMATCH_BOUND, 2.0 / hq_gpu.size), frac      # tiny cases: one byte is already more than 1e-4
    sh_dev = cuda(torch.from_numpy(s_h))
    y = sp.spense_down(pk, cuda(torch.from_numpy(hq_gpu)), sh_dev, ws)
    y2 = sp.spense_mlp(pk, cuda(c.x), cuda(c.s_x), sh_dev, ws)
    torch.cuda.synchronize()
    assert_down_parity(y.cpu().numpy(), hq_gpu, s_h, c.wd, c.L.w_scale[2], "down")
    assert torch.equal(y, y2)
    assert sp.spense_device_status() == "SPENSE_OK"


def test_changing_token_counts_on_one_workspace(sp):
    """300 back-to-back layers on ONE workspace with the token count changing every call (every launch geometry: one block,
    the single-buffer tile, several blocks, static and dynamic requant): the epoch-valued flags need no reset in between,
    no launch times out, and a token count seen again gives the same bits."""
    c = Case(640, 896, 0.43, 8, seed=123)
    pk = c.pack_gpu(sp)
    ws = sp.spense_workspace(pk, 1024)
    rng = np.random.default_rng(7)
    seen = {}
    for it in range(300):
        M = int(rng.choice([1, 5, 16, 48, 64, 100, 128, 200, 240, 250, 256, 300, 481, 700]))
        x, s_x = si.make_activations(M, 640, seed=M)
        sh = torch.full((M,), 0.05, device="cuda")
        if it % 3 == 2:
            y, _, _, _ = sp.spense_mlp_dyn(pk, cuda(x), cuda(s_x), ws)
            key = ("dyn", M)
        else:
            y = sp.spense_mlp(pk, cuda(x), cuda(s_x), sh, ws, next_layer=pk)
            key = ("static", M)
        if key in seen:
            assert torch.equal(seen[key], y), key
        seen[key] = y
    torch.cuda.synchronize()
    assert sp.spense_device_status() == "SPENSE_OK"


def test_scalar_requant_scale(sp):
    c = Case(256, 1024, 0.25, 8, seed=77)
    pk = c.pack_gpu(sp)
    s_h = np.float32(np.abs(c.oracle_gate_up(1.0)["h"]).max() / 448)
    r = c.oracle_gate_up(s_h)
    h_gpu, hq_gpu = run_gate_up(sp, c, pk, np.array([s_h], np.float32))
    assert_gate_up_parity(r, h_gpu, hq_gpu, s_h, "scalar s_h")


def test_one_hot_tokens_return_weight_columns_exactly(sp):
    """A one-hot activation row makes g = one column of W~gate: exact in fp32 whatever the MMA order.
    A wrong nibble order / lane mapping / swizzle shows up here as a permuted or zeroed column."""
    H, I = 512, 1024
    L = si.make_layer(H, I, 0.5, seed=21)
    ks = [0, 1, 2, 3, 5, 31, 32, 63, 64, 127, 128, 255, 256, 300, 511, 17]
    x = torch.zeros(len(ks), H, dtype=torch.uint8)
    for r_, k in enumerate(ks):
        x[r_, k] = 0x38
    c = Case(H, I, 0.5, len(ks), seed=21, layer=L, x=x, s_x=torch.ones(len(ks)))
    pk = c.pack_gpu(sp)
    # u = g for identical weights is not available; instead read h = silu(g) * u against the oracle with
    # tolerance ZERO on the accumulators: g and u are single products, so h is deterministic up to expf
    r = c.oracle_gate_up(1.0)
    h_gpu, _ = run_gate_up(sp, c, pk, np.array([1.0], np.float32))
    assert np.allclose(h_gpu, r["h"], rtol=2e-6, atol=1e-30)
    nz_ref = r["h"] != 0
    assert np.array_equal(h_gpu != 0, nz_ref)           # exactly the same support: no column is dropped or moved
    # down: one-hot Hq rows select columns of W~down exactly
    hq = torch.zeros(len(ks), I, dtype=torch.uint8)
    cols = [0, 1, 2, 3, 4, 7, 64, 127, 128, 255, 256, 511, 512, 700, 1000, 1023]
    for r_, k in enumerate(cols):
        hq[r_, k] = 0x38
    ws = sp.spense_workspace(pk, len(ks))
    y = sp.spense_down(pk, cuda(hq), cuda(torch.ones(1)), ws).cpu().numpy()
    want = (o.e4m3_decode(c.wd[:, cols]).T * np.float32(L.w_scale[2])).astype(np.float32)
    assert np.array_equal(y, want)


def test_small_integer_inputs_are_exact(sp):
    """Small-integer weights and activations: every partial sum is an integer < 2^24, so the fp32
    result must equal the oracle EXACTLY in any accumulation order (split-K partials included)."""
    H, I, I_d, M = 1024, 2048, 512, 32
    wg, wu, wd, x = si.make_small_int_case(H, I, I_d, M, seed=4)
    pk = sp.spense_pack(cuda(wg), cuda(wu), cuda(wd), (1.0, 1.0, 1.0), None, I_d)
    ws = sp.spense_workspace(pk, M)
    hq = x.new_zeros(M, I)
    hq[:, ::3] = 0x38
    hq[:, 1::5] = 0xC0
    y = sp.spense_down(pk, cuda(hq), cuda(torch.ones(1)), ws).cpu().numpy()
    ref = o.down(hq.numpy(), 1.0, np.where((wd.numpy() & 0x7F) == 0, 0, wd.numpy()), 1.0)
    assert np.array_equal(y.astype(np.float64), ref["y"])
    # gate_up accumulators are exact too; h goes through expf, so compare with a tight relative bound
    r = o.gate_up(x.numpy(), np.ones(M), wg.numpy(), wu.numpy(), 1.0, 1.0, 1.0)
    h = torch.empty(M, I, dtype=torch.float32, device="cuda")
    sp.spense_gate_up(pk, cuda(x), cuda(torch.ones(M)), cuda(torch.ones(1)), ws, h_f32=h)
    assert np.allclose(h.cpu().numpy(), r["h"], rtol=3e-6, atol=1e-6)


def test_dense_fraction_invariance_on_gpu(sp):
    L0 = si.make_layer(512, 1024, 0.0, seed=31, all_2_4=True)
    x, sx = si.make_activations(24, 512, seed=31)
    ys = []
    for I_d in (0, 128, 512, 1024):
        pk = sp.spense_pack(cuda(L0.wgate), cuda(L0.wup), cuda(L0.wdown), L0.w_scale, None, I_d)
        ws = sp.spense_workspace(pk, 24)
        h = torch.empty(24, 1024, dtype=torch.float32, device="cuda")
        sp.spense_gate_up(pk, cuda(x), cuda(sx), cuda(torch.full((1,), 0.01)), ws, h_f32=h)
        ys.append(h.cpu().numpy())
    ref = o.gate_up(x.numpy(), sx.numpy(), *[np.where((w.numpy() & 0x7F) == 0, 0, w.numpy()) for w in (L0.wgate, L0.wup)],
                    L0.w_scale[0], L0.w_scale[1], 0.01)
    for y in ys:
        assert (np.abs(y - ref["h"]) <= o.tol_glu(ref)).all()


def test_gemm_argument_errors(sp):
    c = Case(256, 1024, 0.25, 8, seed=3)
    pk = c.pack_gpu(sp)
    ws = sp.spense_workspace(pk, 8)
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_gate_up(pk, cuda(c.x), cuda(c.s_x), cuda(torch.ones(1)), ws[:1024])
    assert e.value.code == "SPENSE_ERR_BUFFER_TOO_SMALL"
    # a blob whose header does not match the stated shape is detected ON THE DEVICE (the GEMM calls never read device
    # memory on the host): the launch runs, spense_device_status reports it, later calls refuse until it is cleared
    assert sp.spense_device_status() == "SPENSE_OK"
    bad = sp.PackedLayer(256, 1024, 128, pk.blob)       # header says I_dense = 256
    sp.spense_gate_up(bad, cuda(c.x), cuda(c.s_x), cuda(torch.ones(1)), ws)
    torch.cuda.synchronize()
    assert sp.spense_device_status() == "SPENSE_ERR_BAD_BLOB"
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_gate_up(pk, cuda(c.x), cuda(c.s_x), cuda(torch.ones(1)), ws)
    assert e.value.code == "SPENSE_ERR_BAD_BLOB"
    assert sp.spense_device_status(clear=True) == "SPENSE_ERR_BAD_BLOB" and sp.spense_device_status() == "SPENSE_OK"
    sp.spense_gate_up(pk, cuda(c.x), cuda(c.s_x), cuda(torch.ones(1)), ws)
    torch.cuda.synchronize()
    assert sp.spense_device_status() == "SPENSE_OK"


@pytest.mark.parametrize("M", [8, 200])
def test_first_call_on_a_fresh_blob_inside_stream_capture(sp, M):
    """The GEMM calls neither synchronise nor read the blob header on the host (weight scales are read by the kernels):
    the very first spense_mlp on a freshly packed blob can be captured into a CUDA graph, and a blob rewritten in place
    at the same address (new weights, new scales) is picked up by the replay."""
    c = Case(256, 1024, 0.25, M, seed=4100 + M)
    pk = c.pack_gpu(sp)
    s_h = c.default_s_h()
    ws = sp.spense_workspace(pk, M)
    xd, sxd, shd = cuda(c.x), cuda(c.s_x), cuda(torch.from_numpy(s_h))
    hq = torch.zeros(M, c.I, dtype=torch.uint8, device="cuda")
    y = torch.zeros(M, c.H, dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            sp.spense_mlp(pk, xd, sxd, shd, ws, hq_scratch=hq, y=y)      # first use of this blob, of this workspace
    torch.cuda.current_stream().wait_stream(s)
    g.replay()
    torch.cuda.synchronize()
    r = c.oracle_gate_up(s_h)
    assert (hq.cpu().numpy() != r["hq"]).mean() < HQ_MISMATCH_BOUND
    assert_down_parity(y.cpu().numpy(), hq.cpu().numpy(), s_h, c.wd, c.L.w_scale[2], "captured first call")
    # same address, another layer with other scales: the replay must use the NEW header
    c2 = Case(256, 1024, 0.25, M, seed=4200 + M, x=c.x, s_x=c.s_x)
    pk2 = c2.pack_gpu(sp)
    assert c2.L.w_scale[2] != c.L.w_scale[2]
    pk.blob.copy_(pk2.blob)
    g.replay()
    torch.cuda.synchronize()
    assert_down_parity(y.cpu().numpy(), hq.cpu().numpy(), s_h, c2.wd, c2.L.w_scale[2], "replay after the blob was replaced in place")


def test_first_call_in_a_fresh_process_is_capturable(sp, tmp_path):
    """A process that loads a pre-packed blob and never calls spense_pack: its first spense_mlp, captured under torch's
    default global capture mode, must not need any set-up that is illegal during capture (spense_workspace_init did it).
    The child's replayed hq and y equal this process's eager result bit for bit."""
    import os
    import subprocess
    import sys
    M = 40
    c = Case(256, 1024, 0.25, M, seed=4300)
    pk = c.pack_gpu(sp)
    s_h = torch.from_numpy(c.default_s_h())
    ws = sp.spense_workspace(pk, M)
    hq = torch.zeros(M, c.I, dtype=torch.uint8, device="cuda")
    y = sp.spense_mlp(pk, cuda(c.x), cuda(c.s_x), cuda(s_h), ws, hq_scratch=hq)
    torch.cuda.synchronize()
    d = str(tmp_path)
    torch.save(torch.tensor([c.H, c.I, c.I_d, M]), f"{d}/meta.pt")
    torch.save(pk.blob.cpu(), f"{d}/blob.pt")
    for n, t in (("x", c.x), ("sx", c.s_x), ("sh", s_h)):
        torch.save(t, f"{d}/{n}.pt")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-m", "tests.capture_child", d], cwd=root, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    out = torch.load(f"{d}/out.pt")
    assert torch.equal(out["hq"], hq.cpu()) and torch.equal(out["y"], y.cpu())


def test_mlp_host_buffers_equal_device_call(sp):
    """spense_mlp_host (HOST pinned x, scales and y; copies inside the call) == spense_mlp on device buffers."""
    H, I, p, M = 640, 896, 0.43, 48
    c = Case(H, I, p, M, seed=123)
    pk = c.pack_gpu(sp)
    s_h = c.default_s_h()
    ws = sp.spense_workspace(pk, M)
    for dtype in (torch.float32, torch.bfloat16):
        y_dev = sp.spense_mlp(pk, cuda(c.x), cuda(c.s_x), cuda(torch.from_numpy(s_h)), ws, dtype=dtype)
        hx, hsx, hsh = c.x.pin_memory(), c.s_x.pin_memory(), torch.from_numpy(s_h).pin_memory()
        hy = torch.empty(M, H, dtype=dtype).pin_memory()
        staging = dict(d_x=torch.empty(M, H, dtype=torch.uint8, device="cuda"), d_scales=torch.empty(2 * M, device="cuda"),
                       d_hq=torch.empty(M, I, dtype=torch.uint8, device="cuda"), d_y=torch.empty(M, H, dtype=dtype, device="cuda"))
        sp.spense_mlp_host(pk, hx, hsx, hsh, hy, staging, ws)
        assert torch.equal(hy, y_dev.cpu())
        hy.zero_()
        sp.spense_mlp_stack_host([pk, pk, pk], hx, hsx, hsh, hy, staging, ws)     # every layer reads x: the last y is the same
        assert torch.equal(hy, y_dev.cpu())
