"""-m gpu: spense_mlp_dyn (dynamic per-token requant) through the C ABI against the oracle.

Floating point decides bytes here (s_h, then Hq), so both sides take the decision in fp32 from the SAME h:
s_h must be fp32(max|h_gpu|) / 448 bit for bit, Hq must be the oracle's E4M3 encoder applied to h_gpu / s_h,
and y is checked against the oracle's down fed those bytes and that scale.  h itself is held to tol_glu."""
import numpy as np
import pytest
import torch

import spense_inputs as si
from oracle import spense_oracle as o
from tests.gpu_common import HQ_MISMATCH_BOUND, Case, assert_down_parity, cuda

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    from paper_2606_10445_b200 import build, spense
    build.build()
    assert torch.cuda.is_available()
    return spense


CASES = [(256, 1024, 0.25, 8), (256, 1024, 0.25, 1), (256, 1024, 0.0, 33), (256, 1024, 1.0, 64),
         (256, 1024, 0.25, 200), (1024, 4096, 0.25, 64), (640, 896, 0.43, 48)]


@pytest.mark.parametrize("H,I,p,M", CASES)
def test_mlp_dyn_parity(sp, H, I, p, M):
    c = Case(H, I, p, M, seed=7000 + H + I + M)
    if M > 2:                                            # an all-zero token: scale 1, zero bytes, zero y
        c.x = c.x.clone()
        c.x[1] = 0
    if M > 4:                                            # a token whose h is ~1e-37: s_h = amax / 448 is below 2^-128 and has
        c.s_x = c.s_x.clone()                            # no finite fp32 reciprocal (the quotients must still be IEEE's)
        c.s_x[3] = 1e-20
    pk = c.pack_gpu(sp)
    ws = sp.spense_workspace(pk, M)
    ref = o.mlp_dynamic(c.x.numpy(), c.s_x.numpy(), c.wg, c.wu, c.wd, c.L.w_scale)
    if M > 4:                                            # h ~ s_x^2: steer the row's scale into (2^-138, 2^-129)
        for _ in range(4):
            if 2.0 ** -138 < ref["s_h"][3] < 2.0 ** -129:
                break
            c.s_x[3] *= float(np.sqrt(2.0 ** -133 / max(float(ref["s_h"][3]), 1e-45)))
            ref = o.mlp_dynamic(c.x.numpy(), c.s_x.numpy(), c.wg, c.wu, c.wd, c.L.w_scale)
        assert 2.0 ** -138 < ref["s_h"][3] < 2.0 ** -129, ref["s_h"][3]
    y, s_h, hq, h = sp.spense_mlp_dyn(pk, cuda(c.x), cuda(c.s_x), ws)
    torch.cuda.synchronize()
    h_gpu, hq_gpu, sh_gpu, y_gpu = h.cpu().numpy(), hq.cpu().numpy(), s_h.cpu().numpy(), y.cpu().numpy()
    # h against the oracle
    err = np.abs(h_gpu.astype(np.float64) - ref["h"])
    tol = o.tol_glu(ref)
    assert (err <= tol).all(), f"h: worst {err.max():.3e}"
    # the scale: fp32 max of the kernel's own h, IEEE division by 448
    assert np.array_equal(sh_gpu, o.requant_scale_from_h(h_gpu))
    assert np.allclose(sh_gpu, ref["s_h"], rtol=2e-3, atol=0)
    # the bytes: the oracle's encoder on the kernel's own h and scale
    own = o.e4m3_encode((h_gpu / sh_gpu[:, None]).astype(np.float32))
    assert np.array_equal(hq_gpu, own)
    live = np.abs(h_gpu).max(axis=1) > 0
    assert ((hq_gpu[live] & 0x7F).max(axis=1) == 0x7E).all()       # the row maximum lands on +-448
    if M > 4:
        assert 0 < sh_gpu[3] < 2.0 ** -128, sh_gpu[3]
        assert (hq_gpu[3] & 0x7F).max() == 0x7E and not ((hq_gpu[3] & 0x7F) == 0x7F).any()
        # the static path given that tiny scale divides by it in its epilogue: same bytes
        hq_s = sp.spense_gate_up(pk, cuda(c.x), cuda(c.s_x), s_h, ws)
        torch.cuda.synchronize()
        assert torch.equal(hq_s, hq)
    if M > 2:
        assert sh_gpu[1] == 1.0 and not hq_gpu[1].any() and not y_gpu[1].any()
    diff = (hq_gpu != ref["hq"]).mean()
    print(f"[hq-mismatch] dynamic requant {H}x{I} p={p} M={M}: {diff:.3e}")
    assert diff < 4 * HQ_MISMATCH_BOUND, diff             # a scale one ulp off moves a few more rounding boundaries
    # y against the oracle's down fed the GPU's own bytes and scale
    assert_down_parity(y_gpu, hq_gpu, sh_gpu, c.wd, c.L.w_scale[2], "down after dynamic requant")
    # reproducible, and bf16 = RNE of fp32
    y2, s2, hq2, _ = sp.spense_mlp_dyn(pk, cuda(c.x), cuda(c.s_x), ws)
    yb, _, _, _ = sp.spense_mlp_dyn(pk, cuda(c.x), cuda(c.s_x), ws, dtype=torch.bfloat16)
    torch.cuda.synchronize()
    assert torch.equal(y, y2) and torch.equal(s_h, s2) and torch.equal(hq, hq2)
    assert torch.equal(yb, y.to(torch.bfloat16))
    # the static path with the same scale gives the same bytes and the same y
    y3 = sp.spense_mlp(pk, cuda(c.x), cuda(c.s_x), s_h, ws)
    torch.cuda.synchronize()
    assert torch.equal(y3, y)
