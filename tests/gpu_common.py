"""Helpers shared by the -m gpu parity tests: build a synthetic layer, pack it through the C ABI,
run the oracle on the same bytes."""
import numpy as np
import torch

import spense_inputs as si
from oracle import spense_oracle as o


# Share of Hq bytes that may differ from the ORACLE's Hq: the kernel's fp32 h differs from the oracle's float64 h in the
# last bits (accumulation order, hardware exp2 / rcp in SiLU), so a value sitting on an E4M3 rounding boundary can land
# on the neighbouring byte.  Measured on B200 over all 56 cases of the GPU suite (each prints an [hq-mismatch] line):
# 0 to 9e-6 at full size, worst 2.96e-5 (one byte of a 33 792-byte case); the bound is ~3x the worst, which is also what
# SURVEY.md 8c-O6 expected ("<~ 1e-4").  The dynamic path (its scale can be one ulp off) measured at most 9.4e-6 and is allowed 4x the bound.
HQ_MISMATCH_BOUND = 1e-4


def cuda(t):
    return t.cuda().contiguous()


class Case:
    """One synthetic layer + activations, on CPU (numpy for the oracle) and on the GPU."""

    def __init__(self, H, I, p, M, seed, I_dense=None, layer=None, x=None, s_x=None):
        self.L = layer if layer is not None else si.make_layer(H, I, p, seed, I_dense=I_dense)
        self.H, self.I, self.I_d, self.M = H, I, self.L.I_dense, M
        if x is None:
            x, s_x = si.make_activations(M, H, seed)
        self.x, self.s_x = x, s_x
        self.canon = o.pack_canonical(self.L.wgate.numpy(), self.L.wup.numpy(), self.L.wdown.numpy(),
                                      self.L.perm.numpy(), self.I_d)
        self.wg, self.wu, self.wd = o.unpack_canonical(self.canon)

    def pack_gpu(self, sp, want_canon=False):
        return sp.spense_pack(cuda(self.L.wgate), cuda(self.L.wup), cuda(self.L.wdown), self.L.w_scale,
                              cuda(self.L.perm), self.I_d, want_canon=want_canon)

    def oracle_gate_up(self, s_h):
        return o.gate_up(self.x.numpy(), self.s_x.numpy(), self.wg, self.wu, self.L.w_scale[0], self.L.w_scale[1], s_h)

    def default_s_h(self):
        r = self.oracle_gate_up(1.0)
        return o.requant_scale_from_h(r["h"])


def assert_gate_up_parity(r, h_gpu, hq_gpu, s_h, label=""):
    """fp32 dump of h against the oracle within tol_glu; Hq bytes: equal to the oracle's except where
    the fp32 h differs enough to cross a rounding boundary (at most one E4M3 step, rare)."""
    tol = o.tol_glu(r)
    err = np.abs(h_gpu.astype(np.float64) - r["h"])
    bad = err > tol
    assert not bad.any(), f"{label}: {bad.sum()} of {bad.size} h values out of tolerance; worst {err.max():.3e} " \
                          f"(tol there {tol.flat[err.argmax()]:.3e}) at {np.unravel_index(err.argmax(), err.shape)}"
    # the GPU's Hq must be the E4M3 rounding of ITS OWN h
    sh = np.broadcast_to(np.asarray(s_h, np.float32).reshape(-1, 1), (h_gpu.shape[0], 1))
    own = o.e4m3_encode((h_gpu.astype(np.float32) / sh).astype(np.float32))
    assert np.array_equal(own, hq_gpu), f"{label}: Hq is not the RNE E4M3 cast of the kernel's own h"
    diff = hq_gpu != r["hq"]
    frac = diff.mean()
    print(f"[hq-mismatch] {label}: {frac:.3e} of {diff.size} bytes")
    if diff.any():
        a, b = o.e4m3_decode(hq_gpu[diff]), o.e4m3_decode(r["hq"][diff])
        # neighbours on the E4M3 grid: |a-b| <= one step of the larger magnitude (2^-3 relative), or both tiny
        step = np.maximum(np.abs(a), np.abs(b)) * 0.126 + 2.0 ** -9
        assert (np.abs(a - b) <= step).all(), f"{label}: an Hq byte differs by more than one E4M3 step"
    return frac


def assert_down_parity(y_gpu, hq_bytes, s_h, wd, s_wd, label=""):
    r = o.down(hq_bytes, s_h, wd, s_wd)
    err = np.abs(y_gpu.astype(np.float64) - r["y"])
    tol = o.tol_gemm(r["absY"])
    bad = err > tol
    assert not bad.any(), f"{label}: {bad.sum()} of {bad.size} y values out of tolerance; worst {err.max():.3e} " \
                          f"(tol there {tol.flat[err.argmax()]:.3e}) at {np.unravel_index(err.argmax(), err.shape)}"
    return (err / tol).max()
