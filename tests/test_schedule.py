"""Host logic of the stream-K schedule (no GPU): spans partition the linear stage sequence, are balanced in the
library's cost model, and the fused variant never leaves a gate_up tile to three spans where it can avoid it."""
import ctypes

import numpy as np
import pytest


@pytest.fixture(scope="module")
def lib():
    from paper_2606_10445_b200 import build, spense
    build.build()
    L = ctypes.CDLL(spense.LIB_PATH)
    L.spense_debug_schedule.argtypes = [ctypes.POINTER(spense.Shape), ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                        ctypes.c_int32, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32)]
    L.spense_debug_schedule.restype = ctypes.c_int
    return L, spense


def schedule(lib, H, I, I_d, M, mode, fused=0, sms=148):
    L, sp = lib
    sb = (ctypes.c_int32 * 161)()
    info = (ctypes.c_int32 * 4)()
    n = L.spense_debug_schedule(ctypes.byref(sp.Shape(H, I, I_d)), M, mode, fused, sms, sb, info)
    assert n > 0, n
    return np.array(sb[:n + 1]), list(info)


def stage_layout(H, I, I_d, mode, nb):
    """stage counts per tile and bytes per stage, written out from the blob layout"""
    I_s = I - I_d
    if mode == 0:
        tiles = [("s", -(-H // 256))] * ((I_s // 128) * nb) + [("d", H // 128)] * ((I_d // 128) * nb)
        return [[40960] * n if k == "s" else [32768] * n for k, n in tiles]
    per = [40960] * (-(-I_s // 256)) + [32768] * (I_d // 128)
    return [per] * (-(-H // 256) * nb)


QWEN = (5120, 25600, 6400)
SEED0 = (5120, 27648, 0)


@pytest.mark.parametrize("shape", [QWEN, SEED0, (5120, 27648, 27648), (256, 1024, 256), (640, 896, 384)])
@pytest.mark.parametrize("M", [1, 64, 128, 200, 1000])
@pytest.mark.parametrize("mode", [0, 1])
def test_spans_partition_the_stage_sequence(lib, shape, M, mode):
    sb, (total, par, n_pad, ring) = schedule(lib, *shape, M, mode)
    tiles = stage_layout(*shape, mode, 1)
    assert total == sum(len(t) for t in tiles)
    nb = 1 if M <= 128 else -(-M // 128)
    # more than 128 tokens: `par` blocks of 128 side by side in one launch, each with 148 // par spans of the same schedule
    assert 1 <= par <= min(nb, 32) and (par == 1) == (nb == 1) and n_pad == (min(128, -(-M // 16) * 16))
    assert sb[0] == 0 and sb[-1] == total and (np.diff(sb) >= 1).all()          # every CTA owns at least one stage
    assert len(sb) - 1 <= 148 // par and 2 <= ring <= 8
    rounds = -(-nb // par)
    assert nb / (rounds * par) * (par * (148 // par) / 148) >= 0.8              # the split keeps most SMs busy
    assert ring * (40960 + 2 * n_pad * 128) + 1024 + 256 + 20 * n_pad <= 232448   # the ring fits the opt-in smem


@pytest.mark.parametrize("M", [1, 64, 128])
@pytest.mark.parametrize("mode", [0, 1])
def test_spans_are_balanced_in_bytes(lib, M, mode):
    sb, (total, nb, n_pad, ring) = schedule(lib, *QWEN, M, mode)
    b = np.concatenate([np.array(t) for t in stage_layout(*QWEN, mode, nb)])
    per_span = np.add.reduceat(b, sb[:-1])
    # the cost model is bytes + a fixed part per stage: spans stay within one stage of each other in bytes
    assert per_span.max() - per_span.min() <= 2 * 40960 + 0.12 * per_span.mean()


def spans_per_tile(sb, tiles):
    first = np.cumsum([0] + [len(t) for t in tiles])
    return [int(np.searchsorted(sb, first[t + 1], "left") - np.searchsorted(sb, first[t], "right") + 1) for t in range(len(tiles))]


def test_fused_gate_up_has_no_three_way_tiles_and_down_balances_the_sum(lib):
    H, I, I_d = QWEN
    tiles = stage_layout(H, I, I_d, 0, 1)
    plain, _ = schedule(lib, H, I, I_d, 64, 0, fused=0)
    fused, _ = schedule(lib, H, I, I_d, 64, 0, fused=1)
    assert max(spans_per_tile(plain, tiles)) == 3              # a 40-stage dense tile is longer than a ~36-stage span
    assert max(spans_per_tile(fused, tiles)) == 2
    assert np.abs(fused - plain).max() <= 4                    # boundaries are only nudged
    # down spans of the fused schedule make up for gate_up spans of unequal cost: the per-CTA byte sum is level
    fd, _ = schedule(lib, H, I, I_d, 64, 1, fused=1)
    bg = np.concatenate([np.array(t) for t in tiles])
    bd = np.concatenate([np.array(t) for t in stage_layout(H, I, I_d, 1, 1)])
    tot = np.add.reduceat(bg, fused[:-1]) + np.add.reduceat(bd, fd[:-1])
    assert tot.max() - tot.min() <= 3 * 40960 + 0.06 * tot.mean()


def test_fewer_sms_and_tiny_shapes(lib):
    sb, (total, nb, n_pad, ring) = schedule(lib, 128, 128, 0, 8, 0, sms=148)
    assert total == 1 and len(sb) == 2                          # one stage: one span
    sb, _ = schedule(lib, *QWEN, 64, 1, sms=20)
    assert len(sb) == 21
    L, sp = lib
    sbuf = (ctypes.c_int32 * 161)()
    assert L.spense_debug_schedule(ctypes.byref(sp.Shape(100, 128, 0)), 8, 0, 0, 148, sbuf, None) == -3   # SPENSE_ERR_SHAPE
    assert L.spense_debug_schedule(ctypes.byref(sp.Shape(128, 128, 0)), 0, 0, 0, 148, sbuf, None) == -1   # SPENSE_ERR_ARG
