"""Host logic of the launch geometry and the stream-K schedule (no GPU): token blocks, spans that partition the
linear stage sequence, balance in the library's cost model, the shared-memory ring that must fit."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def sp():
    from paper_2606_10445_b200 import build, spense
    build.build()
    return spense


def stage_layout(H, I, I_d, mode):
    """stage counts per pair tile and bytes per stage, written out from the blob layout"""
    I_s = I - I_d
    if mode == 0:
        tiles = [("s", -(-H // 256))] * (I_s // 128) + [("d", H // 128)] * (I_d // 128)
        return [[40960] * n if k == "s" else [32768] * n for k, n in tiles]
    per = [40960] * (-(-I_s // 256)) + [32768] * (I_d // 128)
    return [per] * (-(-H // 256))


QWEN = (5120, 25600, 6400)
SEED0 = (5120, 27648, 0)


@pytest.mark.parametrize("shape", [QWEN, SEED0, (5120, 27648, 27648), (256, 1024, 256), (640, 896, 384)])
@pytest.mark.parametrize("M", [1, 48, 49, 64, 112, 113, 128, 200, 240, 256, 1000, 2048, 8192])
@pytest.mark.parametrize("mode", [0, 1])
def test_spans_partition_the_stage_sequence(sp, shape, M, mode):
    sb, info = sp.spense_schedule(*shape, M, mode)
    sb = np.array(sb)
    tiles = stage_layout(*shape, mode)
    assert info["stages"] == sum(len(t) for t in tiles)
    assert sb[0] == 0 and sb[-1] == info["stages"] and (np.diff(sb) >= 1).all()          # every span owns at least one stage
    n_pad, nb, par, ring, cps = info["n_pad"], info["blocks"], info["blocks_per_launch"], info["ring"], info["ctas_per_span"]
    assert n_pad % 16 == 0 and nb * n_pad >= M > (nb - 1) * n_pad                         # the blocks cover the tokens, none is empty
    # CTA pairs: one block of at most 256 tokens (241..256: one 256-column tile with a single accumulator buffer), else
    # blocks of at most 240 tokens, `par` blocks side by side with 74 // par spans each
    assert cps == 2 and n_pad <= (256 if M <= 256 else 240) and nb == (1 if M <= 256 else max(-(-M // 240), 3 if mode == 1 else 2)) and 1 <= par <= min(nb, 37)
    if nb == 1:
        assert n_pad == -(-M // 16) * 16
    assert len(sb) - 1 <= 74 // par
    rounds = -(-nb // par)
    assert nb / (rounds * par) * (par * (74 // par) / 74) >= 0.8                      # the split keeps most SMs busy
    slot = 20480 + (n_pad // 2) * 256                                                 # one operand + half of the token tile
    assert 2 <= ring <= 8 and ring * slot + 1024 + 256 + 20 * n_pad <= 232448             # the ring fits the opt-in smem
    assert par * (len(sb) - 1) * cps <= 148                                                # all CTAs of a launch are resident


@pytest.mark.parametrize("M", [1, 64, 112, 128, 256])
@pytest.mark.parametrize("mode", [0, 1])
def test_weight_streaming_spans_are_balanced_in_bytes(sp, M, mode):
    sb, info = sp.spense_schedule(*QWEN, M, mode)
    b = np.concatenate([np.array(t) for t in stage_layout(*QWEN, mode)])
    per_span = np.add.reduceat(b, np.array(sb[:-1]))
    # the cost model is bytes + a fixed part per stage: spans stay within one stage of each other in bytes
    assert per_span.max() - per_span.min() <= 2 * 40960 + 0.12 * per_span.mean()


@pytest.mark.parametrize("M", [2048, 8192])
def test_prefill_spans_are_balanced_in_stages(sp, M):
    # tensor-paced (3 or more token blocks): a sparse stage (K 256) and a dense one (K 128) issue the same four MMAs,
    # so spans hold equal stage counts
    for mode in (0, 1):
        sb, info = sp.spense_schedule(*QWEN, M, mode)
        n = np.diff(np.array(sb))
        assert n.max() - n.min() <= 1


def test_many_blocks_run_as_few_launches(sp):
    # 35 token blocks (M = 8192): every launch streams all weights again, so the plan takes as many blocks per launch as
    # the activation working set allows instead of the split that merely wastes no CTA pair (one or two blocks)
    _, info = sp.spense_schedule(*QWEN, 8192, 0)
    assert info["blocks"] == 35 and info["blocks_per_launch"] == 12
    _, info = sp.spense_schedule(*QWEN, 8192, 1)
    assert info["blocks"] == 35 and info["blocks_per_launch"] == 9           # 9 x 240 x 25600 B of Hq stay below 64 MB
    _, info = sp.spense_schedule(*QWEN, 2048, 0)
    assert info["blocks"] == 9 and info["blocks_per_launch"] == 9


def test_fewer_sms_and_tiny_shapes(sp):
    sb, info = sp.spense_schedule(128, 128, 0, 8, 0)
    assert info["stages"] == 1 and len(sb) == 2                          # one stage: one span
    sb, info = sp.spense_schedule(*QWEN, 64, 1, sms=20)
    assert len(sb) == 11 and info["ctas_per_span"] == 2
    sb, info = sp.spense_schedule(*QWEN, 256, 1, sms=20)
    assert info["ctas_per_span"] == 2 and info["blocks_per_launch"] * (len(sb) - 1) <= 10
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_schedule(100, 128, 0, 8, 0)
    assert e.value.code == "SPENSE_ERR_SHAPE"
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_schedule(128, 128, 0, 0, 0)
    assert e.value.code == "SPENSE_ERR_ARG"
