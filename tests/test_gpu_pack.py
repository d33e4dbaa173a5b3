"""-m gpu: spense_pack through the C ABI must be BIT-EXACT against the oracle (values, metadata,
permutation) and the blob must be the documented re-tiling of the canonical arrays."""
import numpy as np
import pytest
import torch

import spense_inputs as si
from oracle import spense_oracle as o
from tests.blob_layout import HEADER, expected_blob_body
from tests.gpu_common import Case, cuda

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    from paper_2606_10445_b200 import build, spense
    build.build()
    assert torch.cuda.is_available()
    return spense


CASES = [  # H, I, p, I_dense override
    (256, 1024, 0.25, None),      # Tiny (BASELINE.json configs[0])
    (256, 1024, 0.0, None),       # all sparse
    (256, 1024, 1.0, None),       # all dense
    (384, 640, None, 128),        # H % 256 == 128 and I_s % 256 == 0: padded sparse stage, odd down tile
    (128, 384, None, 0),          # I_s % 256 == 128 (padded down K stage), single down half tile
    (640, 896, None, 384),        # several tiles, ragged everything
]


@pytest.mark.parametrize("H,I,p,I_d", CASES)
def test_pack_bit_exact(sp, H, I, p, I_d):
    c = Case(H, I, p if p is not None else 0.0, 1, seed=H + I, I_dense=I_d)
    pk = c.pack_gpu(sp, want_canon=True)
    for k, ref in c.canon.items():
        got = pk.canon[k].cpu().numpy()
        assert got.shape == ref.shape and np.array_equal(got, ref), k
    blob = pk.blob.cpu().numpy()
    exp = expected_blob_body(c.canon, H, I, c.I_d)
    assert blob.size == HEADER + exp.size
    assert np.array_equal(blob[HEADER:], exp)
    hdr = blob[:HEADER].view(np.int32)
    assert hdr[2] == H and hdr[3] == I and hdr[4] == c.I_d
    assert np.array_equal(blob[20:32].view(np.float32), np.array(c.L.w_scale, np.float32))


def test_pack_identity_perm_and_signed_zero(sp):
    wg, wu, wd, _ = si.make_small_int_case(256, 512, 128, 1, seed=3)      # 2:4 in identity order
    wg = wg.clone()
    wg[wg == 0] = 0x80                                   # every zero becomes -0: must be normalised to +0
    ref = o.pack_canonical(wg.numpy(), wu.numpy(), wd.numpy(), None, 128)
    pk = sp.spense_pack(cuda(wg), cuda(wu), cuda(wd), (1.0, 1.0, 1.0), None, 128, want_canon=True)
    for k, r in ref.items():
        assert np.array_equal(pk.canon[k].cpu().numpy(), r), k
    assert not (pk.canon["gate_sp_val"].cpu().numpy() == 0x80).any()


def test_pack_error_paths(sp):
    L = si.make_layer(256, 512, 0.25, seed=9)
    perm = L.perm.numpy().astype(np.int64)
    I_s = 512 - L.I_dense
    args = lambda wg=L.wgate, wd=L.wdown, pm=L.perm: (cuda(wg), cuda(L.wup), cuda(wd), L.w_scale, cuda(pm), L.I_dense)
    # > 2 non-zeros in a sparse-region group: first offender in (matrix, row, group) order is reported
    wg = L.wgate.clone()
    wg[int(perm[7]), 12:16] = 0x38
    wg[int(perm[9]), 0:4] = 0x38
    wd = L.wdown.clone()
    wd[3, torch.from_numpy(perm[0:4])] = 0x38
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_pack(*args(wg=wg, wd=wd))
    assert e.value.code == "SPENSE_ERR_NOT_2_4" and e.value.where[:3] == (0, 7, 3) and e.value.where[3] == 3
    with pytest.raises(o.SpenseOracleError) as eo:
        o.pack_canonical(wg.numpy(), L.wup.numpy(), wd.numpy(), L.perm.numpy(), L.I_dense)
    assert eo.value.code == e.value.code and eo.value.where[:3] == e.value.where[:3]
    # the same bytes in the dense region are fine
    wg = L.wgate.clone()
    wg[int(perm[I_s + 3]), 0:4] = 0x38
    sp.spense_pack(*args(wg=wg))
    # NaN byte anywhere (here: dense region of down)
    wd = L.wdown.clone()
    wd[5, int(perm[I_s + 9])] = 0xFF
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_pack(*args(wd=wd))
    assert e.value.code == "SPENSE_ERR_NAN_WEIGHT" and e.value.where[:3] == (2, 5, (I_s + 9) // 4)
    # perm not a bijection
    pm = L.perm.clone()
    pm[1] = pm[0]
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_pack(*args(pm=pm))
    assert e.value.code == "SPENSE_ERR_BAD_PERM"
    # shape / alignment / buffer errors never reach the device
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_pack(cuda(L.wgate), cuda(L.wup), cuda(L.wdown), L.w_scale, cuda(L.perm), 100)
    assert e.value.code == "SPENSE_ERR_SHAPE"


def test_quantize_helper_bit_exact(sp):
    g = torch.Generator().manual_seed(0)
    x = torch.randn(37, 1000, generator=g) * torch.exp(torch.randn(37, 1, generator=g) * 3)
    x[3] = 0
    x[5, 7] = 1e30
    for mode, ref in ((sp.SPENSE_PER_ROW, o.quantize_per_row), (sp.SPENSE_PER_TENSOR, o.quantize_per_tensor)):
        q, s = sp.spense_quantize_e4m3(x.cuda(), mode)
        rq, rs = ref(x.numpy())
        assert np.array_equal(s.cpu().numpy().reshape(-1), np.asarray(rs, np.float32).reshape(-1))
        assert np.array_equal(q.cpu().numpy(), rq)


def test_read_probe_reads_every_chunk(sp):
    """spense_probe_read (measurement helper): each CTA's sink word is the XOR of one word of every 32 KB chunk it was dealt
    (chunk c -> CTA c % grid, word at byte (4 c) % 32768 of the chunk) -- recomputed here from the buffer."""
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    for n_chunks in (5, sms, 6 * sms + 17, 2048 + 5):           # fewer chunks than CTAs, one each, a ragged last ring pass, many
        buf = torch.empty(n_chunks * 32768, dtype=torch.uint8, device="cuda")
        buf.view(torch.int64).random_()
        sink = sp.spense_probe_read(buf)
        torch.cuda.synchronize()
        words = buf.cpu().numpy().view(np.uint32).reshape(n_chunks, 8192)
        grid = min(sms, n_chunks)
        want = np.zeros(256, np.uint32)
        for c in range(n_chunks):
            want[c % grid] ^= words[c, c % 8192]
        assert np.array_equal(sink.cpu().numpy().view(np.uint32), want), n_chunks
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_probe_read(torch.empty(32768 + 128, dtype=torch.uint8, device="cuda"))
    assert e.value.code == "SPENSE_ERR_ARG"
