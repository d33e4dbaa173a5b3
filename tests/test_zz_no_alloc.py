"""-m gpu: spense_quantize_e4m3_static, the one entry point that needs no scratch buffer from the caller.

Who it is for: code that has to quantise activations at a moment when it cannot obtain device memory -- a serving engine
that gave every free byte of HBM to its cache pool at start-up, a plug-in called from a host callback or from inside a
framework's allocator hook (a cudaMalloc there re-enters or deadlocks), a loop that cannot afford the device-wide
synchronisation hidden in cudaMalloc / cudaFree.  Its scratch is a fixed 256 KB array inside libspense.so, so the row
count is capped at SPENSE_QUANTIZE_STATIC_MAX_ROWS and all calls on a device share (and must not overlap on) that array.

What is checked: on two calls in a row -- the second with a different shape and mode, so that it finds the first call's
maxima still in the shared array -- the output bytes and the scales are IDENTICAL to those of spense_quantize_e4m3 (the
existing path with a caller-provided workspace), which tests/test_gpu_pack.py holds bit-exact against the oracle.  The
bar is the one that test uses: integer/byte results, bit for bit.  The size cap is checked on the host side of the call.

This file is named to be collected LAST: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (first call = address look-up) and after the rest of the suite.
"""
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    from paper_2606_10445_b200 import build, spense
    build.build()
    assert torch.cuda.is_available()
    return spense


def _inputs(rows, cols, seed, spike):
    g = torch.Generator().manual_seed(seed)
    x = torch.randn(rows, cols, generator=g) * torch.exp(torch.randn(rows, 1, generator=g) * 3)
    x[rows // 3] = 0                       # an all-zero row: scale 1
    if spike:
        x[rows // 2, cols // 5] = 1e30     # every other element of its row quantises to zero
    return x.cuda()


def test_static_scratch_quantize_equals_workspace_path_on_two_calls_in_a_row(sp):
    # call 1: many rows, per row.  call 2: fewer rows of another width, per tensor -- its [rows] slot (the tensor maximum)
    # and every row slot it reads were written by call 1 with other values; stale contents must not leak into the result.
    # call 3 repeats call 1's configuration on fresh data after the per-tensor call.
    calls = [(300, 1000, sp.SPENSE_PER_ROW, 1), (37, 4096, sp.SPENSE_PER_TENSOR, 2), (300, 1000, sp.SPENSE_PER_TENSOR, 3),
             (1, 128, sp.SPENSE_PER_ROW, 4)]
    xs = [_inputs(r, c, seed, spike=(m == sp.SPENSE_PER_ROW)) for r, c, m, seed in calls]
    # outputs are the caller's: allocate them all BEFORE the calls under test, as a caller that cannot allocate would have
    outs = [torch.full((r, c), 0xAA, dtype=torch.uint8, device="cuda") for r, c, _, _ in calls]
    scs = [torch.full((r if m == sp.SPENSE_PER_ROW else 1,), -1.0, dtype=torch.float32, device="cuda") for r, _, m, _ in calls]
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for x, out, sc, (_, _, mode, _) in zip(xs, outs, scs, calls):       # back to back on one stream, no sync between
        sp.spense_quantize_e4m3_static(x, mode, out, sc)
    assert torch.cuda.memory_allocated() == before                        # the binding created no tensor either
    torch.cuda.synchronize()
    for x, out, sc, (_, _, mode, _) in zip(xs, outs, scs, calls):
        q_ref, s_ref = sp.spense_quantize_e4m3(x, mode)                   # existing path, scratch from the caller
        assert torch.equal(sc, s_ref.reshape(-1))
        assert torch.equal(out, q_ref)
        assert not bool((out == 0x7F).any() | (out == 0xFF).any())        # no NaN byte


def test_static_scratch_row_cap_is_a_clear_host_side_error(sp):
    cap = sp.SPENSE_QUANTIZE_STATIC_MAX_ROWS
    x = torch.ones(cap + 1, 4, device="cuda")
    out = torch.full((cap + 1, 4), 0xAA, dtype=torch.uint8, device="cuda")
    sc = torch.full((cap + 1,), -1.0, device="cuda")
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_quantize_e4m3_static(x, sp.SPENSE_PER_ROW, out, sc)
    assert e.value.code == "SPENSE_ERR_STATIC_SCRATCH" and "built-in scratch" in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 0xAA).all()) and bool((sc == -1.0).all())         # nothing was launched
    # exactly at the cap it runs, and agrees with the workspace path
    q, s = sp.spense_quantize_e4m3_static(x[:cap], sp.SPENSE_PER_ROW, out[:cap], sc[:cap])
    q_ref, s_ref = sp.spense_quantize_e4m3(x[:cap], sp.SPENSE_PER_ROW)
    assert torch.equal(q, q_ref) and torch.equal(s, s_ref)
