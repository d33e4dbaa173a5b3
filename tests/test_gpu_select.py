"""-m gpu: spense_select_dense (SpenseGPT+ dense-index selection) against the oracle.

Floating point decides an index set here, so: scores are compared in value (fp32 sums vs the oracle's float64);
the selection must equal the oracle's TopK rule applied to the GPU's OWN scores exactly; against the oracle's own
selection it may differ only at indices whose score lies within the rounding tolerance of the threshold."""
import numpy as np
import pytest
import torch

from oracle import spense_oracle as o

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    from paper_2606_10445_b200 import build, spense
    build.build()
    assert torch.cuda.is_available()
    return spense


def _case(I, H, seed, heavy_tail=True):
    g = torch.Generator().manual_seed(seed)
    wg = torch.randn(I, H, generator=g) * 0.02
    wu = torch.randn(I, H, generator=g) * 0.02
    wd = torch.randn(H, I, generator=g) * 0.02
    if heavy_tail:                                        # per-index scales so the scores are well spread
        sc = torch.exp(0.5 * torch.randn(I, generator=g))
        wg *= sc[:, None]; wu *= sc[:, None]; wd *= sc[None, :]
    hx = torch.rand(H, generator=g) * 4 + 0.1
    hh = torch.rand(I, generator=g) * 4 + 0.1
    return wg, wu, wd, hx, hh


@pytest.mark.parametrize("I,H,I_d", [(256, 128, 128), (1024, 256, 256), (1024, 256, 0), (1024, 256, 1024),
                                     (2176, 384, 640), (25600, 5120, 6400)])
def test_select_matches_oracle(sp, I, H, I_d):
    wg, wu, wd, hx, hh = _case(I, H, seed=I + H)
    score, dense_idx, perm = sp.spense_select_dense(wg.cuda(), wu.cuda(), wd.cuda(), hx.cuda(), hh.cuda(), I_d, eps=1e-8)
    s2, d2, p2 = sp.spense_select_dense(wg.cuda(), wu.cuda(), wd.cuda(), hx.cuda(), hh.cuda(), I_d, eps=1e-8)
    torch.cuda.synchronize()
    assert torch.equal(score, s2) and torch.equal(dense_idx, d2) and torch.equal(perm, p2)      # reproducible
    s_gpu, d_gpu, p_gpu = score.cpu().numpy(), dense_idx.cpu().numpy(), perm.cpu().numpy()
    s_ref = o.spensegpt_plus_scores(wg.numpy(), wu.numpy(), wd.numpy(), hx.numpy(), hh.numpy(), 1e-8)
    # fp32 sums of H (or 32-way tree of H/32) positive terms: relative error far below 1e-4
    assert np.allclose(s_gpu, s_ref, rtol=2e-5, atol=0), np.abs(s_gpu / s_ref - 1).max()
    # the decision, taken in the kernel's precision: the oracle's rule on the GPU's own scores
    assert np.array_equal(d_gpu, o.topk_dense_idx(s_gpu, I_d))
    assert np.array_equal(p_gpu, o.perm_from_dense_idx(I, d_gpu))
    # against the oracle's own decision: only indices within the tolerance of the threshold may differ
    d_ref = o.spensegpt_plus_dense_idx(wg.numpy(), wu.numpy(), wd.numpy(), hx.numpy(), hh.numpy(), I_d, 1e-8)
    sym = np.setxor1d(d_gpu, d_ref)
    if 0 < I_d < I:
        thr = np.sort(s_ref)[::-1][I_d - 1]
        assert (np.abs(s_ref[sym] - thr) <= 4e-5 * thr).all()
        assert sym.size <= max(2, I // 1000)
    else:
        assert sym.size == 0


def test_select_ties_and_planted_indices(sp):
    I, H = 512, 128
    ones = [torch.ones(I, H), torch.ones(I, H), torch.ones(H, I), torch.ones(H), torch.ones(I)]
    score, d, perm = sp.spense_select_dense(*[t.cuda() for t in ones], 128, eps=0.0)
    assert torch.equal(score.cpu(), torch.full((I,), 3.0))
    assert torch.equal(d.cpu(), torch.arange(128, dtype=torch.int32))           # ties go to the lower index
    wg, wu, wd, hx, hh = _case(I, H, seed=1, heavy_tail=False)
    wg[300] *= 50.0
    wg[17] = 0; wu[17] = 0; wd[:, 17] = 0
    score, d, perm = sp.spense_select_dense(wg.cuda(), wu.cuda(), wd.cuda(), hx.cuda(), hh.cuda(), 128)
    assert int(score.argmax()) == 300 and float(score[17]) == 0.0
    assert 300 in d.cpu().tolist() and 17 not in d.cpu().tolist()
    assert perm.cpu().tolist()[-128:] == d.cpu().tolist()


def test_select_prune_quantise_pack_chain(sp):
    """The offline chain on the GPU, step by step against the oracle's: SpenseGPT+ selection (Eqs. 8-12) -> magnitude 2:4
    pruning of the sparse region in PERMUTED order -> per-tensor E4M3 quantisation -> spense_pack.  Every
    step is bit-exact (scores aside, which decide the same index set), the packed layer passes Eq. 1, its dense block holds
    exactly the selected indices D, and the packed layer computes the oracle's MLP."""
    I, H, I_d, M = 1024, 256, 256, 8
    wg, wu, wd, hx, hh = _case(I, H, seed=11)
    # 1. selection
    _, d, perm = sp.spense_select_dense(wg.cuda(), wu.cuda(), wd.cuda(), hx.cuda(), hh.cuda(), I_d)
    d_or = o.spensegpt_plus_dense_idx(wg.numpy(), wu.numpy(), wd.numpy(), hx.numpy(), hh.numpy(), I_d)
    d_ref = d.cpu().numpy()                                # fp32 scores may swap indices that tie at the threshold: go on with the GPU's set
    assert len(np.setxor1d(d_ref, d_or)) <= 2
    perm_ref = o.perm_from_dense_idx(I, d_ref)
    assert np.array_equal(perm.cpu().numpy(), perm_ref)
    # 2. prune (in place on device copies)
    g_d, u_d, d_d = wg.cuda().clone(), wu.cuda().clone(), wd.cuda().clone()
    sp.spense_prune_2to4_magnitude(g_d, u_d, d_d, perm, I_d)
    g_ref, u_ref, dn_ref = o.prune_2to4_magnitude(wg.numpy(), wu.numpy(), wd.numpy(), perm_ref, I_d)
    for got, ref in ((g_d, g_ref), (u_d, u_ref), (d_d, dn_ref)):
        assert np.array_equal(got.cpu().numpy().view(np.uint32), ref.astype(np.float32).view(np.uint32))
    # 3. quantise, per tensor
    q, scales = zip(*[sp.spense_quantize_e4m3(t, sp.SPENSE_PER_TENSOR) for t in (g_d, u_d, d_d)])
    for (qb, sc), ref in zip(zip(q, scales), (g_ref, u_ref, dn_ref)):
        rb, rs = o.quantize_per_tensor(ref.astype(np.float32))
        assert float(sc) == float(rs) and np.array_equal(qb.cpu().numpy(), rb)
    w_scale = tuple(float(s) for s in scales)
    # 4. pack: accepts the layer (Eq. 1 holds in permuted order), canonical arrays equal the oracle's
    pk = sp.spense_pack(q[0], q[1], q[2], w_scale, perm, I_d, want_canon=True)
    canon = o.pack_canonical(q[0].cpu().numpy(), q[1].cpu().numpy(), q[2].cpu().numpy(), perm_ref, I_d)
    for k, ref in canon.items():
        assert np.array_equal(pk.canon[k].cpu().numpy(), ref), k
    assert np.array_equal(pk.canon["perm"].cpu().numpy()[I - I_d:], d_ref)      # the dense block is D, ascending (Q8, Q9)
    assert np.array_equal(pk.canon["gate_dn"].cpu().numpy(), q[0].cpu().numpy()[d_ref])
    # 5. and the packed layer runs: y against the oracle's down fed the GPU's Hq
    import spense_inputs as si
    x, s_x = si.make_activations(M, H, seed=3)
    ug, uu, ud = o.unpack_canonical(canon)
    r1 = o.gate_up(x.numpy(), s_x.numpy(), ug, uu, w_scale[0], w_scale[1], 1.0)
    s_h = o.requant_scale_from_h(r1["h"])
    ws = sp.spense_workspace(pk, M)
    hq = torch.empty(M, I, dtype=torch.uint8, device="cuda")
    y = sp.spense_mlp(pk, x.cuda(), s_x.cuda(), torch.from_numpy(s_h).cuda(), ws, hq_scratch=hq)
    torch.cuda.synchronize()
    ref = o.down(hq.cpu().numpy(), s_h, ud, w_scale[2])
    assert (np.abs(y.cpu().numpy() - ref["y"]) <= o.tol_gemm(ref["absY"])).all()


def test_dense_idx_last_is_eq5(sp):
    """SpenseGPT's choice (Eq. 5, reading Q1): the last n indices; feeds the same permutation helper."""
    d = sp.spense_dense_idx_last(1024, 256)
    assert np.array_equal(d.numpy(), o.spensegpt_dense_idx(1024, 256))
    assert np.array_equal(sp.spense_perm_from_dense_idx(1024, d.tolist()).numpy(), np.arange(1024))   # already at the back
    assert sp.spense_dense_idx_last(128, 0).numel() == 0


def test_select_argument_errors(sp):
    w = torch.zeros(256, 128, device="cuda")
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_select_dense(w, w, w.t().contiguous(), torch.ones(128, device="cuda"), torch.ones(256, device="cuda"), 100)
    assert e.value.code == "SPENSE_ERR_SHAPE"
