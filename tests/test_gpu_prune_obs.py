"""-m gpu: spense_prune_obs_2to4 (SparseGPT 2:4 column sweep with the dense columns on the right as compensation buffer;
SURVEY.md 8f NEXT-4; Eqs. 2-3) through the C ABI against the float64 oracle.

Floating point decides the masks here (eps = w^2 / [H^-1]_mm on weights that carry the rounding of every earlier update),
so several results are correct: what is unique is checked exactly (2:4 compliance, nothing pruned in the dense columns,
the identity-Hessian case = magnitude pruning bit for bit), the rest is checked for validity: the masks agree with the
oracle's on all but a tiny share of the groups, rows whose masks agree carry the oracle's weights within fp32 tolerance,
and the reconstruction loss of Eq. 2 equals the oracle's within 1 %."""
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


def make_problem(N, K, seed, damp=0.01):
    """weights N(0, 0.02^2); inputs with correlated channels and a few outlier channels (the recipe of spense_inputs for
    activations); H = X^T X + damp * mean(diag) * I; U = upper Cholesky factor of H^-1 (float64 library routines), fp32"""
    rng = np.random.default_rng(seed)
    w = (rng.normal(size=(N, K)) * 0.02).astype(np.float32)
    X = rng.normal(size=(2 * K, K)) @ (np.eye(K) + 0.2 * rng.normal(size=(K, K)) / np.sqrt(K))
    X[:, rng.choice(K, max(1, K // 64), replace=False)] *= 20.0
    H = X.T @ X
    H += damp * np.mean(np.diag(H)) * np.eye(K)
    U = np.ascontiguousarray(np.linalg.cholesky(np.linalg.inv(H)).T).astype(np.float32)
    return w, X, U


def check_against_oracle(sp, N, K, ks, seed):
    w, X, U = make_problem(N, K, seed)
    got = sp.spense_prune_obs_2to4(torch.from_numpy(w).cuda(), torch.from_numpy(U).cuda(), ks).cpu().numpy()
    torch.cuda.synchronize()
    U64 = U.astype(np.float64)
    eps_all = np.empty((N, ks // 4, 4))                         # the criterion values every group was decided on

    d_all = np.empty((ks // 4, 4))                              # and the diagonals [Hi_c]_cc of Eq. 3 behind them

    def keep_eps(j, eps, d):
        eps_all[:, j // 4] = eps
        d_all[j // 4] = d
    ref, pruned = o.sparsegpt_2to4(w, U64.T @ U64, ks, on_group=keep_eps)   # the oracle sees exactly the fp32 factor the GPU got
    # unique: Eq. 1 holds on the sparse region, exactly 2 pruned per group; the dense columns hold no forced zeros
    gz = (got[:, :ks] == 0).reshape(N, ks // 4, 4)
    assert (gz.sum(axis=2) == 2).all()
    assert not (got[:, ks:] == 0).any()
    # masks: equal to the oracle's except where two eps were a rounding error apart
    same_group = (gz == pruned[:, :ks].reshape(N, ks // 4, 4)).all(axis=2)
    assert same_group.mean() > 0.999, same_group.mean()
    rows = same_group.all(axis=1)
    assert rows.mean() > (0.9 if ks <= 1024 else 0.5)          # a long row has many groups to meet a near-tie in
    err = np.abs(got[rows].astype(np.float64) - ref[rows])
    scale = np.abs(ref[rows]).max(axis=1, keepdims=True)
    assert (err <= 2e-3 * scale + 1e-7).all(), (err / scale).max()
    # rows whose masks differ somewhere, checked group by group: up to the first differing group the row followed the
    # oracle (frozen columns equal within tolerance), and AT that group the GPU's choice is a valid one -- the eps (Eq. 3)
    # of what it pruned exceed the eps of what it kept by no more than a weight error of 1e-4 of the row's scale moves them
    worst = 0.0
    for r in np.where(~rows)[0]:
        g0 = int(np.argmin(same_group[r]))
        c0 = 4 * g0
        sc = np.abs(ref[r]).max()
        assert (np.abs(got[r, :c0].astype(np.float64) - ref[r, :c0]) <= 2e-3 * sc + 1e-7).all(), (r, g0)
        e, gp, d = eps_all[r, g0], gz[r, g0], d_all[g0]
        a = np.where(gp)[0][np.argmax(e[gp])]                   # the GPU pruned a although it kept b with a smaller eps
        b = np.where(~gp)[0][np.argmin(e[~gp])]
        gap = e[a] - e[b]
        # eps = w^2 / d, so a weight error dw moves it by 2 sqrt(eps / d) dw + dw^2 / d; dw = 1e-4 of the row's scale
        dw = 1e-4 * sc
        allow = sum(2 * np.sqrt(e[c] / d[c]) * dw + dw * dw / d[c] for c in (a, b))
        worst = max(worst, gap / allow)
        assert gap <= allow, (r, g0, e, gp)
    print(f"[obs] N={N} K={K} ks={ks}: {int((~rows).sum())} rows differ somewhere, worst eps gap / allowance {worst:.3e}")
    # validity of everything (Eq. 2): the reconstruction loss is the oracle's
    loss = lambda a: np.linalg.norm(X @ (a.astype(np.float64) - w).T) ** 2
    assert abs(loss(got) - loss(ref)) <= 0.01 * loss(ref)
    assert loss(got) < loss(np.where(got == 0, 0.0, w))        # and compensation beats the bare mask
    return got


@pytest.mark.parametrize("N,K,ks", [(64, 128, 128), (200, 256, 192), (130, 384, 100), (512, 512, 512), (96, 640, 388), (256, 256, 0)])
def test_obs_sweep_parity(sp, N, K, ks):
    if ks == 0:
        w, X, U = make_problem(N, K, 1)
        got = sp.spense_prune_obs_2to4(torch.from_numpy(w).cuda(), torch.from_numpy(U).cuda(), 0).cpu().numpy()
        assert np.array_equal(got, w)                            # nothing to prune: untouched
        return
    check_against_oracle(sp, N, K, ks, seed=100 + N + K + ks)


def test_identity_hessian_is_magnitude_pruning_bit_for_bit(sp):
    rng = np.random.default_rng(5)
    N, K, ks = 300, 256, 192
    w = (rng.normal(size=(N, K)) * 0.02).astype(np.float32)
    got = sp.spense_prune_obs_2to4(torch.from_numpy(w).cuda(), torch.eye(K, device="cuda"), ks).cpu().numpy()
    ref, _ = o.sparsegpt_2to4(w, np.eye(K), ks)
    assert np.array_equal(got.astype(np.float64), ref)
    want = w.copy()
    blk = want[:, :ks].reshape(N, ks // 4, 4)
    for c in np.argsort(np.abs(blk), axis=2, kind="stable")[:, :, :2].transpose(2, 0, 1):
        np.put_along_axis(blk, c[..., None], 0.0, axis=2)
    assert np.array_equal(got, want)


def test_obs_mid_size_down_shaped(sp):
    # a down-projection-shaped case: more columns than rows, a quarter of them dense on the right
    check_against_oracle(sp, 256, 1024, 768, seed=9)


def test_obs_many_column_blocks(sp):
    """fp32 error growth over many 128-column blocks, on a sample of rows (rows are independent): a gate/up-shaped sweep
    (K_sparse = K, 20 blocks) and a down-shaped one whose sweep crosses 24 blocks with 1024 dense columns on the right."""
    check_against_oracle(sp, 64, 2560, 2560, seed=31)
    check_against_oracle(sp, 64, 4096, 3072, seed=32)


@pytest.mark.skipif(not __import__("os").environ.get("SPENSE_SLOW_TESTS"), reason="5 min of oracle on the host: set SPENSE_SLOW_TESTS=1")
def test_obs_gate_up_real_reduction_length(sp):
    """the Qwen3-32B gate/up reduction length, K = K_sparse = 5120 (40 column blocks), 64 rows"""
    check_against_oracle(sp, 64, 5120, 5120, seed=33)


def test_obs_pruned_layer_packs_and_runs(sp):
    """select-free chain on a small layer: permute -> OBS prune (gate / up rows along H, down columns along the permuted
    intermediate dimension with the dense columns as buffer) -> quantise -> spense_pack accepts it (Eq. 1 holds)."""
    import spense_inputs as si
    H, I, I_d = 256, 512, 128
    rng = np.random.default_rng(11)
    I_s = I - I_d
    wg, wu = [(rng.normal(size=(I, H)) * 0.02).astype(np.float32) for _ in range(2)]
    wd = (rng.normal(size=(H, I)) * 0.02).astype(np.float32)
    perm = np.concatenate([np.sort(rng.permutation(I)[:I_s]), []]).astype(np.int64)
    dense = np.setdiff1d(np.arange(I), perm)
    perm = np.concatenate([np.sort(perm), dense])
    _, _, U_x = make_problem(1, H, 21)                          # Hessian factor of the layer input (H x H)
    _, _, U_h = make_problem(1, I, 22)                          # Hessian factor of down's input, in PERMUTED order (I x I)
    dev = "cuda"
    g = sp.spense_prune_obs_2to4(torch.from_numpy(wg[perm[:I_s]]).to(dev), torch.from_numpy(U_x).to(dev), H)
    u = sp.spense_prune_obs_2to4(torch.from_numpy(wu[perm[:I_s]]).to(dev), torch.from_numpy(U_x).to(dev), H)
    d = sp.spense_prune_obs_2to4(torch.from_numpy(np.ascontiguousarray(wd[:, perm])).to(dev), torch.from_numpy(U_h).to(dev), I_s)
    wg2, wu2, wd2 = torch.from_numpy(wg).to(dev), torch.from_numpy(wu).to(dev), torch.from_numpy(wd).to(dev)
    pt = torch.from_numpy(perm).to(dev)
    wg2[pt[:I_s]] = g
    wu2[pt[:I_s]] = u
    wd2[:, pt] = d
    qs = [sp.spense_quantize_e4m3(t.contiguous(), sp.SPENSE_PER_TENSOR) for t in (wg2, wu2, wd2)]
    pk = sp.spense_pack(qs[0][0], qs[1][0], qs[2][0], [float(q[1]) for q in qs], pt.to(torch.int32), I_d)
    x, s_x = si.make_activations(8, H, seed=3)
    ws = sp.spense_workspace(pk, 8)
    y = sp.spense_mlp(pk, x.cuda(), s_x.cuda(), torch.full((8,), 0.05, device=dev), ws)
    torch.cuda.synchronize()
    assert torch.isfinite(y).all() and sp.spense_device_status() == "SPENSE_OK"
