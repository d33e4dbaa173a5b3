"""Pins for the oracle's magnitude 2:4 pruning front-end (first slice)."""
import os

import numpy as np

import spense_inputs as si
from oracle import spense_oracle as o


def test_group_rule_matches_the_hand_table(golden_dir):
    n = 0
    for line in open(os.path.join(golden_dir, "prune_2of4_table.txt")):
        if line.startswith("#") or not line.strip():
            continue
        lhs, rhs = line.split("->")
        vals = [float(v) for v in lhs.split()]
        want = [c == "1" for c in rhs.strip()]
        assert o.prune_2to4_group(vals) == want, line
        # the vectorised array version agrees with the scalar rule on a [1, 4] gate matrix (H = 4, I = 1, no dense part)
        g, _, _ = o.prune_2to4_magnitude(np.array([vals]), np.array([vals]), np.array([[v] for v in vals]).reshape(4, 1), None, 0)
        assert np.array_equal(g[0], np.where(want, vals, 0.0))
        n += 1
    assert n == 14


def test_result_is_2_4_in_permuted_order_and_dense_region_untouched():
    rng = np.random.default_rng(3)
    I, H, I_d = 256, 64, 128
    wg, wu, wd = rng.normal(size=(I, H)), rng.normal(size=(I, H)), rng.normal(size=(H, I))
    d = np.sort(rng.choice(I, I_d, replace=False))
    perm = o.perm_from_dense_idx(I, d)
    g, u, dn = o.prune_2to4_magnitude(wg, wu, wd, perm, I_d)
    I_s = I - I_d
    for m, ref in ((g, wg), (u, wu)):
        blk = m[perm[:I_s]].reshape(I_s, H // 4, 4)
        assert ((blk != 0).sum(axis=2) == 2).all()                          # T1 (Eq. 1) with generic values: exactly 2 kept
        assert np.array_equal(m[perm[I_s:]], ref[perm[I_s:]])               # the protected dense rows are untouched
        kept = blk != 0
        mag = np.abs(ref[perm[:I_s]].reshape(I_s, H // 4, 4))
        assert (np.where(kept, mag, np.inf).min(axis=2) >= np.where(kept, -np.inf, mag).max(axis=2)).all()   # kept >= dropped
    blk = dn[:, perm[:I_s]].reshape(H, I_s // 4, 4)                         # W_down: groups along the PERMUTED columns (Q9b)
    assert ((blk != 0).sum(axis=2) == 2).all()
    assert np.array_equal(dn[:, perm[I_s:]], wd[:, perm[I_s:]])
    # brute force: every group against the scalar rule
    src = wd[:, perm[:I_s]].reshape(H, I_s // 4, 4)
    for r in range(0, H, 7):
        for gi in range(0, I_s // 4, 5):
            assert list(blk[r, gi] != 0) == o.prune_2to4_group(src[r, gi])


def test_matches_the_generators_pruning_and_packs_cleanly():
    """The seeded generator (spense_inputs) prunes by the same rule with torch: the oracle reproduces its mask, and the
    pruned, quantised layer satisfies Eq. 1, i.e. pack_canonical accepts it."""
    L0 = si.make_layer(256, 512, 0.25, seed=5, prune=False)
    L1 = si.make_layer(256, 512, 0.25, seed=5, prune=True)
    dec = lambda b: o.e4m3_decode(b.numpy())
    # prune the fp32 weights the generator drew: here reconstructed from L0's bytes only for the mask comparison
    g, u, d = o.prune_2to4_magnitude(dec(L0.wgate), dec(L0.wup), dec(L0.wdown), L1.perm.numpy(), L1.I_dense)
    perm, I_s = L1.perm.numpy().astype(np.int64), 512 - L1.I_dense
    assert (((g[perm[:I_s]] != 0).reshape(I_s, -1, 4).sum(axis=2)) <= 2).all()
    c = o.pack_canonical(L1.wgate.numpy(), L1.wup.numpy(), L1.wdown.numpy(), perm, L1.I_dense)   # raises on a 2:4 violation
    assert c["gate_sp_val"].shape == (I_s, 128)


# ---------------------------------------------------------------------------------------------------------------
# SparseGPT 2:4 column sweep with dense columns on the right (Eqs. 2-3)
# ---------------------------------------------------------------------------------------------------------------
def _hessian(rng, K, n=None):
    X = rng.normal(size=(n or 4 * K, K)) @ (np.eye(K) + 0.3 * rng.normal(size=(K, K)))     # correlated inputs
    return X, X.T @ X


def test_obs_identity_hessian_is_magnitude_pruning():
    # H = I: Eq. 3 gives eps_m = w_m^2 and delta_m only touches w_m itself -> the 2 smallest |w| of every group go
    rng = np.random.default_rng(0)
    w = rng.normal(size=(6, 16))
    got, pruned = o.sparsegpt_2to4(w, np.eye(16), 12)
    want = w.copy()
    for r in range(6):
        for g in range(3):
            idx = np.argsort(np.abs(w[r, 4 * g:4 * g + 4]), kind="stable")[:2]
            want[r, 4 * g + idx] = 0
    assert np.array_equal(got, want)
    assert pruned[:, 12:].sum() == 0 and (pruned[:, :12].reshape(6, 3, 4).sum(axis=2) == 2).all()


def test_obs_single_pruned_weight_is_the_constrained_least_squares_optimum():
    """Eq. 3 is the minimiser of ||X (w + delta)^T - X w^T|| subject to (w + delta)_m = 0.  Take one row, one group whose
    first column is by far the cheapest to prune: after column 0 the oracle's row must equal the least-squares fit of X w
    on the other columns (numpy.linalg.lstsq: a library routine, not the oracle's formula)."""
    rng = np.random.default_rng(1)
    K = 8
    X, H = _hessian(rng, K)
    w = rng.normal(size=(1, K)) + 3.0
    w[0, 0] = 1e-3                                              # cheapest by orders of magnitude
    # stop the sweep after the first group column by making columns 1..3 dense: k_sparse must be a multiple of 4, so
    # check column 0's update through a 1-column elimination done by hand instead
    Hi = np.linalg.inv(H)
    delta = -w[0, 0] / Hi[0, 0] * Hi[0, :]                      # Eq. 3 as printed
    ref, *_ = np.linalg.lstsq(X[:, 1:], X @ w[0], rcond=None)   # best weights on columns 1.. with w_0 forced to 0
    assert np.allclose((w[0] + delta)[1:], ref, rtol=1e-9, atol=1e-12) and abs((w[0] + delta)[0]) < 1e-15
    # and the oracle applies exactly that update when it prunes column 0 first: compare its row after the full sweep of a
    # 4-column sparse region with a step-by-step replay that uses numpy.linalg.inv of the remaining sub-matrix each time
    got, pruned = o.sparsegpt_2to4(w, Hi, 4)
    assert pruned[0, 0]
    cur = w[0].copy()
    for j in range(4):
        Hj = np.linalg.inv(H[j:, j:])                           # inverse Hessian of the unprocessed columns, from scratch
        if pruned[0, j]:
            cur[j:] += -cur[j] / Hj[0, 0] * Hj[0, :]
            cur[j] = 0.0
    assert np.allclose(got[0], cur, rtol=1e-9, atol=1e-12)
    assert pruned[0, :4].sum() == 2 and pruned[0, 4:].sum() == 0


def test_obs_group_choice_uses_the_diagonal_each_column_will_see():
    # reading Q24: eps_c = w_c^2 / [inverse of H[c:, c:]]_00 -- recompute with numpy.linalg.inv and compare the masks
    rng = np.random.default_rng(2)
    K, N = 12, 40
    X, H = _hessian(rng, K)
    w = rng.normal(size=(N, K))
    got, pruned = o.sparsegpt_2to4(w, np.linalg.inv(H), 8)
    cur = w.copy()
    for j in range(8):
        if j % 4 == 0:
            d = np.array([np.linalg.inv(H[c:, c:])[0, 0] for c in range(j, j + 4)])
            eps = cur[:, j:j + 4] ** 2 / d
            want = np.zeros((N, 4), bool)
            for r in range(N):
                want[r, np.argsort(eps[r], kind="stable")[:2]] = True
            assert np.array_equal(pruned[:, j:j + 4], want)
        Hj = np.linalg.inv(H[j:, j:])
        e = np.where(pruned[:, j], cur[:, j] / Hj[0, 0], 0.0)
        cur[:, j:] -= e[:, None] * Hj[0][None, :]
        cur[pruned[:, j], j] = 0.0
    assert np.allclose(got, cur, rtol=1e-8, atol=1e-11)


def test_obs_invariances_and_the_compensation_buffer():
    rng = np.random.default_rng(3)
    K, N, ks = 32, 24, 20
    X, H = _hessian(rng, K)
    Hi = np.linalg.inv(H)
    w = rng.normal(size=(N, K))
    got, pruned = o.sparsegpt_2to4(w, Hi, ks)
    # 2:4 in the sparse region, nothing pruned beyond it, the dense columns moved (they are the compensation buffer)
    assert (pruned[:, :ks].reshape(N, ks // 4, 4).sum(axis=2) == 2).all() and not pruned[:, ks:].any()
    assert ((got[:, :ks] != 0).reshape(N, ks // 4, 4).sum(axis=2) == 2).all()
    assert not np.allclose(got[:, ks:], w[:, ks:])
    # rows are independent (Eq. 2 separates over rows); scaling H changes nothing (Eq. 3 is homogeneous of degree 0 in H)
    p = rng.permutation(N)
    got_p, pr_p = o.sparsegpt_2to4(w[p], Hi, ks)
    assert np.array_equal(got_p, got[p]) and np.array_equal(pr_p, pruned[p])
    got_s, pr_s = o.sparsegpt_2to4(w, Hi / 7.0, ks)                  # not a power of two on purpose
    assert np.array_equal(pr_s, pruned) and np.allclose(got_s, got, rtol=1e-9, atol=1e-12)
    # the point of the method (Eq. 2): less reconstruction error than pruning the same mask without compensation, and the
    # right-hand buffer helps: with the dense columns frozen (not passed as buffer) the error is larger
    loss = lambda a: np.linalg.norm(X @ (a - w).T) ** 2
    assert loss(got) < 0.8 * loss(np.where(pruned, 0.0, w))
    nobuf, _ = o.sparsegpt_2to4(w[:, :ks], np.linalg.inv(H[:ks, :ks]), ks)
    assert loss(got) < loss(np.concatenate([nobuf, w[:, ks:]], axis=1))


def test_obs_cholesky_rows_are_the_eliminated_inverse():
    # what the GPU entry point takes: U upper triangular with H^-1 = U^T U; row j of the inverse Hessian of the unprocessed
    # columns is U[j, j] * U[j, j:] -- the oracle's Gaussian elimination reaches the same rows
    rng = np.random.default_rng(4)
    K = 10
    _, H = _hessian(rng, K)
    Hi = np.linalg.inv(H)
    U = np.linalg.cholesky(Hi).T
    assert np.allclose(U.T @ U, Hi)
    cur = Hi.copy()
    for j in range(K):
        assert np.allclose(cur[j, j:], U[j, j] * U[j, j:], rtol=1e-9)
        cur[j + 1:, j + 1:] -= np.outer(cur[j + 1:, j], cur[j, j + 1:]) / cur[j, j]
