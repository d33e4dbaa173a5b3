"""Pins for the oracle's SpenseGPT+ dense-index selection (Eqs. 8-12): brute force,
closed forms, invariances the equations imply."""
import numpy as np

from oracle import spense_oracle as o


def _case(I=64, H=48, seed=0):
    r = np.random.default_rng(seed)
    return (r.normal(size=(I, H)), r.normal(size=(I, H)), r.normal(size=(H, I)),
            r.uniform(0.1, 4.0, size=H), r.uniform(0.1, 4.0, size=I))


def test_scores_match_a_plain_python_loop():
    wg, wu, wd, hx, hh = _case(I=12, H=7)
    I, H = wg.shape
    eps = 1e-8
    sg, su, sd = [0.0] * I, [0.0] * I, [0.0] * I
    for i in range(I):
        for j in range(H):
            sg[i] += abs(wg[i, j]) * hx[j] ** 0.5 / H            # Eq. 8 summed as Eq. 9
            su[i] += abs(wu[i, j]) * hx[j] ** 0.5 / H
            sd[i] += abs(wd[j, i]) * hh[i] ** 0.5 / H            # index i is a column of W_down
    mean = lambda v: sum(v) / len(v)
    ref = [sg[i] / (mean(sg) + eps) + su[i] / (mean(su) + eps) + sd[i] / (mean(sd) + eps) for i in range(I)]
    assert np.allclose(o.spensegpt_plus_scores(wg, wu, wd, hx, hh, eps), ref, rtol=1e-12, atol=0)


def test_closed_forms_and_invariances():
    I, H = 32, 16
    ones = (np.ones((I, H)), np.ones((I, H)), np.ones((H, I)), np.ones(H), np.ones(I))
    s = o.spensegpt_plus_scores(*ones, eps=0.0)
    assert np.allclose(s, 3.0)                                   # every Norm(.) is 1 when all indices are equal
    assert np.array_equal(o.topk_dense_idx(s, 8), np.arange(8))  # ties go to the lower index
    wg, wu, wd, hx, hh = _case()
    s = o.spensegpt_plus_scores(wg, wu, wd, hx, hh, eps=0.0)
    assert abs(s.mean() - 3.0) < 1e-12                           # each normalised vector has mean 1
    # Eq. 10 removes the scale of each projection and of each Hessian
    s2 = o.spensegpt_plus_scores(7.0 * wg, 0.01 * wu, -3.0 * wd, 5.0 * hx, 0.2 * hh, eps=0.0)
    assert np.allclose(s, s2, rtol=1e-12)
    # permuting the intermediate indices (rows of gate/up, columns of down, entries of H_down) permutes the scores
    perm = np.random.default_rng(1).permutation(wg.shape[0])
    sp = o.spensegpt_plus_scores(wg[perm], wu[perm], wd[:, perm], hx, hh[perm], eps=0.0)
    assert np.allclose(sp, s[perm], rtol=1e-12)
    # an index with a planted heavy row/column is selected first; a zeroed one last
    wg2, wd2 = wg.copy(), wd.copy()
    wg2[5] *= 100.0
    wg2[9] = 0.0
    wu2 = wu.copy(); wu2[9] = 0.0
    wd2[:, 9] = 0.0
    s3 = o.spensegpt_plus_scores(wg2, wu2, wd2, hx, hh)
    assert s3.argmax() == 5 and s3.argmin() == 9 and s3[9] == 0.0
    assert 5 in o.topk_dense_idx(s3, 1) and 9 not in o.topk_dense_idx(s3, wg.shape[0] - 1)


def test_topk_is_sorted_unique_and_feeds_the_permutation():
    wg, wu, wd, hx, hh = _case(I=256, H=32, seed=3)
    d = o.spensegpt_plus_dense_idx(wg, wu, wd, hx, hh, 128)
    assert d.dtype == np.int32 and d.size == 128 and np.all(np.diff(d) > 0)
    s = o.spensegpt_plus_scores(wg, wu, wd, hx, hh)
    rest = np.setdiff1d(np.arange(256), d)
    assert s[d].min() >= s[rest].max()
    perm = o.perm_from_dense_idx(256, d)
    assert np.array_equal(perm[128:], d) and np.array_equal(perm[:128], rest)    # dense block last, stable (Q8, Q9)
