"""Pins for the oracle's stand-alone Spense linears (Sec. 3.2): none of them re-calls the function
under test on both sides -- expected values are Python-integer sums, the unpermuted dense product, or hand-written bytes."""
import numpy as np
import pytest

import spense_inputs as si
from oracle import spense_oracle as o
from tests.test_oracle_mlp import _units


@pytest.mark.parametrize("split", ["out", "in"])
def test_pack_unpack_round_trip_is_the_permuted_weight(split):
    L = si.make_linear(512, 384, 0.25, split, seed=3)
    w, perm = L.w.numpy(), L.perm.numpy().astype(np.int64)
    c = o.pack_linear_canonical(w, perm, L.n_dense, split)
    wp = w[perm] if split == "out" else w[:, perm]
    wp = np.where((wp & 0x7F) == 0, 0, wp)                      # the pack stores -0 as +0 (Q7)
    rec = o.unpack_linear_canonical(c)
    n_s = (512 if split == "out" else 384) - L.n_dense
    # the sparse region is reconstructed exactly (zero bytes normalised), the dense region is a verbatim copy
    if split == "out":
        assert np.array_equal(rec[:n_s], wp[:n_s]) and np.array_equal(rec[n_s:], w[perm][n_s:])
        assert c["sp_val"].shape == (n_s, 192) and c["sp_meta"].shape == (n_s, 48) and c["dn"].shape == (L.n_dense, 384)
    else:
        assert np.array_equal(rec[:, :n_s], wp[:, :n_s]) and np.array_equal(rec[:, n_s:], w[:, perm][:, n_s:])
        assert c["sp_val"].shape == (512, n_s // 2) and c["sp_meta"].shape == (512, n_s // 8) and c["dn"].shape == (512, L.n_dense)
    # Eq. 1: at most 2 non-zeros in every group of 4 along K of the sparse region, nibbles in the valid set
    sp = rec[:n_s] if split == "out" else rec[:, :n_s]
    assert (((sp & 0x7F) != 0).reshape(sp.shape[0], -1, 4).sum(axis=2) <= 2).all()
    nib = np.concatenate([(c["sp_meta"] & 0xF).ravel(), (c["sp_meta"] >> 4).ravel()])
    assert set(np.unique(nib)) <= set(o.NIBBLES_VALID)


def test_hand_written_out_split_example():
    # N = 4 rows (the alignment of the C ABI is not the oracle's business), K = 8; rows 1 and 3 dense -> perm = [0, 2, 1, 3]
    w = np.array([[0x38, 0, 0, 0x40, 0, 0, 0, 0],          # groups: nz {0,3} -> nibble 0|3<<2 = 12; {} -> 0|1<<2 = 4
                  [0x38, 0x38, 0x38, 0x38, 1, 2, 3, 4],      # dense row: copied verbatim
                  [0, 0, 0x44, 0, 0, 0xB8, 0xC0, 0],         # nz {2} -> (0,2) = 8, values (0, 0x44); nz {1,2} -> 1|2<<2 = 9
                  [9, 9, 9, 9, 9, 9, 9, 9]], np.uint8)
    c = o.pack_linear_canonical(w, np.array([0, 2, 1, 3]), 2, "out")
    assert c["sp_val"].tolist() == [[0x38, 0x40, 0, 0], [0, 0x44, 0xB8, 0xC0]]
    assert c["sp_meta"].tolist() == [[12 | 4 << 4], [8 | 9 << 4]]
    assert c["dn"].tolist() == [w[1].tolist(), w[3].tolist()]


def test_hand_written_in_split_example():
    # K = 8 columns, the dense ones are {1, 6} -> perm = [0, 2, 3, 4, 5, 7 | 1, 6]; sparse K range = 6 is not a multiple of 8,
    # so use K = 12 with dense {1, 6, 9, 10}: perm = [0, 2, 3, 4, 5, 7, 8, 11 | 1, 6, 9, 10]
    perm = np.array([0, 2, 3, 4, 5, 7, 8, 11, 1, 6, 9, 10])
    w = np.zeros((1, 12), np.uint8)
    w[0, [2, 5, 8, 11]] = [0x38, 0x40, 0x44, 0x48]          # permuted positions 1, 4, 6, 7 -> groups {1}, {0, 2, 3}?  no: see below
    # permuted sparse row = w[0, perm[:8]] = [w0, w2, w3, w4, w5, w7, w8, w11] = [0, 0x38, 0, 0 | 0x40, 0, 0x44, 0x48] -> 3 non-zeros
    with pytest.raises(o.SpenseOracleError) as e:
        o.pack_linear_canonical(w, perm, 4, "in")
    assert e.value.code == "SPENSE_ERR_NOT_2_4" and e.value.where[:3] == (0, 0, 1)
    w[0, 11] = 0
    w[0, [1, 6]] = [0x50, 0x58]
    c = o.pack_linear_canonical(w, perm, 4, "in")
    assert c["sp_val"].tolist() == [[0, 0x38, 0x40, 0x44]]      # group 0: nz {1} -> (0, 1); group 1: nz {0, 2}
    assert c["sp_meta"].tolist() == [[(0 | 1 << 2) | (0 | 2 << 2) << 4]]
    assert c["dn"].tolist() == [[0x50, 0x58, 0, 0]]


@pytest.mark.parametrize("split", ["out", "in"])
def test_linear_equals_python_integer_sums_of_the_original_weight(split):
    """y of the packed linear against a Python-integer triple loop over the ORIGINAL (unpermuted, uncompressed) bytes:
    pins the permutation direction, the reconstruction and the s_x[m] * s_w scaling at once."""
    N, K, M = 16, 24, 3
    rng = np.random.default_rng(9)
    codes = np.array([0x00, 0x38, 0x40, 0x44, 0xB8, 0xC0, 0xC4, 0x30, 0x28], np.uint8)
    w = codes[rng.integers(0, len(codes), (N, K))]
    n = N if split == "out" else K
    n_dense = 8
    dense = np.sort(rng.choice(n, n_dense, replace=False))
    perm = o.perm_from_dense_idx(n, dense).astype(np.int64)
    wp = w[perm] if split == "out" else w[:, perm]
    keep = np.zeros_like(wp, bool)                               # make the sparse region 2:4 in PERMUTED order
    n_s = n - n_dense
    if split == "out":
        for r in range(n_s):
            for g in range(K // 4):
                keep[r, 4 * g + rng.choice(4, 2, replace=False)] = True
        keep[n_s:] = True
        w[perm] = wp * keep
    else:
        for r in range(N):
            for g in range(n_s // 4):
                keep[r, 4 * g + rng.choice(4, 2, replace=False)] = True
        keep[:, n_s:] = True
        w[:, perm] = wp * keep
    x = codes[rng.integers(0, len(codes), (M, K))]
    s_x = np.array([0.5, 2.0, 0.25], np.float32)
    s_w = 0.125
    c = o.pack_linear_canonical(w, perm, n_dense, split)
    xin = x if split == "out" else x[:, perm]                    # the in-split consumes x in permuted column order
    r = o.linear(xin, s_x, o.unpack_linear_canonical(c), s_w)
    for m in range(M):
        for nn in range(N):
            row = perm[nn] if split == "out" else nn               # the out-split returns y in permuted row order
            acc = sum(_units(x[m, k]) * _units(w[row, k]) for k in range(K))
            ab = sum(abs(_units(x[m, k]) * _units(w[row, k])) for k in range(K))
            assert r["y"][m, nn] == acc * 2.0 ** -18 * float(s_x[m]) * s_w
            assert r["absY"][m, nn] == ab * 2.0 ** -18 * float(s_x[m]) * s_w


def test_out_split_linear_on_gate_matches_the_mlp_pack():
    # the gate projection of a layer packed as a stand-alone out-split linear holds the same canonical bytes
    L = si.make_layer(256, 1024, 0.25, seed=4)
    c = o.pack_canonical(L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(), L.perm.numpy(), L.I_dense)
    cl = o.pack_linear_canonical(L.wgate.numpy(), L.perm.numpy(), L.I_dense, "out")
    assert np.array_equal(cl["sp_val"], c["gate_sp_val"]) and np.array_equal(cl["sp_meta"], c["gate_sp_meta"])
    assert np.array_equal(cl["dn"], c["gate_dn"])
    cd = o.pack_linear_canonical(L.wdown.numpy(), L.perm.numpy(), L.I_dense, "in")
    assert np.array_equal(cd["sp_val"], c["down_sp_val"]) and np.array_equal(cd["dn"], c["down_dn"])


def test_linear_error_paths():
    w = np.zeros((8, 8), np.uint8)
    w[2, 4:8] = [0x38, 0x38, 0x38, 0]
    with pytest.raises(o.SpenseOracleError) as e:
        o.pack_linear_canonical(w, None, 0, "out")
    assert e.value.code == "SPENSE_ERR_NOT_2_4" and e.value.where[:3] == (0, 2, 1)
    w[2, 4] = 0x7F
    with pytest.raises(o.SpenseOracleError) as e:
        o.pack_linear_canonical(w, None, 8, "out")               # NaN bytes are rejected in the dense region too
    assert e.value.code == "SPENSE_ERR_NAN_WEIGHT"
    with pytest.raises(o.SpenseOracleError) as e:
        o.pack_linear_canonical(np.zeros((8, 8), np.uint8), np.array([0, 0, 1, 2, 3, 4, 5, 6]), 0, "in")
    assert e.value.code == "SPENSE_ERR_BAD_PERM"
