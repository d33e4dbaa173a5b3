"""Pins for the oracle's permutation + 2:4 canonical pack / unpack (O3, O4; T1, T4, T6)."""
import os

import numpy as np
import pytest

import spense_inputs as si
from oracle import spense_oracle as o


def _table(golden_dir):
    rows = []
    with open(os.path.join(golden_dir, "pack_2of4_table.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            lhs, rhs = line.split("->")
            rows.append(([int(t, 16) for t in lhs.split()], [int(t, 16) for t in rhs.split()]))
    return rows


def test_group_rule_matches_hand_table(golden_dir):
    for b4, (nib, v0, v1) in _table(golden_dir):
        assert o.compress_group(b4) == (nib, v0, v1), b4
        assert nib in o.NIBBLES_VALID


def test_vectorised_pack_matches_group_rule_exhaustive():
    # every group over a 5-symbol alphabet {+0,-0,a,b,-a} with <= 2 non-zeros, packed 2 groups / row
    alpha = [0x00, 0x80, 0x38, 0x41, 0xB8]
    groups = [(a, b, c, d) for a in alpha for b in alpha for c in alpha for d in alpha
              if sum((v & 0x7F) != 0 for v in (a, b, c, d)) <= 2]
    w = np.array(groups + groups[::-1], dtype=np.uint8).reshape(2, len(groups), 4)
    w = np.concatenate([w[0], w[1]], axis=1)                   # [G, 8]: two groups per row
    vals, meta = o.compress_rows(w)
    for r in range(w.shape[0]):
        n0, a0, a1 = o.compress_group(w[r, 0:4])
        n1, b0, b1 = o.compress_group(w[r, 4:8])
        assert list(vals[r]) == [a0, a1, b0, b1]
        assert meta[r, 0] == (n0 | (n1 << 4))                  # low nibble = lower K
        assert (meta[r, 0] & 0xF) in o.NIBBLES_VALID and (meta[r, 0] >> 4) in o.NIBBLES_VALID
    # unpack(pack(W)) == W with -0 -> +0
    back = o.expand_rows(vals, meta)
    assert np.array_equal(back, np.where((w & 0x7F) == 0, 0, w))


def test_errors_not_2_4_nan_perm():
    w = np.zeros((4, 16), dtype=np.uint8)
    w[2, 4:7] = 0x38                                            # 3 non-zeros in row 2 group 1
    with pytest.raises(o.SpenseOracleError) as e:
        o.compress_rows(w, matrix_id=1)
    assert e.value.code == "SPENSE_ERR_NOT_2_4" and e.value.where[:3] == (1, 2, 1)
    w[:] = 0
    w[1, 3] = 0xFF
    with pytest.raises(o.SpenseOracleError) as e:
        o.compress_rows(w)
    assert e.value.code == "SPENSE_ERR_NAN_WEIGHT"
    with pytest.raises(o.SpenseOracleError) as e:
        o.check_perm(np.array([0, 1, 1, 3]), 4)
    assert e.value.code == "SPENSE_ERR_BAD_PERM"
    with pytest.raises(o.SpenseOracleError):
        o.compress_group([0x38, 0x38, 0x38, 0])


def test_perm_stable_partition_and_dense_last():
    perm = o.perm_from_dense_idx(10, [7, 2, 5])
    assert list(perm) == [0, 1, 3, 4, 6, 8, 9, 2, 5, 7]        # T4: dense block is the LAST block
    assert list(o.perm_from_dense_idx(6, o.spensegpt_dense_idx(6, 2))) == [0, 1, 2, 3, 4, 5]
    assert o.dense_count(27648, 0.10) == 2816 and o.dense_count(25600, 0.25) == 6400
    assert o.dense_count(1024, 0.25) == 256


def test_generator_output_is_2_4_in_permuted_sparse_region_T1():
    L = si.make_layer(256, 1024, 0.25, seed=0)
    perm = L.perm.numpy().astype(np.int64)
    assert np.array_equal(perm, o.perm_from_dense_idx(1024, L.dense_idx.numpy()))
    I_s = 1024 - L.I_dense
    g = L.wgate.numpy()[perm][:I_s].reshape(I_s, -1, 4)
    d = L.wdown.numpy()[:, perm][:, :I_s].reshape(256, -1, 4)
    assert (((g & 0x7F) != 0).sum(axis=2) <= 2).all()
    assert (((d & 0x7F) != 0).sum(axis=2) <= 2).all()
    # and the dense region is NOT 2:4 (otherwise the hybrid is not exercised)
    gd = L.wgate.numpy()[perm][I_s:].reshape(L.I_dense, -1, 4)
    assert (((gd & 0x7F) != 0).sum(axis=2) > 2).any()


def test_pack_unpack_roundtrip_T3_and_layout():
    L = si.make_layer(256, 1024, 0.25, seed=3)
    c = o.pack_canonical(L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(), L.perm.numpy(), L.I_dense)
    I_s = 1024 - L.I_dense
    assert c["gate_sp_val"].shape == (I_s, 128) and c["gate_sp_meta"].shape == (I_s, 32)
    assert c["down_sp_val"].shape == (256, I_s // 2) and c["down_sp_meta"].shape == (256, I_s // 8)
    assert c["gate_dn"].shape == (L.I_dense, 256) and c["down_dn"].shape == (256, L.I_dense)
    for m in (c["gate_sp_meta"], c["up_sp_meta"], c["down_sp_meta"]):                 # T6
        assert np.isin(m & 0xF, o.NIBBLES_VALID).all() and np.isin(m >> 4, o.NIBBLES_VALID).all()
    g, u, d = o.unpack_canonical(c)
    perm = L.perm.numpy().astype(np.int64)
    nz = lambda a: np.where((a & 0x7F) == 0, 0, a)
    assert np.array_equal(g, nz(L.wgate.numpy()[perm]))
    assert np.array_equal(u, nz(L.wup.numpy()[perm]))
    assert np.array_equal(d, nz(L.wdown.numpy()[:, perm]))
    # a violating weight in the sparse region is rejected, the same weight in the dense region is fine
    wg = L.wgate.numpy().copy()
    wg[perm[I_s + 1], 0:4] = 0x38
    o.pack_canonical(wg, L.wup.numpy(), L.wdown.numpy(), L.perm.numpy(), L.I_dense)
    wg[perm[5], 8:12] = 0x38
    with pytest.raises(o.SpenseOracleError) as e:
        o.pack_canonical(wg, L.wup.numpy(), L.wdown.numpy(), L.perm.numpy(), L.I_dense)
    assert e.value.code == "SPENSE_ERR_NOT_2_4" and e.value.where[:3] == (0, 5, 2)
