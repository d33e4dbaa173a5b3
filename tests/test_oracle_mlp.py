"""Pins for the oracle's GEMM / GLU / requant / down chain (O5, O6; T2, T3, T5)."""
import numpy as np
import torch

import spense_inputs as si
from oracle import spense_oracle as o


def _units(b):
    """Independent integer decode: E4M3 byte -> integer multiple of 2^-9 (no table, no floats)."""
    b = int(b)
    e, m = (b >> 3) & 0xF, b & 7
    assert not (e == 15 and m == 7)
    v = m if e == 0 else (8 + m) << (e - 1)
    return -v if b & 0x80 else v


def test_gemm_exact_vs_python_integer_brute_force():
    rng = np.random.default_rng(5)
    M, N, K = 5, 7, 48
    a = rng.integers(0, 256, (M, K)).astype(np.uint8)
    w = rng.integers(0, 256, (N, K)).astype(np.uint8)
    a[(a & 0x7F) == 0x7F] = 0x7E
    w[(w & 0x7F) == 0x7F] = 0x7E
    acc, ab = o.gemm_exact(a, w)
    for m in range(M):
        for n in range(N):
            s = sum(_units(a[m, k]) * _units(w[n, k]) for k in range(K))       # Y = X W^T
            t = sum(abs(_units(a[m, k]) * _units(w[n, k])) for k in range(K))
            assert acc[m, n] * 2.0 ** 18 == s and ab[m, n] * 2.0 ** 18 == t
            assert ab[m, n] >= abs(acc[m, n])


def test_gemm_exactness_bound_at_max_K():
    # worst case: all |448| at K = 27648 stays below 2^53 units of 2^-18 => float64 is exact
    K = 27648
    a = np.full((1, K), 0x7E, np.uint8)
    w = np.full((1, K), 0x7E, np.uint8)
    acc, _ = o.gemm_exact(a, w)
    assert acc[0, 0] == 448.0 * 448.0 * K and 448 * 512 * 448 * 512 * K < 2 ** 53


def test_one_hot_rows_return_weight_columns():
    L = si.make_layer(256, 1024, 0.25, seed=11)
    c = o.pack_canonical(L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(), L.perm.numpy(), L.I_dense)
    g, u, d = o.unpack_canonical(c)
    ks = [0, 3, 130, 255]
    x = np.zeros((len(ks), 256), np.uint8)
    for r, k in enumerate(ks):
        x[r, k] = 0x38                                   # 1.0
    accG, _ = o.gemm_exact(x, g)
    for r, k in enumerate(ks):
        assert np.array_equal(accG[r], o.e4m3_decode(g[:, k]))


def test_dense_case_matches_torch_float8_matmul():
    # p = 100 %: the Spense GEMM is a plain dense FP8 GEMM -> torch's own fp8 decode + matmul
    L = si.make_layer(256, 1024, 1.0, seed=2)
    x, sx = si.make_activations(8, 256, seed=2)
    r, c = o.spense_mlp(x.numpy(), sx.numpy(), L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(),
                        L.w_scale, L.perm.numpy(), L.I_dense, s_h=1.0)
    assert c["gate_sp_val"].shape[0] == 0
    xt = x.view(torch.float8_e4m3fn).double()
    wg = L.wgate[L.perm.long()].view(torch.float8_e4m3fn).double()
    gref = (xt @ wg.T) * (sx.double()[:, None] * L.w_scale[0])
    assert np.array_equal(r["g"], gref.numpy())


def test_permutation_invariance_T2_exact():
    L = si.make_layer(256, 1024, 0.25, seed=0)
    x, sx = si.make_activations(8, 256, seed=0)
    perm = L.perm.numpy().astype(np.int64)
    nz = lambda a: np.where((a & 0x7F) == 0, 0, a)
    # dense MLP on ORIGINAL-order weights, no packing at all
    r0 = o.gate_up(x.numpy(), sx.numpy(), nz(L.wgate.numpy()), nz(L.wup.numpy()), L.w_scale[0], L.w_scale[1], 1.0)
    s_h = o.requant_scale_from_h(r0["h"])
    r0 = o.mlp(x.numpy(), sx.numpy(), nz(L.wgate.numpy()), nz(L.wup.numpy()), nz(L.wdown.numpy()), L.w_scale, s_h)
    r1, _ = o.spense_mlp(x.numpy(), sx.numpy(), L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(),
                         L.w_scale, perm, L.I_dense, s_h)
    assert np.array_equal(r1["h"], r0["h"][:, perm])      # Eq. 4: h is permuted, ...
    assert np.array_equal(r1["hq"], r0["hq"][:, perm])
    assert np.array_equal(r1["y"], r0["y"])               # ... the MLP output is unchanged, exactly
    assert np.abs(r1["y"]).max() > 0


def test_dense_fraction_invariance():
    L = si.make_layer(256, 1024, 0.0, seed=4, all_2_4=True)
    x, sx = si.make_activations(8, 256, seed=4)
    ys = []
    for I_d in (0, 128, 512, 1024):
        r, c = o.spense_mlp(x.numpy(), sx.numpy(), L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(),
                            L.w_scale, None, I_d, s_h=0.01)
        assert c["gate_dn"].shape[0] == I_d
        ys.append(r["y"])
    for y in ys[1:]:
        assert np.array_equal(y, ys[0])


def test_input_split_is_sum_of_two_k_ranges_T5():
    L = si.make_layer(256, 1024, 0.25, seed=6)
    c = o.pack_canonical(L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(), L.perm.numpy(), L.I_dense)
    _, _, d = o.unpack_canonical(c)
    I_s = 1024 - L.I_dense
    hq = np.random.default_rng(0).integers(0, 0x7F, (4, 1024)).astype(np.uint8)
    full = o.down(hq, 0.5, d, L.w_scale[2])["y"]
    sp = o.down(hq[:, :I_s], 0.5, o.expand_rows(c["down_sp_val"], c["down_sp_meta"]), L.w_scale[2])["y"]
    dn = o.down(hq[:, I_s:], 0.5, c["down_dn"], L.w_scale[2])["y"]
    assert np.allclose(full, sp + dn, rtol=0, atol=1e-12 * np.abs(full).max())


def test_glu_closed_forms():
    assert o.silu(np.array([0.0]))[0] == 0.0
    assert abs(o.silu(np.array([40.0]))[0] - 40.0) < 1e-12
    assert abs(o.silu(np.array([-40.0]))[0]) < 1e-12
    assert abs(o.silu(np.array([1.0]))[0] - 1.0 / (1.0 + np.exp(-1.0))) < 1e-15
    # doubling s_x (power of two) doubles g and u exactly
    L = si.make_layer(256, 1024, 0.25, seed=8)
    x, sx = si.make_activations(4, 256, seed=8)
    g, u, _ = o.unpack_canonical(o.pack_canonical(L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(),
                                                  L.perm.numpy(), L.I_dense))
    a = o.gate_up(x.numpy(), sx.numpy(), g, u, L.w_scale[0], L.w_scale[1], 1.0)
    b = o.gate_up(x.numpy(), 2 * sx.numpy(), g, u, L.w_scale[0], L.w_scale[1], 1.0)
    assert np.array_equal(b["g"], 2 * a["g"]) and np.array_equal(b["u"], 2 * a["u"])
    # requant uses the supplied scale: hq = enc(h / s_h)
    s_h = o.requant_scale_from_h(a["h"])
    c = o.gate_up(x.numpy(), sx.numpy(), g, u, L.w_scale[0], L.w_scale[1], s_h)
    assert ((c["hq"] & 0x7F).max(axis=1) == 0x7E).all()
    assert np.array_equal(c["hq"], o.e4m3_encode((c["h"] / s_h[:, None].astype(np.float64)).astype(np.float32)))


def test_small_integer_case_is_integral():
    wg, wu, wd, x = si.make_small_int_case(256, 512, 128, 4, seed=1)
    acc, ab = o.gemm_exact(x.numpy(), wg.numpy())
    assert np.array_equal(acc, np.round(acc)) and ab.max() < 2 ** 24


def test_dynamic_requant_scale_pins():
    """NEXT-1 pins: per token the element of largest |h| lands on +-448 (byte 0x7E / 0xFE), nothing saturates
    beyond it, an all-zero token gets scale 1, and doubling the up-projection's weight scale (a power of
    two: u and so h double exactly, SiLU(g) is untouched) doubles s_h and y while every Hq byte stays the same."""
    L = si.make_layer(256, 1024, 0.25, seed=0)
    x, s_x = si.make_activations(8, 256, seed=0)
    x = x.clone()
    x[3] = 0                                             # an all-zero token
    c = o.pack_canonical(L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(), L.perm.numpy(), L.I_dense)
    wg, wu, wd = o.unpack_canonical(c)
    r = o.mlp_dynamic(x.numpy(), s_x.numpy(), wg, wu, wd, L.w_scale)
    assert r["s_h"].dtype == np.float32 and r["s_h"][3] == 1.0 and not r["hq"][3].any() and not r["y"][3].any()
    for m in range(8):
        if m == 3:
            continue
        j = np.abs(r["h"][m]).argmax()
        assert r["hq"][m, j] & 0x7F == 0x7E
        assert (r["hq"][m] & 0x7F).max() == 0x7E
        assert r["s_h"][m] == np.float32(np.float32(np.abs(r["h"][m]).max()) / np.float32(448.0))
    ws2 = (L.w_scale[0], 2.0 * L.w_scale[1], L.w_scale[2])
    r2 = o.mlp_dynamic(x.numpy(), s_x.numpy(), wg, wu, wd, ws2)
    live = [0, 1, 2, 4, 5, 6, 7]
    assert np.array_equal(r2["s_h"][live], 2.0 * r["s_h"][live])
    assert np.array_equal(r2["hq"], r["hq"])
    assert np.array_equal(r2["y"], 2.0 * r["y"])


def test_down_scale_and_abs_sum_hand_computed():
    """Pin for `down`'s scaling (PAPER.md:125 input-split; Q5/Q10: y = acc * s_h[m] * s_wd): a 3 x 4 x 8
    case written out with a plain Python-integer triple loop over hand-listed small values and explicit
    power-of-two scales, so every product is exact.  Dropping s_wd or s_h[m] from the oracle, applying s_h to the
    wrong axis, or losing the |.| in absY fails here."""
    byte_of = {0: 0x00, 1: 0x38, 2: 0x40, 3: 0x44, -1: 0xB8, -2: 0xC0, -3: 0xC4, 0.5: 0x30, -0.5: 0xB0}
    hq_v = [[1, -2, 0, 3, 0.5, -1, 2, 0],
            [0, 0, -3, 1, 2, -0.5, 1, 1],
            [3, 3, -3, -3, 0, 1, -2, 0.5]]                           # [M=3][K=8]
    wd_v = [[1, 0, -1, 2, 0, 0, 3, -2],
            [0.5, 2, 0, 0, -3, 1, 0, 0],
            [0, -1, 0, 2, 0, -0.5, 0, 1],
            [2, 0, 0, -2, 1, 0, 0, 3]]                               # [N=4][K=8]
    s_h = [0.5, 2.0, 0.25]                                           # per token
    s_wd = 0.25
    hq = np.array([[byte_of[v] for v in row] for row in hq_v], np.uint8)
    wd = np.array([[byte_of[v] for v in row] for row in wd_v], np.uint8)
    r = o.down(hq, np.array(s_h, np.float32), wd, s_wd)
    for m in range(3):
        for n in range(4):
            acc = sum(hq_v[m][k] * wd_v[n][k] for k in range(8))             # Y = Hq Wd^T
            ab = sum(abs(hq_v[m][k] * wd_v[n][k]) for k in range(8))
            assert r["y"][m, n] == acc * s_h[m] * s_wd, (m, n)
            assert r["absY"][m, n] == ab * s_h[m] * s_wd, (m, n)
    assert r["y"][0, 0] == (1 + 6 + 6) * 0.5 * 0.25 and r["y"][1, 1] == (-6 - 0.5) * 2.0 * 0.25   # two entries by hand
    # a scalar s_h applies to every token
    r1 = o.down(hq, 2.0, wd, s_wd)
    assert np.array_equal(r1["y"], r["y"] / np.array(s_h)[:, None] * 2.0)


def test_gate_up_scales_hand_computed():
    """The same for gate_up: g = accG * s_x[m] * s_gate, u = accU * s_x[m] * s_up (Eq. 4)."""
    byte_of = {0: 0x00, 1: 0x38, 2: 0x40, -1: 0xB8, -2: 0xC0}
    x_v = [[1, 2, 0, -1], [0, -2, 2, 1]]
    wg_v = [[1, 0, 0, 2], [0, -1, 1, 0], [2, 2, -2, 0]]
    wu_v = [[0, 1, -1, 0], [1, 1, 0, 0], [0, 0, 2, -2]]
    s_x, s_g, s_u = [0.5, 4.0], 0.25, 2.0
    enc = lambda t: np.array([[byte_of[v] for v in row] for row in t], np.uint8)
    r = o.gate_up(enc(x_v), np.array(s_x, np.float32), enc(wg_v), enc(wu_v), s_g, s_u, 1.0)
    for m in range(2):
        for j in range(3):
            g = sum(x_v[m][k] * wg_v[j][k] for k in range(4)) * s_x[m] * s_g
            u = sum(x_v[m][k] * wu_v[j][k] for k in range(4)) * s_x[m] * s_u
            assert r["g"][m, j] == g and r["u"][m, j] == u
            assert abs(r["h"][m, j] - g / (1.0 + np.exp(-g)) * u) <= 1e-15 * max(1.0, abs(g * u))
