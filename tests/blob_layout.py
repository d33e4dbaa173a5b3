"""Test-side restatement of the packed-blob layout: builds the
expected blob bytes from canonical arrays with plain numpy loops, so the CUDA pack's P3 re-tile
step can be checked byte for byte.  Layout only -- no method arithmetic."""
import numpy as np

OPER = 128 * 128
META = 128 * 32
SPARSE_STAGE = 2 * OPER + 2 * META
DENSE_STAGE = 2 * OPER
HEADER = 1024


def sw128(r, b):
    return (r >> 3) * 1024 + (r & 7) * 128 + ((((b >> 4) ^ (r & 7)) & 7) << 4) + (b & 15)


def _put_rows_sw128(img, rows_bytes):
    """rows_bytes: [128, 128] -> scatter into a 16 KB SWIZZLE_128B K-major image."""
    r = np.arange(128)[:, None]
    b = np.arange(128)[None, :]
    off = (r >> 3) * 1024 + (r & 7) * 128 + ((((b >> 4) ^ (r & 7)) & 7) << 4) + (b & 15)
    img[off] = rows_bytes


def _sparse_stage(vals0, meta0, vals1, meta1):
    """vals*: [128, 128] compressed bytes (K 256 logical), meta*: [128, 32].
    Stage image = operand 0 (values 16 KB, metadata 4 KB as two 128 x 16 B atoms), then operand 1 likewise."""
    st = np.zeros(SPARSE_STAGE, np.uint8)
    for m, (vals, meta) in enumerate(((vals0, meta0), (vals1, meta1))):
        base = m * (OPER + META)
        _put_rows_sw128(st[base:base + OPER], vals)
        for atom in range(2):
            st[base + OPER + atom * 2048: base + OPER + (atom + 1) * 2048] = meta[:, atom * 16:(atom + 1) * 16].reshape(-1)
    return st


def _glu_operands(gate_rows, up_rows):
    """gate_rows, up_rows: [128, n] = the gate / up rows of the 128 intermediate indices of a pair tile.  Operand a
    holds the indices 64 a + [0, 64): operand row 32 q + i = gate row of index 16 q + i, row 32 q + 16 + i = its up row."""
    ops = []
    for a in range(2):
        op = np.zeros_like(gate_rows)
        for q in range(4):
            for i in range(16):
                op[32 * q + i] = gate_rows[64 * a + 16 * q + i]
                op[32 * q + 16 + i] = up_rows[64 * a + 16 * q + i]
        ops.append(op)
    return ops


def _dense_stage(a0, a1):
    st = np.zeros(DENSE_STAGE, np.uint8)
    _put_rows_sw128(st[0:OPER], a0)
    _put_rows_sw128(st[OPER:], a1)
    return st


def _pad_cols(a, n, fill):
    if a.shape[1] >= n:
        return a
    return np.concatenate([a, np.full((a.shape[0], n - a.shape[1]), fill, np.uint8)], axis=1)


def _pad_rows(a, n, fill):
    if a.shape[0] >= n:
        return a
    return np.concatenate([a, np.full((n - a.shape[0], a.shape[1]), fill, np.uint8)], axis=0)


def expected_blob_body(c, H, I, I_d):
    """Everything after the 1 KB header."""
    I_s = I - I_d
    out = []
    ns = (H + 255) // 256
    gv, uv = _pad_cols(c["gate_sp_val"], ns * 128, 0), _pad_cols(c["up_sp_val"], ns * 128, 0)
    gm, um = _pad_cols(c["gate_sp_meta"], ns * 32, 0x44), _pad_cols(c["up_sp_meta"], ns * 32, 0x44)
    for t in range(I_s // 128):
        r = slice(128 * t, 128 * t + 128)
        v0, v1 = _glu_operands(gv[r], uv[r])
        m0, m1 = _glu_operands(gm[r], um[r])
        for j in range(ns):
            out.append(_sparse_stage(v0[:, 128 * j:128 * j + 128], m0[:, 32 * j:32 * j + 32],
                                     v1[:, 128 * j:128 * j + 128], m1[:, 32 * j:32 * j + 32]))
    for t in range(I_d // 128):
        r = slice(128 * t, 128 * t + 128)
        a0, a1 = _glu_operands(c["gate_dn"][r], c["up_dn"][r])
        for j in range(H // 128):
            out.append(_dense_stage(a0[:, 128 * j:128 * j + 128], a1[:, 128 * j:128 * j + 128]))
    # down: 256-row tiles, sparse K stages then dense K stages
    nt = (H + 255) // 256
    ns = (I_s + 255) // 256
    dv = _pad_rows(_pad_cols(c["down_sp_val"], ns * 128, 0), nt * 256, 0)
    dm = _pad_rows(_pad_cols(c["down_sp_meta"], ns * 32, 0x44), nt * 256, 0x44)
    dd = _pad_rows(c["down_dn"], nt * 256, 0)
    for t in range(nt):
        r0, r1 = slice(256 * t, 256 * t + 128), slice(256 * t + 128, 256 * t + 256)
        for j in range(ns):
            out.append(_sparse_stage(dv[r0, 128 * j:128 * j + 128], dm[r0, 32 * j:32 * j + 32],
                                     dv[r1, 128 * j:128 * j + 128], dm[r1, 32 * j:32 * j + 32]))
        for j in range(I_d // 128):
            out.append(_dense_stage(dd[r0, 128 * j:128 * j + 128], dd[r1, 128 * j:128 * j + 128]))
    return np.concatenate(out) if out else np.zeros(0, np.uint8)


def expected_linear_body(c, N, K, n_dense, split):
    """Blob body of spense_pack_linear (everything after the header) from the canonical arrays of ONE matrix.
    in-split : 256-row tiles, each its sparse K stages (K_s padded to 256) then its dense K stages -- the down section.
    out-split: 256-row tiles of the row-permuted matrix, operand a = rows 256 t + 128 a + [0, 128) in natural order; the
               sparse tiles (ceil(K / 256) sparse stages each) first, then the dense tiles (K / 128 dense stages each,
               a last half tile zero padded)."""
    out = []
    if split == "in":
        k_s = K - n_dense
        nt, ns = (N + 255) // 256, (k_s + 255) // 256
        v = _pad_rows(_pad_cols(c["sp_val"], ns * 128, 0), nt * 256, 0)
        m = _pad_rows(_pad_cols(c["sp_meta"], ns * 32, 0x44), nt * 256, 0x44)
        d = _pad_rows(c["dn"], nt * 256, 0)
        for t in range(nt):
            r0, r1 = slice(256 * t, 256 * t + 128), slice(256 * t + 128, 256 * t + 256)
            for j in range(ns):
                out.append(_sparse_stage(v[r0, 128 * j:128 * j + 128], m[r0, 32 * j:32 * j + 32],
                                         v[r1, 128 * j:128 * j + 128], m[r1, 32 * j:32 * j + 32]))
            for j in range(n_dense // 128):
                out.append(_dense_stage(d[r0, 128 * j:128 * j + 128], d[r1, 128 * j:128 * j + 128]))
    else:
        n_s = N - n_dense
        ns = (K + 255) // 256
        v, m = _pad_cols(c["sp_val"], ns * 128, 0), _pad_cols(c["sp_meta"], ns * 32, 0x44)
        for t in range(n_s // 256):
            r0, r1 = slice(256 * t, 256 * t + 128), slice(256 * t + 128, 256 * t + 256)
            for j in range(ns):
                out.append(_sparse_stage(v[r0, 128 * j:128 * j + 128], m[r0, 32 * j:32 * j + 32],
                                         v[r1, 128 * j:128 * j + 128], m[r1, 32 * j:32 * j + 32]))
        ntd = (n_dense + 255) // 256
        d = _pad_rows(c["dn"], ntd * 256, 0)
        for t in range(ntd):
            r0, r1 = slice(256 * t, 256 * t + 128), slice(256 * t + 128, 256 * t + 256)
            for j in range(K // 128):
                out.append(_dense_stage(d[r0, 128 * j:128 * j + 128], d[r1, 128 * j:128 * j + 128]))
    return np.concatenate(out) if out else np.zeros(0, np.uint8)
