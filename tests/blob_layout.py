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
    """vals*: [128, 128] compressed bytes (K 256 logical), meta*: [128, 32]."""
    st = np.zeros(SPARSE_STAGE, np.uint8)
    _put_rows_sw128(st[0:OPER], vals0)
    _put_rows_sw128(st[OPER:2 * OPER], vals1)
    for m, meta in enumerate((meta0, meta1)):
        base = 2 * OPER + m * META
        for atom in range(2):
            st[base + atom * 2048: base + (atom + 1) * 2048] = meta[:, atom * 16:(atom + 1) * 16].reshape(-1)
    return st


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
        for j in range(ns):
            out.append(_sparse_stage(gv[r, 128 * j:128 * j + 128], gm[r, 32 * j:32 * j + 32],
                                     uv[r, 128 * j:128 * j + 128], um[r, 32 * j:32 * j + 32]))
    for t in range(I_d // 128):
        r = slice(128 * t, 128 * t + 128)
        for j in range(H // 128):
            out.append(_dense_stage(c["gate_dn"][r, 128 * j:128 * j + 128], c["up_dn"][r, 128 * j:128 * j + 128]))
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
