"""CPU oracle for the Spense hybrid sparse-dense FP8 GLU MLP (arxiv/paper_2606_10445).

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import it.  It shares no
code with the CUDA path (``paper_2606_10445_b200/``) and never imports it.

What it computes, and where the paper says so (citations are PAPER.md lines):

* 2:4 semi-structured sparsity, ``||W[i,4j:4j+4]||_0 <= 2`` for ``W in R^{N x K}``, groups along K
  -- Eq. 1.  Compressed storage keeps "only non-zero weights and their positions
  ... a few bits per group" -- PAPER.md:74.
* Spense format: each weight is one contiguous 2:4 region plus one contiguous dense region
  -- Sec. 3.2.  Output-split (gate/up: rows split) and input-split (down:
  reduction dim split, sparse product first, dense product accumulated into the same output).
* Intermediate-index permutation P that leaves the MLP unchanged -- Eq. 4, PAPER.md:133-143;
  the dense indices are placed last ("lower/right part") -- PAPER.md:149, 202.
* GLU MLP: ``MLP(X) = (X W_up^T * sigma(X W_gate^T)) W_down^T`` -- Eq. 4.

The Spense GEMM reaches exactly (up to rounding order) the dense GEMM of the reconstructed weight,
so the oracle is that plain definition: decode FP8, expand values + metadata back to a dense
matrix, run the GEMMs in float64.  Every E4M3 value is an integer multiple of 2^-9 with magnitude
<= 448 < 2^9, so every product is an integer multiple of 2^-18 below 2^18 and a K <= 2^15 dot
product stays below 2^51 units: the float64 accumulators are EXACT and independent of summation
order (numpy's BLAS matmul may therefore serve as the GEMM step).

Readings of the paper where it is silent / garbled:
Q1/Q2 dense set = LAST I_d indices; Q4 sigma = SiLU; Q5 E4M3-FN, per-tensor weight scale
amax/448, per-token activation scale, RNE, saturating; Q6 nibble = i0 | i1<<2; Q7 filler rule;
Q8 sparse region first; Q9 stable partition; Q10 requant scale s_h is an input.

Parity pins: tests/test_oracle_*.py (E4M3 vs torch / ml_dtypes, hand-enumerated 2:4 table,
brute-force integer GEMM, permutation invariance, closed forms).  No function here is unpinned.
"""
from __future__ import annotations

import numpy as np

E4M3_MAX = 448.0
NIBBLES_VALID = (4, 8, 9, 12, 13, 14)  # C(4,2) position pairs, nibble = i0 | i1 << 2


class SpenseOracleError(ValueError):
    """Raised for inputs the method rejects; ``code`` names the C-ABI status it corresponds to."""

    def __init__(self, code: str, where=None):
        super().__init__(f"{code} at {where}")
        self.code = code
        self.where = where


# --------------------------------------------------------------------------------------
# O1  E4M3 (FN variant) codec: bias 7, 3 mantissa bits, no inf, NaN = 0x7F / 0xFF, max 448.
# --------------------------------------------------------------------------------------
def e4m3_decode_table() -> np.ndarray:
    """All 256 byte values as float64 (NaN for 0x7F and 0xFF)."""
    t = np.empty(256, dtype=np.float64)
    for b in range(256):
        sign = -1.0 if (b & 0x80) else 1.0
        e = (b >> 3) & 0xF
        m = b & 0x7
        if e == 0xF and m == 0x7:
            t[b] = np.nan
        elif e == 0:
            t[b] = sign * (m / 8.0) * 2.0 ** -6          # subnormal: m * 2^-9
        else:
            t[b] = sign * (1.0 + m / 8.0) * 2.0 ** (e - 7)
    return t


_DEC = e4m3_decode_table()


def e4m3_decode(b: np.ndarray) -> np.ndarray:
    """uint8 -> float64."""
    return _DEC[np.asarray(b, dtype=np.uint8)]


def e4m3_encode(x: np.ndarray) -> np.ndarray:
    """float32 -> E4M3 byte: clamp to [-448, 448] (saturate), then round to nearest even on the
    E4M3 grid (subnormals included).  NaN -> 0x7F | sign.  -0 keeps its sign bit (0x80)."""
    x = np.asarray(x, dtype=np.float32)
    sign = (x.view(np.uint32) >> 31).astype(np.uint8) << 7
    a = np.abs(x.astype(np.float64))
    nan = np.isnan(a)
    a = np.where(nan, 0.0, np.minimum(a, E4M3_MAX))
    out = np.zeros(a.shape, dtype=np.int64)
    sub = a < 2.0 ** -6
    # subnormal grid: multiples of 2^-9; q == 8 is the smallest normal, whose byte is also 8
    out_sub = np.rint(a * 512.0).astype(np.int64)
    # normal: a = f * 2^E with f in [0.5, 1)  ->  a = (2f) * 2^(E-1), mantissa 2f in [1, 2)
    f, E = np.frexp(np.where(sub, 1.0, a))
    e = E.astype(np.int64) - 1
    m = np.rint((2.0 * f - 1.0) * 8.0).astype(np.int64)   # exact product, RNE to 3 bits
    carry = m == 8
    e = np.where(carry, e + 1, e)
    m = np.where(carry, 0, m)
    out_norm = ((e + 7) << 3) | m
    out = np.where(sub, out_sub, out_norm)
    out = np.minimum(out, 0x7E)
    out = np.where(nan, 0x7F, out)
    return (out.astype(np.uint8) | sign).astype(np.uint8)


# --------------------------------------------------------------------------------------
# O2  quantise (Q5): scale = amax / 448 in fp32 (1 if amax == 0); q = enc(x / scale), fp32 divide.
# --------------------------------------------------------------------------------------
def quantize_per_tensor(x: np.ndarray):
    x = np.asarray(x, dtype=np.float32)
    amax = np.float32(np.max(np.abs(x))) if x.size else np.float32(0)
    s = np.float32(amax / np.float32(E4M3_MAX)) if amax > 0 else np.float32(1.0)
    q = e4m3_encode((x / s).astype(np.float32))
    return q, s


def quantize_per_row(x: np.ndarray):
    x = np.asarray(x, dtype=np.float32)
    amax = np.max(np.abs(x), axis=1).astype(np.float32) if x.shape[1] else np.zeros(x.shape[0], np.float32)
    s = np.where(amax > 0, (amax / np.float32(E4M3_MAX)).astype(np.float32), np.float32(1.0)).astype(np.float32)
    q = e4m3_encode((x / s[:, None]).astype(np.float32))
    return q, s


# --------------------------------------------------------------------------------------
# D4/D5  permutation (Eq. 4; Q9: stable partition, sparse first, dense last).
# --------------------------------------------------------------------------------------
def dense_count(I: int, p: float, align: int = 128) -> int:
    """Q3: I_d = round(p*I/align)*align ("approximately pN indices ... alignment")."""
    return int(round(p * I / align)) * align


def perm_from_dense_idx(I: int, dense_idx) -> np.ndarray:
    """perm[new] = old.  Non-dense indices first in ascending original order, then the dense
    indices in ascending original order (dense region last)."""
    dense_idx = np.asarray(dense_idx, dtype=np.int64)
    if dense_idx.size and (dense_idx.min() < 0 or dense_idx.max() >= I):
        raise SpenseOracleError("SPENSE_ERR_ARG", "dense index out of range")
    if np.unique(dense_idx).size != dense_idx.size:
        raise SpenseOracleError("SPENSE_ERR_ARG", "duplicate dense index")
    is_dense = np.zeros(I, dtype=bool)
    is_dense[dense_idx] = True
    idx = np.arange(I, dtype=np.int64)
    return np.concatenate([idx[~is_dense], idx[is_dense]]).astype(np.int32)


def spensegpt_dense_idx(I: int, I_d: int) -> np.ndarray:
    """SpenseGPT choice (Eq. 5 PAPER.md:155 with reading Q1): the last I_d indices."""
    return np.arange(I - I_d, I, dtype=np.int64)


def prune_2to4_group(vals):
    """Magnitude 2:4 mask of ONE group of 4 weights (the test generator's rule; stands in for the
    mask SparseGPT would choose): keep the 2 of largest |w|, ties to the lower index.  Plain Python."""
    order = sorted(range(4), key=lambda i: (-abs(float(vals[i])), i))
    keep = sorted(order[:2])
    return [i in keep for i in range(4)]


def prune_2to4_magnitude(wgate, wup, wdown, perm, I_dense: int):
    """NEXT-4 front-end, first slice: magnitude 2:4 pruning of the SPARSE region in PERMUTED intermediate order
    ("permute ... then apply [the pruner] while protecting the selected dense indices"; Eq. 1
    PAPER.md:67-72: groups of 4 along K): rows [0, I_s) of P^T W_gate / P^T W_up along H, columns [0, I_s) of W_down P
    along the permuted intermediate dimension (reading Q9b).  Pruned entries become +0.  Returns new arrays in the
    ORIGINAL index order (the layout spense_pack takes)."""
    wgate, wup, wdown = (np.array(a, copy=True) for a in (wgate, wup, wdown))
    I, H = wgate.shape
    perm = np.arange(I) if perm is None else np.asarray(perm, dtype=np.int64)
    I_s = I - I_dense

    def mask_lastdim(a):                                   # a [..., 4 g + i]: keep mask by the scalar rule, vectorised
        g = np.abs(a.reshape(-1, 4)).astype(np.float64)
        idx = np.arange(4)
        # rank of element i = number of elements that beat it (larger |w|, or equal |w| and lower index)
        beats = (g[:, None, :] > g[:, :, None]) | ((g[:, None, :] == g[:, :, None]) & (idx[None, None, :] < idx[None, :, None]))
        return (beats.sum(axis=2) < 2).reshape(a.shape)

    for w in (wgate, wup):
        rows = perm[:I_s]
        blk = w[rows]
        w[rows] = np.where(mask_lastdim(blk), blk, 0)
    cols = perm[:I_s]
    blk = wdown[:, cols]
    wdown[:, cols] = np.where(mask_lastdim(blk), blk, 0)
    return wgate, wup, wdown


def sparsegpt_2to4(w, hinv, k_sparse: int, on_group=None):
    """NEXT-4: SparseGPT's 2:4 column sweep with the dense columns on the right as compensation buffer (PAPER.md:98-111,
    Eqs. 2-3; "placing dense columns on the right keeps them available as a compensation buffer";
    PAPER.md:202 "apply SparseGPT ... to the sparse regions while protecting the selected dense indices").

    w: float [N, K], columns in PERMUTED order (sparse columns [0, k_sparse) first, k_sparse % 4 == 0, dense columns
    last); hinv: H^-1 [K, K] of the layer input Hessian H = X^T X (symmetric positive definite; damping is the caller's
    business).  Follows the paper's description step by step, in float64:
      * columns are processed from left to right; "once a column is processed, its values are frozen" and "the induced
        error is then compensated by updating only the columns that have not yet been processed";
      * Hi is the inverse Hessian of the NOT YET PROCESSED columns ("reuse shared inverse-Hessian information across
        rows"): after column j it loses row / column j by Gaussian elimination, which is the textbook inverse of the
        remaining principal sub-matrix of H (pinned against numpy.linalg.inv in the tests);
      * "for 2:4 sparsity, within each group, SparseGPT selects the weights to prune using the OBS-based error criterion"
        (PAPER.md:111): when the sweep reaches a group of 4 columns it computes, per row, eps_c = w_c^2 / [Hi_c]_cc
        (Eq. 3) for its 4 columns c, with the current w and with [Hi_c]_cc the diagonal entry column c will have when it
        is reached (reading Q24: SparseGPT's own choice), and marks the 2 columns of smallest eps for pruning (ties:
        the lower column is pruned first);
      * a marked weight w_m is removed with Eq. 3: w += delta_m = -w_m / [Hi]_mm * Hi[m, :] over the unprocessed
        columns (which makes w_m itself exactly 0); an unmarked weight is kept as it is.
    Columns >= k_sparse are never pruned: they only receive compensation.  Returns (w_new, pruned_mask).
    on_group (test hook, no arithmetic of its own): called as on_group(j, eps, d) with the [N, 4] criterion values the
    group starting at column j was decided on and the 4 diagonal entries [Hi_c]_cc they were divided by."""
    W = np.array(w, dtype=np.float64, copy=True)
    N, K = W.shape
    assert 0 <= k_sparse <= K and k_sparse % 4 == 0
    Hi = np.array(hinv, dtype=np.float64, copy=True)          # rows / columns < j are dead once column j is reached
    pruned = np.zeros((N, K), dtype=bool)
    for j in range(k_sparse):
        if j % 4 == 0:
            blk = Hi[j:j + 4, j:j + 4].copy()                 # the 4 x 4 corner decides the 4 diagonals the group will see
            d = np.empty(4)
            for c in range(4):
                d[c] = blk[c, c]
                blk[c + 1:, c + 1:] -= np.outer(blk[c + 1:, c], blk[c, c + 1:]) / blk[c, c]
            eps = W[:, j:j + 4] ** 2 / d[None, :]
            if on_group is not None:
                on_group(j, eps, d)
            order = np.argsort(eps, axis=1, kind="stable")    # stable: ties -> the lower column first
            for r in range(N):
                pruned[r, j + order[r, 0]] = True
                pruned[r, j + order[r, 1]] = True
        err = np.where(pruned[:, j], W[:, j] / Hi[j, j], 0.0)
        W[:, j:] -= err[:, None] * Hi[j, j:][None, :]
        W[pruned[:, j], j] = 0.0
        Hi[j + 1:, j + 1:] -= np.outer(Hi[j + 1:, j], Hi[j, j + 1:]) / Hi[j, j]
    return W, pruned


def check_perm(perm: np.ndarray, I: int):
    perm = np.asarray(perm)
    if perm.shape != (I,) or perm.min(initial=0) < 0 or perm.max(initial=0) >= I \
            or np.unique(perm).size != I:
        raise SpenseOracleError("SPENSE_ERR_BAD_PERM")


# --------------------------------------------------------------------------------------
# O3  canonical pack (P1 permute, P2 validate + compress).  Eq. 1 PAPER.md:69.
# --------------------------------------------------------------------------------------
def compress_group(b4):
    """One group of 4 consecutive bytes along K -> (nibble, v0, v1).  The definition (Q6, Q7):

    "non-zero" <=> (byte & 0x7F) != 0.  kept = positions of the non-zero bytes (at most 2, Eq. 1);
    while fewer than 2 are kept, add the smallest position not yet kept; sort -> i0 < i1.
    nibble = i0 | i1 << 2.  v0, v1 = the bytes at i0, i1, except that a zero byte (+0 or -0)
    is stored as 0x00.  Plain Python; the vectorised routine below is checked against it."""
    b4 = [int(v) for v in b4]
    for v in b4:
        if (v & 0x7F) == 0x7F:
            raise SpenseOracleError("SPENSE_ERR_NAN_WEIGHT")
    kept = [i for i in range(4) if (b4[i] & 0x7F) != 0]
    if len(kept) > 2:
        raise SpenseOracleError("SPENSE_ERR_NOT_2_4")
    i = 0
    while len(kept) < 2:
        if i not in kept:
            kept.append(i)
        i += 1
    kept.sort()
    i0, i1 = kept
    v0 = b4[i0] if (b4[i0] & 0x7F) else 0
    v1 = b4[i1] if (b4[i1] & 0x7F) else 0
    return i0 | (i1 << 2), v0, v1


def _mask_lut():
    """non-zero mask (bit i = position i non-zero) -> (i0, i1), from compress_group's rule."""
    lut = np.full((16, 2), -1, dtype=np.int64)
    for mask in range(16):
        if bin(mask).count("1") > 2:
            continue
        nib, _, _ = compress_group([0x38 if (mask >> i) & 1 else 0 for i in range(4)])
        lut[mask] = (nib & 3, nib >> 2)
    return lut


_LUT = _mask_lut()


def compress_rows(w: np.ndarray, matrix_id: int = 0):
    """w: uint8 [R, K] with K % 8 == 0, every group of 4 along K 2:4-compliant.
    Returns vals uint8 [R, K/2] and meta uint8 [R, K/8] (2 nibbles per byte, low nibble = lower K).
    Raises NAN_WEIGHT / NOT_2_4 with where = (matrix, row, group, count) of the first offender in
    (row, group) order."""
    w = np.asarray(w, dtype=np.uint8)
    R, K = w.shape
    assert K % 8 == 0
    g = w.reshape(R, K // 4, 4)
    nanb = (g & 0x7F) == 0x7F
    if nanb.any():
        r, c = np.argwhere(nanb.any(axis=2))[0]
        raise SpenseOracleError("SPENSE_ERR_NAN_WEIGHT", (matrix_id, int(r), int(c), int(nanb.any(axis=2).sum())))
    nz = (g & 0x7F) != 0
    bad = nz.sum(axis=2) > 2
    if bad.any():
        r, c = np.argwhere(bad)[0]
        raise SpenseOracleError("SPENSE_ERR_NOT_2_4", (matrix_id, int(r), int(c), int(bad.sum())))
    mask = (nz * np.array([1, 2, 4, 8])).sum(axis=2)
    i0 = _LUT[mask, 0]
    i1 = _LUT[mask, 1]
    v0 = np.take_along_axis(g, i0[..., None], axis=2)[..., 0]
    v1 = np.take_along_axis(g, i1[..., None], axis=2)[..., 0]
    v0 = np.where((v0 & 0x7F) != 0, v0, 0).astype(np.uint8)
    v1 = np.where((v1 & 0x7F) != 0, v1, 0).astype(np.uint8)
    vals = np.stack([v0, v1], axis=2).reshape(R, K // 2)
    nib = (i0 | (i1 << 2)).astype(np.uint8)                       # [R, K/4]
    meta = (nib[:, 0::2] | (nib[:, 1::2] << 4)).astype(np.uint8)  # [R, K/8]
    return vals, meta


def expand_rows(vals: np.ndarray, meta: np.ndarray) -> np.ndarray:
    """Inverse of compress_rows: zeros where the metadata does not point (O4)."""
    vals = np.asarray(vals, dtype=np.uint8)
    meta = np.asarray(meta, dtype=np.uint8)
    R, K8 = meta.shape
    K = K8 * 8
    nib = np.empty((R, K // 4), dtype=np.uint8)
    nib[:, 0::2] = meta & 0xF
    nib[:, 1::2] = meta >> 4
    i0 = (nib & 3).astype(np.int64)
    i1 = (nib >> 2).astype(np.int64)
    out = np.zeros((R, K // 4, 4), dtype=np.uint8)
    v = vals.reshape(R, K // 4, 2)
    np.put_along_axis(out, i0[..., None], v[..., 0:1], axis=2)
    np.put_along_axis(out, i1[..., None], v[..., 1:2], axis=2)
    return out.reshape(R, K)


def pack_canonical(wgate, wup, wdown, perm, I_dense: int) -> dict:
    """P1 + P2.  wgate, wup: uint8 [I, H] (original index order); wdown: uint8 [H, I];
    perm[new] = old or None (identity).  Sparse region = permuted indices [0, I_s), dense region
    = [I_s, I) (Q8).  gate/up are 2:4 along H; down is 2:4 along the PERMUTED intermediate
    dimension (Q9b).  Returns the canonical arrays of include/spense.h."""
    wgate = np.asarray(wgate, dtype=np.uint8)
    wup = np.asarray(wup, dtype=np.uint8)
    wdown = np.asarray(wdown, dtype=np.uint8)
    I, H = wgate.shape
    assert wup.shape == (I, H) and wdown.shape == (H, I)
    if perm is None:
        perm = np.arange(I, dtype=np.int32)
    check_perm(perm, I)
    perm = np.asarray(perm, dtype=np.int64)
    I_s = I - I_dense
    g = wgate[perm]            # P^T W_gate : rows permuted
    u = wup[perm]
    d = wdown[:, perm]         # W_down P   : columns permuted
    for mid, m in enumerate((g, u, d)):
        if ((m & 0x7F) == 0x7F).any():
            r, c = np.argwhere((m & 0x7F) == 0x7F)[0]
            raise SpenseOracleError("SPENSE_ERR_NAN_WEIGHT", (mid, int(r), int(c) // 4, -1))
    gv, gm = compress_rows(g[:I_s], 0) if I_s else (np.zeros((0, H // 2), np.uint8), np.zeros((0, H // 8), np.uint8))
    uv, um = compress_rows(u[:I_s], 1) if I_s else (np.zeros((0, H // 2), np.uint8), np.zeros((0, H // 8), np.uint8))
    if I_s:
        dv, dm = compress_rows(d[:, :I_s], 2)
    else:
        dv, dm = np.zeros((H, 0), np.uint8), np.zeros((H, 0), np.uint8)
    return dict(perm=perm.astype(np.int32),
                gate_sp_val=gv, gate_sp_meta=gm, up_sp_val=uv, up_sp_meta=um,
                gate_dn=g[I_s:].copy(), up_dn=u[I_s:].copy(),
                down_sp_val=dv, down_sp_meta=dm, down_dn=d[:, I_s:].copy())


def unpack_canonical(c: dict):
    """O4: rebuild dense W~gate, W~up [I, H] and W~down [H, I] (bytes, PERMUTED index order)."""
    g = np.concatenate([expand_rows(c["gate_sp_val"], c["gate_sp_meta"]), c["gate_dn"]], axis=0)
    u = np.concatenate([expand_rows(c["up_sp_val"], c["up_sp_meta"]), c["up_dn"]], axis=0)
    d = np.concatenate([expand_rows(c["down_sp_val"], c["down_sp_meta"]), c["down_dn"]], axis=1)
    return g, u, d


# --------------------------------------------------------------------------------------
# O5/O6  the MLP itself (Eq. 4; Sec. 3.2) in exact / float64 arithmetic.
# --------------------------------------------------------------------------------------
def silu(g: np.ndarray) -> np.ndarray:
    """sigma(g)*g with sigma the logistic function (Q4): g / (1 + exp(-g)), float64."""
    g = np.asarray(g, dtype=np.float64)
    with np.errstate(over="ignore"):
        return g / (1.0 + np.exp(-g))


def gemm_exact(a_bytes: np.ndarray, w_bytes: np.ndarray):
    """acc[m, n] = sum_k dec(a[m,k]) * dec(w[n,k])  (Y = X W^T, PAPER.md:67 + footnote PAPER.md:92)
    and abs[m, n] = sum_k |dec(a[m,k]) * dec(w[n,k])|; both exact in float64 (module docstring)."""
    a = e4m3_decode(a_bytes)
    w = e4m3_decode(w_bytes)
    return a @ w.T, np.abs(a) @ np.abs(w).T


def gate_up(xq, s_x, wg_bytes, wu_bytes, s_wg, s_wu, s_h):
    """G1-G3.  xq uint8 [M, H], s_x f32 [M]; wg/wu bytes [I, H]; s_h scalar or [M].
    g = accG * (s_x[m] * s_wg), u likewise (float64), h = silu(g) * u,
    hq = enc(float32(h / s_h[m])).  Returns dict with g, u, h, hq, absG, absU (scaled like g, u)."""
    s_x = np.asarray(s_x, dtype=np.float64).reshape(-1, 1)
    accG, absG = gemm_exact(xq, wg_bytes)
    accU, absU = gemm_exact(xq, wu_bytes)
    g = accG * (s_x * float(s_wg))
    u = accU * (s_x * float(s_wu))
    h = silu(g) * u
    s_h = np.broadcast_to(np.asarray(s_h, dtype=np.float64).reshape(-1, 1), (xq.shape[0], 1))
    hq = e4m3_encode((h / s_h).astype(np.float32))
    return dict(g=g, u=u, h=h, hq=hq, absG=absG * (s_x * float(s_wg)), absU=absU * (s_x * float(s_wu)))


def down(hq, s_h, wd_bytes, s_wd):
    """D1-D2.  y = accY * (s_h[m] * s_wd) with accY = sum over the sparse K range + sum over the
    dense K range of the reconstructed weight (input-split) = one exact sum."""
    M = hq.shape[0]
    s_h = np.broadcast_to(np.asarray(s_h, dtype=np.float64).reshape(-1, 1), (M, 1))
    acc, ab = gemm_exact(hq, wd_bytes)
    sc = s_h * float(s_wd)
    return dict(y=acc * sc, absY=ab * sc)


def mlp(xq, s_x, wg_bytes, wu_bytes, wd_bytes, w_scale, s_h):
    """Whole path on dense (reconstructed, permuted-order) weight bytes."""
    r = gate_up(xq, s_x, wg_bytes, wu_bytes, w_scale[0], w_scale[1], s_h)
    r.update(down(r["hq"], s_h, wd_bytes, w_scale[2]))
    return r


def spense_mlp(xq, s_x, wgate, wup, wdown, w_scale, perm, I_dense, s_h):
    """The method end to end: pack (permute + compress) -> reconstruct -> dense MLP (T3)."""
    c = pack_canonical(wgate, wup, wdown, perm, I_dense)
    g, u, d = unpack_canonical(c)
    return mlp(xq, s_x, g, u, d, w_scale, s_h), c


# --------------------------------------------------------------------------------------
# Stand-alone Spense linears (Sec. 3.2): the format is defined per weight matrix.
# --------------------------------------------------------------------------------------
def pack_linear_canonical(w, perm, n_dense: int, split: str) -> dict:
    """ONE weight W [N, K] as "the semi-structured sparse part and the dense part".
    split == "out" (output-split): perm[new] = old over the N rows; in permuted order the
    sparse rows [0, N_s) are 2:4 along K, the dense rows [N_s, N) come last.
    split == "in" (input-split): perm over the K columns; the sparse columns [0, K_s) are 2:4 along the
    PERMUTED K (Q9b), the dense columns come last.  Returns perm, sp_val, sp_meta, dn as in
    include/spense.h (spense_linear_canon_t)."""
    w = np.asarray(w, dtype=np.uint8)
    N, K = w.shape
    assert split in ("out", "in")
    n = N if split == "out" else K
    if perm is None:
        perm = np.arange(n, dtype=np.int32)
    check_perm(perm, n)
    perm = np.asarray(perm, dtype=np.int64)
    wp = w[perm] if split == "out" else w[:, perm]
    if ((wp & 0x7F) == 0x7F).any():
        r, c = np.argwhere((wp & 0x7F) == 0x7F)[0]
        raise SpenseOracleError("SPENSE_ERR_NAN_WEIGHT", (0, int(r), int(c) // 4, -1))
    n_s = n - n_dense
    if split == "out":
        sp, dn = wp[:n_s], wp[n_s:]
    else:
        sp, dn = wp[:, :n_s], wp[:, n_s:]
    if sp.size:
        v, m = compress_rows(sp, 0)
    else:
        v, m = np.zeros((sp.shape[0], sp.shape[1] // 2), np.uint8), np.zeros((sp.shape[0], sp.shape[1] // 8), np.uint8)
    return dict(perm=perm.astype(np.int32), sp_val=v, sp_meta=m, dn=dn.copy(), split=split)


def unpack_linear_canonical(c: dict) -> np.ndarray:
    """Rebuild the dense W~ [N, K] bytes in PERMUTED order (zeros where the metadata does not point)."""
    sp = expand_rows(c["sp_val"], c["sp_meta"])
    return np.concatenate([sp, c["dn"]], axis=0 if c["split"] == "out" else 1)


def linear(xq, s_x, w_bytes, s_w):
    """y[m, n] = (sum_k dec(x[m,k]) dec(w[n,k])) * s_x[m] * s_w (Y = X W^T) and its
    sum|a*w| companion.  Output-split: the sparse and the dense rows' outputs concatenated; input-split:
    the sparse K range plus the dense K range in one sum.  Either way it is the dense GEMM
    of the reconstructed weight, exact in float64 (module docstring)."""
    M = xq.shape[0]
    s_x = np.broadcast_to(np.asarray(s_x, dtype=np.float64).reshape(-1, 1), (M, 1))
    acc, ab = gemm_exact(xq, w_bytes)
    sc = s_x * float(s_w)
    return dict(y=acc * sc, absY=ab * sc)


def requant_scale_from_h(h: np.ndarray) -> np.ndarray:
    """Harness helper (Q10): per-token s_h[m] = max_j |h[m, j]| / 448 in fp32 (1 if zero)."""
    amax = np.max(np.abs(h), axis=1).astype(np.float32)
    return np.where(amax > 0, (amax / np.float32(E4M3_MAX)).astype(np.float32), np.float32(1)).astype(np.float32)


def mlp_dynamic(xq, s_x, wg_bytes, wu_bytes, wd_bytes, w_scale):
    """The layer with DYNAMIC per-token re-quantisation (Q10: the paper is
    silent on how h is re-quantised, its vLLM FP8 runs quantise activations dynamically):
    s_h[m] = max_j |h[m, j]| / 448 from the layer's own h, then the static path with that scale."""
    r = gate_up(xq, s_x, wg_bytes, wu_bytes, w_scale[0], w_scale[1], 1.0)
    s_h = requant_scale_from_h(r["h"])
    r = gate_up(xq, s_x, wg_bytes, wu_bytes, w_scale[0], w_scale[1], s_h)
    r.update(down(r["hq"], s_h, wd_bytes, w_scale[2]))
    r["s_h"] = s_h
    return r


# ---------------------------------------------------------------------------------------------
# Dense-index selection: SpenseGPT (Eq. 5) is `spensegpt_dense_idx` above;
# SpenseGPT+ (Eqs. 8-12) follows.  Readings: for W_down the index i is
# a COLUMN, so Eq. 9 aggregates column i over the H rows and H_down is the Hessian of down's input h
# (diag over the intermediate dimension); epsilon of Eq. 10 is an argument (the paper gives no value);
# "approximately pN ... under the required alignment constraint" = exactly I_dense indices (a multiple
# of 128); ties go to the lower index.
# ---------------------------------------------------------------------------------------------
def spensegpt_plus_scores(wgate, wup, wdown, hdiag_x, hdiag_h, eps=1e-8):
    """s_i of Eq. 11 in float64.  wgate, wup [I, H]; wdown [H, I]; hdiag_x [H] = diag(X^T X) of the MLP
    input (gate and up share it); hdiag_h [I] = diag of down's input Hessian."""
    wg, wu, wd = (np.asarray(a, dtype=np.float64) for a in (wgate, wup, wdown))
    rx = np.sqrt(np.asarray(hdiag_x, dtype=np.float64))
    rh = np.sqrt(np.asarray(hdiag_h, dtype=np.float64))
    I, H = wg.shape
    s_gate = (np.abs(wg) * rx[None, :]).sum(axis=1) / H          # Eq. 9, rows of W_gate
    s_up = (np.abs(wu) * rx[None, :]).sum(axis=1) / H            # Eq. 9, rows of W_up
    s_down = (np.abs(wd) * rh[None, :]).sum(axis=0) / H          # Eq. 9, columns of W_down (K = its H rows)
    norm = lambda v: v / (v.mean() + eps)                        # Eq. 10
    return norm(s_gate) + norm(s_up) + norm(s_down)              # Eq. 11


def topk_dense_idx(score, I_dense: int) -> np.ndarray:
    """Eq. 12: the I_dense indices of largest score, ties to the lower index; returned ascending."""
    score = np.asarray(score)
    order = np.lexsort((np.arange(score.size), -score))          # by score descending, then index ascending
    return np.sort(order[:I_dense]).astype(np.int32)


def spensegpt_plus_dense_idx(wgate, wup, wdown, hdiag_x, hdiag_h, I_dense: int, eps=1e-8) -> np.ndarray:
    return topk_dense_idx(spensegpt_plus_scores(wgate, wup, wdown, hdiag_x, hdiag_h, eps), I_dense)


# tolerance companions (O6): north_star bound |gpu - oracle| <= 2e-3 * sum|a*w| + 1e-5
def tol_gemm(abs_sum):
    return 2e-3 * np.asarray(abs_sum) + 1e-5


def tol_glu(r):
    """tau_h = 1.1*|u|*tau_g + |silu(g)|*tau_u + 1e-5 with tau_g = 2e-3*absG, tau_u = 2e-3*absU
    (|SiLU'| <= 1.0999): first-order propagation of the GEMM tolerance through h = silu(g)*u,
    plus the second-order cross term."""
    tg = 2e-3 * r["absG"]
    tu = 2e-3 * r["absU"]
    return 1.1 * np.abs(r["u"]) * tg + np.abs(silu(r["g"])) * tu + 1.1 * tg * tu + 1e-5
