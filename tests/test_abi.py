"""CPU-side checks of the C-ABI boundary: libspense.so builds, loads and exports every symbol that
include/spense.h declares; host-only entry points behave; argument errors are caught on the host."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import spense_oracle as o

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sp():
    from paper_2606_10445_b200 import build, spense
    build.build()
    return spense


def test_every_declared_symbol_is_exported(sp):
    hdr = open(os.path.join(ROOT, "include", "spense.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(spense_[a-z0-9_]+)\s*\(", hdr))
    assert names == set(sp.EXPORTS), names ^ set(sp.EXPORTS)
    L = ctypes.CDLL(sp.LIB_PATH)
    for n in names:
        assert hasattr(L, n), n
    # and nothing else: the default build exports exactly what the header declares (no debug hooks)
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", sp.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if ln.split()[-2] in ("T", "t") and ln.split()[-1].startswith("spense_")}
    assert exported == names, exported ^ names
    assert sp.spense_version() >= 1
    assert sp.lib().spense_strerror(-5).decode().startswith("a group of 4")


def test_perm_from_dense_idx_matches_oracle(sp):
    rng = np.random.default_rng(0)
    for I, nd in ((10, 3), (1024, 256), (128, 0), (128, 128)):
        d = rng.choice(I, nd, replace=False)
        got = sp.spense_perm_from_dense_idx(I, d.tolist()).numpy()
        assert np.array_equal(got, o.perm_from_dense_idx(I, d))
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_perm_from_dense_idx(8, [1, 1])
    assert e.value.code == "SPENSE_ERR_ARG"


def test_size_queries_and_host_side_argument_errors(sp):
    blob, ws = sp.spense_pack_sizes(5120, 25600, 6400)
    assert blob == 1024 + 282_624_000          # Qwen3-32B-shaped, p = 25 %
    blob, _ = sp.spense_pack_sizes(5120, 27648, 0)
    assert blob == 1024 + 265_420_800
    blob, _ = sp.spense_pack_sizes(256, 1024, 256)
    assert blob == 1024 + 565_248
    for bad in ((100, 1024, 0), (256, 1000, 0), (256, 1024, 100), (256, 1024, 2048)):
        with pytest.raises(sp.SpenseError) as e:
            sp.spense_pack_sizes(*bad)
        assert e.value.code == "SPENSE_ERR_SHAPE"
    assert sp.spense_workspace_size(256, 1024, 256, 8) > 4096
    with pytest.raises(sp.SpenseError) as e:
        sp.spense_workspace_size(256, 1024, 256, 0)
    assert e.value.code == "SPENSE_ERR_ARG"
    # null pointers are rejected before anything touches CUDA (works on a box without a GPU)
    L = sp.lib()
    shp = sp.Shape(256, 1024, 256)
    st = L.spense_gate_up(ctypes.byref(shp), None, None, None, 8, None, 0, None, None, None, 0, None)
    assert sp.STATUS[st] == "SPENSE_ERR_ARG"
    st = L.spense_down(ctypes.byref(shp), ctypes.c_void_p(1024), ctypes.c_void_p(3), ctypes.c_void_p(4), 0, 8,
                       ctypes.c_void_p(16), 0, ctypes.c_void_p(128), 1 << 30, None, None)
    assert sp.STATUS[st] == "SPENSE_ERR_ALIGN"


def test_linear_size_queries_and_argument_errors(sp):
    L = sp.lib()
    b, w = ctypes.c_size_t(), ctypes.c_size_t()
    # in-split W [5120, 25600] with 6400 dense columns = the down section of the Qwen3-32B-shaped layer
    shp = sp.LinearShape(5120, 25600, 6400, sp.SPENSE_SPLIT_IN)
    assert L.spense_linear_pack_sizes(ctypes.byref(shp), ctypes.byref(b), ctypes.byref(w)) == 0
    assert b.value == 1024 + 94_208_000 and w.value == 128 + 4 * 25600
    # out-split W [25600, 5120] with 6400 dense rows: 19200 x 5120 x 0.625 + 6400 x 5120 bytes
    shp = sp.LinearShape(25600, 5120, 6400, sp.SPENSE_SPLIT_OUT)
    assert L.spense_linear_pack_sizes(ctypes.byref(shp), ctypes.byref(b), ctypes.byref(w)) == 0
    assert b.value == 1024 + 19200 * 5120 * 5 // 8 + 6400 * 5120 and w.value == 128 + 4 * 25600
    # a dense half tile at the end is padded to a whole 256-row tile
    shp = sp.LinearShape(640, 256, 128, sp.SPENSE_SPLIT_OUT)
    assert L.spense_linear_pack_sizes(ctypes.byref(shp), ctypes.byref(b), None) == 0
    assert b.value == 1024 + 2 * 40960 + 2 * 32768
    for bad in ((640, 256, 256, 0), (100, 256, 0, 0), (256, 256, 64, 1), (256, 256, 512, 1)):
        assert sp.STATUS[L.spense_linear_pack_sizes(ctypes.byref(sp.LinearShape(*bad)), ctypes.byref(b), None)] == "SPENSE_ERR_SHAPE"
    assert sp.STATUS[L.spense_linear_pack_sizes(ctypes.byref(sp.LinearShape(256, 256, 0, 7)), ctypes.byref(b), None)] == "SPENSE_ERR_ARG"
    shp = sp.LinearShape(256, 256, 0, sp.SPENSE_SPLIT_OUT)
    st = L.spense_linear_out_split(ctypes.byref(shp), None, None, None, 0, 8, None, 0, None, 0, None)
    assert sp.STATUS[st] == "SPENSE_ERR_ARG"
    st = L.spense_linear_in_split(ctypes.byref(shp), ctypes.c_void_p(128), ctypes.c_void_p(128), ctypes.c_void_p(4), 0, 8,
                                  ctypes.c_void_p(16), 0, ctypes.c_void_p(128), 1 << 30, None)
    assert sp.STATUS[st] == "SPENSE_ERR_ARG"                      # an out-split shape handed to the in-split call


def test_prune_obs_size_query_and_argument_errors(sp):
    L = sp.lib()
    b = ctypes.c_size_t()
    assert L.spense_prune_obs_workspace_size(5120, 25600, ctypes.byref(b)) == 0 and b.value == 5120 * 128 * 4
    assert sp.STATUS[L.spense_prune_obs_workspace_size(0, 128, ctypes.byref(b))] == "SPENSE_ERR_ARG"
    assert sp.STATUS[L.spense_prune_obs_workspace_size(8, 130, ctypes.byref(b))] == "SPENSE_ERR_ARG"      # K % 4 != 0
    # the trailing update indexes 64-row tiles on gridDim.y: 65535 tiles is the last row count that fits
    assert L.spense_prune_obs_workspace_size(65535 * 64, 128, ctypes.byref(b)) == 0
    assert sp.STATUS[L.spense_prune_obs_workspace_size(65535 * 64 + 1, 128, ctypes.byref(b))] == "SPENSE_ERR_ARG"
    one = ctypes.c_void_p(1 << 20)
    for ks in (-4, 6, 132):                                       # negative, not a multiple of 4, beyond K
        assert sp.STATUS[L.spense_prune_obs_2to4(8, 128, ks, one, one, one, 1 << 30, None)] == "SPENSE_ERR_ARG"
    assert sp.STATUS[L.spense_prune_obs_2to4(8, 128, 64, None, one, one, 1 << 30, None)] == "SPENSE_ERR_ARG"
    assert sp.STATUS[L.spense_prune_obs_2to4(8, 128, 64, ctypes.c_void_p(4), one, one, 1 << 30, None)] == "SPENSE_ERR_ALIGN"
    assert sp.STATUS[L.spense_prune_obs_2to4(8, 128, 64, one, one, one, 16, None)] == "SPENSE_ERR_BUFFER_TOO_SMALL"


def test_build_never_replaces_the_production_library_with_a_debug_build(sp, tmp_path):
    from paper_2606_10445_b200 import build
    with pytest.raises(ValueError):
        build.build(debug_hooks=True)                              # no out: would overwrite libspense.so
    with pytest.raises(ValueError):
        build.build(debug_hooks=True, out=build.LIB)
    # out= is honoured without debug hooks too (used to return libspense.so untouched when the tree was not stale)
    out = str(tmp_path / "libspense_copy.so")
    assert build.build(out=out) == out and os.path.getsize(out) > 0
