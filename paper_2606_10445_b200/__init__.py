"""B200-native Spense hybrid sparse-dense FP8 GLU-MLP path (arxiv/paper_2606_10445).

``paper_2606_10445_b200.spense`` is the thin ctypes binding over ``libspense.so`` (C ABI declared in
``include/spense.h``, hand-written sm_100a CUDA under ``csrc/``).  Importing this package does not
load the library; the first call does, and it fails loudly if the library is missing.
"""
from . import spense  # noqa: F401
from .spense import (PackedLayer, SpenseError, spense_down, spense_gate_up, spense_mlp, spense_mlp_host,  # noqa: F401
                     spense_pack, spense_pack_sizes, spense_perm_from_dense_idx, spense_quantize_e4m3,
                     spense_version, spense_workspace, spense_workspace_size)
