"""Child process of test_gpu_gemm.py::test_first_call_in_a_fresh_process_is_capturable: a process that never packs.
It loads a packed blob from bytes, initialises a workspace (the library's one-time set-up happens there) and captures
its FIRST spense_mlp in a CUDA graph under torch's default (global) capture mode, replays it and saves hq and y.
usage: python -m tests.capture_child <dir>   (dir holds blob.pt, x.pt, sx.pt, sh.pt, meta.pt; writes out.pt)"""
import sys

import torch

from paper_2606_10445_b200 import spense as sp


def main(d):
    H, I, I_d, M = torch.load(f"{d}/meta.pt").tolist()
    blob = torch.load(f"{d}/blob.pt").cuda()
    x, sx, sh = (torch.load(f"{d}/{n}.pt").cuda() for n in ("x", "sx", "sh"))
    pk = sp.PackedLayer(H, I, I_d, blob)
    ws = sp.spense_workspace(pk, M)                       # spense_workspace_init: outside capture
    hq = torch.zeros(M, I, dtype=torch.uint8, device="cuda")
    y = torch.zeros(M, H, dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):               # capture_error_mode = "global"
            sp.spense_mlp(pk, x, sx, sh, ws, hq_scratch=hq, y=y)     # the first GEMM call of this process
    torch.cuda.current_stream().wait_stream(s)
    g.replay()
    torch.cuda.synchronize()
    assert sp.spense_device_status() == "SPENSE_OK"
    torch.save({"hq": hq.cpu(), "y": y.cpu()}, f"{d}/out.pt")


if __name__ == "__main__":
    main(sys.argv[1])
