"""Profiling case for profiles/: one hsp_create at C3 (the Gram on the tensor cores). Not a test."""
import os
import sys
import time

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))   # repo root
import torch  # noqa: E402
import hsp_synth  # noqa: E402
import paper_1608_04329_b200 as hsp  # noqa: E402

if __name__ == "__main__":
    wl = hsp_synth.make(sys.argv[1] if len(sys.argv) > 1 else "C3", "cuda")
    for _ in range(2):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        g = hsp.HorseshoeProbit(wl.X, wl.y, 1)
        g.sync()
        print("hsp_create ms", 1e3 * (time.perf_counter() - t0))
        g.close()
