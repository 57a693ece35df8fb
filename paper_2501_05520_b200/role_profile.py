"""Per-role wait cycles of the fused S4 kernel (profiles/r1_fused_roles_v3.md).  Needs a profiling build of the library:

    TRK_NVCC_EXTRA=-DTRK_FUSED_PROF python -m paper_2501_05520_b200.build --force
    python -m paper_2501_05520_b200.role_profile
    python -m paper_2501_05520_b200.build --force          # back to the product build

Runs one pileup-200 trk_infer and prints, for the first two CTAs of the last edge-update launch, the fraction of the CTA's
lifetime each warp role spent in its instrumented waits (slots 0-3, see the FPW() uses in csrc/gnn_fused*.cuh).
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np


def main():
    import torch
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    if root not in sys.path:
        sys.path.insert(0, root)
    from paper_2501_05520_b200 import lib, trk_from_config
    from synth.configs import get_config, load_calibration, make_events
    from synth.weights import make_model
    L = lib()
    if not hasattr(L, "trk_debug_fused_prof"):
        raise SystemExit("libtrk.so is not a profiling build (TRK_NVCC_EXTRA=-DTRK_FUSED_PROF)")
    cfg = get_config("pileup200")
    calib = load_calibration("pileup200")
    ev, model = make_events(cfg), make_model(cfg)
    n = len(ev["hits"])
    trk = trk_from_config(cfg, model, calib, max_hits=n, max_cand_edges=n * cfg["frnn_k"], max_kept_edges=int(calib["n_kept_edges"] * 1.5))
    hits = torch.from_numpy(ev["hits"]).cuda()
    out = trk.infer(hits, ev["event_offsets"])
    torch.cuda.synchronize()
    trk.infer(hits, ev["event_offsets"], out=out)
    torch.cuda.synchronize()
    buf = (C.c_ulonglong * (4 * 24 * 8))()
    if L.trk_debug_fused_prof(buf) != 0:
        raise SystemExit("reading the profile counters failed")
    a = np.array(list(buf), dtype=np.int64).reshape(4, 24, 8)
    for blk in range(2):
        print("CTA", blk)
        for w in range(24):
            tot = a[blk, w, 7]
            if tot > 0:
                print(f"  warp {w:2d}  lifetime {tot:9d} cycles  wait fractions " + " ".join(f"{a[blk, w, i] / tot:6.3f}" for i in range(4)))
    trk.close()


if __name__ == "__main__":
    main()
