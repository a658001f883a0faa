"""Not collected by pytest (minutes of CPU): every pixel of the BASELINE configs against the long-double oracle, all
three modes, through the C ABI.  The -m gpu tests check sampled pixels at full size; this is the exhaustive version.

    python tests/fullgrid_parity.py 1 4 2 3         (config 3: ~7 minutes of oracle time on 16 cores)
"""
import os
import sys
import time

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from oracle import lt_oracle as O                      # noqa: E402
from paper_1902_03252_b200 import lt, workloads        # noqa: E402

for cfg in [int(a) for a in sys.argv[1:]] or [1]:
    W = workloads.make(cfg)
    t0 = time.time()
    ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    t_or = time.time() - t0
    s = np.abs(ref).reshape(-1, 2).max(axis=0)
    L = torch.from_numpy(W.lenses).cuda()
    res = {}
    for mode, name in ((lt.LT_FP64, "fp64"), (lt.LT_FP32, "fp32"), (lt.LT_MIXED, "mixed")):
        out = lt.lt_gradient_grid(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode).cpu().numpy().astype(np.float64)
        e = np.abs(out - ref).reshape(-1, 2)
        res[name] = ((e.max(axis=0) / s).max(), (np.sqrt((e ** 2).mean(axis=0)) / s).max())
    print("cfg%d full grid %dx%d x %d lenses: oracle %.0f s on %d threads | " % (cfg, W.nx, W.ny, len(W.lenses), t_or,
                                                                                 O.max_threads())
          + " | ".join("%s max %.3e rms %.3e" % (k, v[0], v[1]) for k, v in res.items()), flush=True)
    assert res["fp64"][0] < 1e-12 and res["fp32"][0] < 1e-5 and res["mixed"][0] < 1e-5
