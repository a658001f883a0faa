"""Not collected by pytest (minutes of CPU): every pixel of the BASELINE configs against the long-double oracle, all
three modes, through the C ABI.  The -m gpu tests check sampled pixels at full size; this is the exhaustive version.

    python tests/fullgrid_parity.py 1 4 2 3         (config 3: ~7 minutes of oracle time on 16 cores)
    python tests/fullgrid_parity.py sie nfw         (the paper-like SIE benchmark, 6730^2 x 702; the NFW cluster, 2048^2 x 64)
"""
import os
import sys
import time

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from oracle import lt_oracle, lt_oracle_nfw, lt_oracle_sie       # noqa: E402
from paper_1902_03252_b200 import lt, workloads                   # noqa: E402

for cfg in sys.argv[1:] or ["1"]:
    if cfg == "sie":
        W, O, grid, mixed = workloads.make_sie("paper"), lt_oracle_sie, lt.lt_gradient_grid_sie, (3.26, 0.0104 / 0.03, 6.0, 0.3, 1.0)
    elif cfg == "nfw":
        W, O, grid, mixed = workloads.make_nfw(n_override=2048), lt_oracle_nfw, lt.lt_gradient_grid_nfw, None
    else:
        W, O, grid, mixed = workloads.make(int(cfg)), lt_oracle, lt.lt_gradient_grid, None
    t0 = time.time()
    ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    t_or = time.time() - t0
    s = np.abs(ref).reshape(-1, 2).max(axis=0)
    L = torch.from_numpy(W.lenses).cuda()
    res = {}
    for mode, name in ((lt.LT_FP64, "fp64"), (lt.LT_FP32, "fp32"), (lt.LT_MIXED, "mixed")):
        out = grid(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, mixed=mixed).cpu().numpy().astype(np.float64)
        e = np.abs(out - ref).reshape(-1, 2)
        res[name] = ((e.max(axis=0) / s).max(), (np.sqrt((e ** 2).mean(axis=0)) / s).max())
    print("%s full grid %dx%d x %d lenses: oracle %.0f s on %d threads | " % (W.name, W.nx, W.ny, len(W.lenses), t_or,
                                                                              lt_oracle.max_threads())
          + " | ".join("%s max %.3e rms %.3e" % (k, v[0], v[1]) for k, v in res.items()), flush=True)
    assert res["fp64"][0] < 1e-12 and res["fp32"][0] < 1e-5 and res["mixed"][0] < 1e-5
