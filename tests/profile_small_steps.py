"""One casgd_outer_steps call of 512 iterations on a small shape, for ncu captures of the one-launch kernels
(profiles/r2j_ncu_small.md):   python tests/profile_small_steps.py WORKLOAD S     (0 = tiny-logistic, 1 = SUSY-shaped, ...)"""
import sys

import numpy as np
import torch

sys.path.insert(0, ".")
from paper_2606_18463_b200 import binding, synth  # noqa: E402

w, s = int(sys.argv[1]), int(sys.argv[2])
cfg = synth.config(w, m=200000)
ds = synth.make_dataset(cfg, seed=42, device="cuda")
steps = 512
idx = torch.from_numpy(np.random.default_rng(0).integers(0, cfg.m, steps * s * cfg.b, dtype=np.int32)).cuda()
with binding.Casgd(ds.X_bf16, ds.y, cfg.loss) as cg:
    x = torch.zeros(cfg.n, device="cuda")
    cg.outer_steps(idx, x, s, cfg.b, cfg.eta * 0.1)
    cg.sync()
print("ok")
