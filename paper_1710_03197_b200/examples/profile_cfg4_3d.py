"""One forward + adjoint of BASELINE config 4 (3-D 128^3, kooshball, M = 2,097,152) after warm-up: the command profiles/
r01i_cfg4_3d.md was captured with.  Usage: python paper_1710_03197_b200/examples/profile_cfg4_3d.py"""
import os
import sys

import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import paper_1710_03197_b200 as nb  # noqa: E402
import workloads as wl  # noqa: E402

cfg = wl.config(3)
p = nb.NufftPlan(cfg["Nd"], cfg["Kd"], cfg["Jd"], cfg["om"], max_batch=1)
x = torch.from_numpy(wl.image_gaussian(cfg["Nd"])).cuda().reshape(1, *cfg["Nd"])
y = p.forward(x)
xo = p.adjoint(y)
for _ in range(2):
    p.forward(x, y)
    p.adjoint(y, xo)
torch.cuda.synchronize()
print("cfg4 forward+adjoint done; launches", p.launch_count())
p.destroy()
