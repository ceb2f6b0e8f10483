"""Codebook / scale distortion study on the GPU (the shape of Fig. 2b):
relative MSE of 4-bit quantisers of the coordinates of random unit vectors (what a rotated key looks like), d = 64,
128, 256, all through uq_calibrate_c.  `python -m paper_2606_20474_b200.distortion` prints a markdown table.

Schemes (32-element groups, m = group absmax unless stated):
  lloyd-max   16-level Lloyd-Max codebook of N(0,1) at the fixed scale 1/sqrt(d) (per-vector norm known: the
              analytical reference of Fig. 2a; no per-group scale is stored)
  fp4 c=1.0   E2M1, s = m ("raw absmax with no shrinkage")
  fp4 mx      E2M1, s = 2^(floor(log2 m) - 2): the OCP MX rule = the power-of-two scale at c = 2^-2.5
  fp4 0.156   E2M1, s = 0.156 m (Eq.(2) at the paper's constant, continuous scale)
  fp4 0.156p  E2M1, s = 2^round(log2(0.156 m)): what Alg. 1 stores
  fp4 0.195p  the same at the paper's "power-of-two-optimal" constant (:333)
  int4        uniform symmetric 15-level grid, s = m / 7
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as uq

# Lloyd-Max centroids of a 16-level quantiser of N(0,1) (fixed point of Lloyd's iteration on the Gaussian integrals)
LLOYD_MAX_16 = (0.1284, 0.3881, 0.6568, 0.9424, 1.2562, 1.6181, 2.0690, 2.7326)


def study(n_vectors: int = 1 << 15, seed: int = 0, device="cuda"):
    cfg = uq.UQConfig(num_q_heads=8, num_kv_heads=1)
    g = torch.Generator(device="cpu"); g.manual_seed(seed)
    lm = torch.tensor(LLOYD_MAX_16, dtype=torch.float32, device=device)
    i4 = torch.arange(8, dtype=torch.float32, device=device)
    rows = {}
    for d in (64, 128, 256):
        u = torch.randn((n_vectors * 128 // d, d), generator=g)
        u = (u / u.norm(dim=1, keepdim=True)).to(torch.bfloat16).reshape(-1, 128).contiguous().to(device)

        def rel(c, mode, levels=None):
            sq, nrm = uq.calibrate_c(cfg, u, torch.tensor([c], dtype=torch.float32, device=device), rotate=False,
                                     scale_mode=mode, levels=levels)
            return float(sq[0].item() / nrm[0].item())

        rows[d] = {"lloyd-max": rel(d ** -0.5, 2, lm), "fp4 c=1.0": rel(1.0, 0), "fp4 mx": rel(2.0 ** -2.5, 1),
                   "fp4 0.156": rel(0.156, 0), "fp4 0.156p": rel(0.156, 1), "fp4 0.195p": rel(0.195, 1),
                   "int4": rel(1.0 / 7.0, 0, i4)}
    return rows


def main():
    rows = study()
    names = list(next(iter(rows.values())).keys())
    print("| d | " + " | ".join(names) + " |")
    print("|---|" + "---|" * len(names))
    for d, r in rows.items():
        print(f"| {d} | " + " | ".join(f"{r[n]:.5f}" for n in names) + " |")


if __name__ == "__main__":
    main()
