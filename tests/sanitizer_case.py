"""Small driver for compute-sanitizer (SURVEY section 4 tier 5): a few steps of config 1 and of a 64-env config 5
with the read-delay ring, radius noise and Gaussian crosstalk on, in both kernel forms, over a reset.

    compute-sanitizer --tool memcheck|racecheck|initcheck python tests/sanitizer_case.py

Not collected by pytest (no test_ prefix); the summaries of the three runs are kept under profiles/.
"""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2606_22332_b200 import workloads as W            # noqa: E402
from paper_2606_22332_b200.binding import TactileSim        # noqa: E402


def run(w, steps, noise=None, form="auto"):
    sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=dict(w.physics, kernel_form=form), noise=noise, outputs=w.outputs)
    sim.set_geometry(w.types, w.params, w.bank, w.voxel)
    acc = 0.0
    for s in range(steps):
        if s == steps // 2:
            mask = torch.from_numpy((np.arange(w.E) % 2 == 0).astype(np.uint8)).cuda()
            sim.reset(mask)
        out = sim.step(sim.upload(w.inputs(s)))
        torch.cuda.synchronize()
        acc += float(sum(v.float().abs().sum().item() for v in out.values()))
    sim.close()
    return acc


def main():
    assert torch.cuda.is_available()
    w1 = W.config(1)
    print("config 1:", run(w1, 3))
    w5 = W.config(5, n_envs=64)
    print("config 5 (64 envs, headline knobs, fused):", run(w5, 4, noise=w5.noise))
    ext = dict(w5.noise, read_delay=2, read_jitter=1, radius_noise=3e-4, xtalk_sigma=0.8, chi=0.3, bias_force=0.01,
               sigma_white_force=2e-3, gain_min=0.9, gain_max=1.1, quant_force=1e-3)
    print("config 5 (64 envs, all knobs, split):", run(w5, 6, noise=ext, form="split"))
    print("config 5 (64 envs, all knobs, fused):", run(w5, 6, noise=ext, form="fused"))
    w2 = W.config(2, n_envs=64)
    print("config 2 (64 envs, no noise):", run(w2, 2))


if __name__ == "__main__":
    main()
