"""A/B: SDF queries from a TMA-staged per-patch brick in shared memory vs the product's quad-layout gather.

    python -m paper_2606_22332_b200.experiments.brick_ab            (builds libbrick_ab.so if needed; needs a B200)

Shapes of BASELINE configs 3 and 5: star grids (64^3 @ 2 mm / 96^3 @ 4/3 mm), pads of 5 x 5 / 8 x 8 taxels (20 x 20 mm),
poses from the near-surface recipe (pad 0-20 mm outside the surface, normal towards the object, 10 deg tilt), first query
plus a 16-evaluation march of 20 mm.  Prints one JSON line per case: time of both kernels, agreement, fallback share.
"""
import ctypes as C
import json
import os
import subprocess
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(HERE, "libbrick_ab.so")
SRC = os.path.join(HERE, "brick_ab.cu")


def build(no_tma=False):
    """libbrick_ab.so (TMA tensor copy) or libbrick_ab_notma.so (the same brick filled by plain loads)."""
    so = SO.replace(".so", "_notma.so") if no_tma else SO
    if os.path.exists(so) and os.path.getmtime(so) >= os.path.getmtime(SRC):
        return so
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
                    "-shared", "-cudart", "shared"] + (["-DBRICK_NO_TMA"] if no_tma else []) + [SRC, "-o", so], check=True)
    return so


def case(cid, n_patches, brick, reps=20, no_tma=False):
    sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
    from paper_2606_22332_b200 import workloads as W
    w = W.config(cid, n_envs=64)
    N, G = w.bank.shape[1], w.bank.shape[0]
    nu, nv, pitch = (5, 5, 0.004) if cid == 3 else (8, 8, 0.0025)
    rng = np.random.default_rng(cid)
    u = rng.normal(size=(n_patches, 3)); u /= np.linalg.norm(u, axis=1, keepdims=True)
    grid = rng.integers(0, G, n_patches)
    rad = np.array([W.star_radius(u[i], w.stars[grid[i]]["scale"], w.stars[grid[i]]["rot"]) for i in range(n_patches)])
    c = u * (rad + rng.uniform(0.0, 0.02, n_patches))[:, None]                  # pad centre 0-20 mm outside the surface
    n = -u + rng.normal(0, np.tan(np.deg2rad(10.0)), (n_patches, 3)); n /= np.linalg.norm(n, axis=1, keepdims=True)
    t = np.cross(n, rng.normal(size=(n_patches, 3))); t /= np.linalg.norm(t, axis=1, keepdims=True)
    b = np.cross(n, t)
    P = np.concatenate([c, t, b, n, grid[:, None].astype(np.float64)], axis=1).astype(np.float32)
    L = C.CDLL(build(no_tma))
    L.brick_ab_run.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_float, C.c_float,
                               C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    og = np.zeros(n_patches * nu * nv, np.float32); ob = np.zeros_like(og); ms = np.zeros(2, np.float32); fb = np.zeros(1, np.uint32)
    bank = np.ascontiguousarray(w.bank, np.float32)
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    rc = L.brick_ab_run(p(bank), G, N, C.c_float(w.voxel), p(P), n_patches, nu, nv, C.c_float(pitch), C.c_float(0.02), 16, brick, reps,
                        p(og), p(ob), p(ms), p(fb))
    assert rc == 0, rc
    evals = n_patches * nu * nv * 16
    return dict(config=cid, staging="plain loads" if no_tma else "TMA bulk copies (cp.async.bulk, one per brick row)", grid="%d^3 x %d" % (N, G), voxel_mm=round(w.voxel * 1e3, 3), patches=n_patches, taxels_per_patch=nu * nv,
                brick="%d^3 voxels = %.1f KB shared memory per patch" % (brick, brick ** 3 * 4 / 1024.0),
                gather_ms=float(ms[0]), brick_ms=float(ms[1]), brick_over_gather=float(ms[1] / ms[0]),
                max_abs_diff_m=float(np.abs(og - ob).max()), fallback_share=float(fb[0]) / (evals * reps))


if __name__ == "__main__":
    for no_tma in (False, True):
        for cid, brick in ((5, 24), (5, 32), (3, 16), (3, 24)):
            try:
                print(json.dumps(case(cid, 40960 if cid == 3 else 20480, brick, no_tma=no_tma)), flush=True)
            except AssertionError as ex:
                print(json.dumps(dict(config=cid, brick=brick, no_tma=no_tma, failed="brick_ab_run returned %s" % ex)), flush=True)
                sys.exit(0)     # a CUDA fault is sticky: nothing after it in this process would run
