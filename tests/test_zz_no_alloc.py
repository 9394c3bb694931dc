"""ts_depth_static (include/ts.h): the allocation-free entry point -- contact depth against one primitive per env with the
relative poses in the library's static device array instead of ctx-owned cudaMalloc'd scratch.

Collected last on purpose (the suite runs with pytest -x): it must pass alone in a fresh process and after every other
test has created and destroyed contexts in this process.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2606_22332_b200 import workloads as W

ATOL, RTOL = 1e-6, 1e-4        # the tolerance of tests/parity.py


def test_sizes_beyond_the_static_scratch_are_rejected_before_any_cuda_call():
    """No GPU needed: the size check comes first and names the limit."""
    from paper_2606_22332_b200 import binding as B
    assert B.STATIC_MAX_FRAMES == (8 << 20) // 96
    L = B.lib()
    null = C.c_void_p(0)
    args = [null] * 11
    rc = L.ts_depth_static(B.STATIC_MAX_FRAMES // 16 + 1, 16, 100, *args)
    assert rc == B.TS_ERR_INVALID_ARG
    msg = L.ts_last_error(None).decode()
    assert "TS_STATIC_MAX_FRAMES" in msg and str(B.STATIC_MAX_FRAMES) in msg, msg
    assert L.ts_depth_static(0, 16, 100, *args) == B.TS_ERR_INVALID_ARG
    # inside the limit but without buffers: still refused on the host
    assert L.ts_depth_static(4, 16, 100, *args) == B.TS_ERR_INVALID_ARG
    assert "null pointer" in L.ts_last_error(None).decode()


@pytest.mark.gpu
def test_depth_static_equals_the_ctx_path_on_two_calls_in_a_row():
    """Config-2 scene (spheres, boxes, capsules; 16 links x 12 taxels + fillers): the depth of ts_depth_static against the
    depth output of ts_step on the same inputs, element by element within the parity tolerance,
    on two calls in a row that share the static scratch -- the second with other poses and fewer envs, so stale records of
    the first call would show -- and with no device memory taken by either call."""
    import torch
    from paper_2606_22332_b200 import binding as B
    w = W.config(2, n_envs=1500)
    assert w.E * w.L <= B.STATIC_MAX_FRAMES and w.K == 1
    sim = B.TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=w.physics, noise=None, outputs=("depth",))
    sim.set_geometry(w.types, w.params, w.bank, w.voxel)
    lay = sim.layout.view()
    dev = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dt)).cuda()
    tpos, trad, tlink = dev(lay["pos"], np.float32), dev(lay["radius"], np.float32), dev(lay["link"], np.int32)
    gtype, gprm = dev(w.types.reshape(-1), np.int32), dev(w.params.reshape(-1, 4), np.float32)
    out = torch.full((w.E, w.T), -1.0, dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    touched = 0
    for call, (step, n_env) in enumerate(((0, w.E), (7, 700))):
        x = sim.upload(w.inputs(step))
        want = sim.step(x)["depth"][:n_env].clone()
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        out.fill_(-1.0)
        torch.cuda.synchronize()
        B.depth_static(n_env, w.L, w.T, tpos, trad, tlink, x["link_pos"], x["link_quat"], x["obj_pos"], x["obj_quat"], gtype, gprm,
                       out, stream)
        torch.cuda.synchronize()
        if call == 1:                        # first call may page the kernels in (lazy module loading); the second takes nothing
            assert torch.cuda.mem_get_info()[0] == free0
        got = out[:n_env].double().cpu().numpy()
        ref = want.double().cpu().numpy()
        assert np.all(np.abs(got - ref) <= ATOL + RTOL * np.abs(ref)), float(np.abs(got - ref).max())
        assert (out[n_env:] == -1.0).all()   # rows past n_envs are not written
        touched += int((ref > 0).sum())
    assert touched > 10000                   # the comparison is not vacuous
    sim.close()
