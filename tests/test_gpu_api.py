"""-m gpu: behaviour of the C ABI itself (include/ts.h): host-buffer step, timing introspection, error paths."""
import ctypes as C
import os

import numpy as np
import pytest

from paper_2606_22332_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _sim(w, **kw):
    from paper_2606_22332_b200.binding import TactileSim
    sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=w.physics, noise=kw.get("noise", w.noise), outputs=kw.get("outputs", w.outputs))
    if kw.get("geometry", True):
        sim.set_geometry(w.types, w.params, w.bank, w.voxel)
    return sim


def test_step_host_equals_step_on_device_tensors():
    """ts_step_host = H2D + the same kernels + D2H on the caller's stream: bit-identical outputs, state advances alike."""
    import torch
    w = W.config(5, n_envs=24)
    a, b = _sim(w), _sim(w)
    host_out = b.alloc_outputs(pinned_host=True)
    for s in range(4):
        inp = w.inputs(s)
        dev = a.step(a.upload(inp))
        host_in = {k: torch.from_numpy(np.ascontiguousarray(v)).pin_memory() for k, v in inp.items()}
        b.step_host(host_in, host_out)
        torch.cuda.synchronize()
        for k, v in dev.items():
            assert torch.equal(v.cpu(), host_out[k]), (k, s)


def test_kernel_time_introspection():
    import torch
    w = W.config(4, n_envs=64)
    sim = _sim(w)
    inp = sim.upload(w.inputs(0))
    out = sim.alloc_outputs()
    assert sim.kernel_time_ms(True) == (0.0, 0)
    for _ in range(5):
        sim.step(inp, out)
    torch.cuda.synchronize()
    ms, n = sim.kernel_time_ms(False)
    assert n == 5 and 0.0 < ms < 50.0
    assert 0.0 < sim.first_kernel_time_ms() <= ms * 1.001
    # TS_SPLIT=1 selects the two-kernel variant (readout, then the stand-alone noise kernel)
    assert sim.launches_per_step() == (3 if os.environ.get("TS_SPLIT") == "1" else 2)
    sim.step(inp, out)                         # recording is off again
    assert sim.kernel_time_ms(False) == (0.0, 0)


def test_error_paths_return_status_and_message():
    import torch
    from paper_2606_22332_b200 import binding as B
    w = W.config(2, n_envs=8)
    sim = _sim(w, geometry=False)
    inp = sim.upload(w.inputs(0))
    out = sim.alloc_outputs()
    with pytest.raises(B.TsError, match="TS_ERR_STATE"):
        sim.step(inp, out)                                                  # before ts_set_geometry
    sim.set_geometry(w.types, w.params, w.bank, w.voxel)
    sim.step(inp, out)
    L = B.lib()
    si, so = sim._structs(inp, out, host=False)
    # NULL input pointer
    si.link_quat = None
    assert L.ts_step(sim.h, C.byref(si), C.byref(so), sim._stream()) == 1
    assert b"NULL input" in L.ts_last_error(sim.h)
    si, so = sim._structs(inp, out, host=False)
    # misaligned output pointer
    so.depth = out["depth"].data_ptr() + 4
    assert L.ts_step(sim.h, C.byref(si), C.byref(so), sim._stream()) == 1
    assert b"aligned" in L.ts_last_error(sim.h)
    # ft_noisy requested from a context without noise
    si, so = sim._structs(inp, out, host=False)
    so.ft_noisy = out["ft"].data_ptr()
    assert L.ts_step(sim.h, C.byref(si), C.byref(so), sim._stream()) == 1
    # bad geometry: grid id out of range, unknown type
    types = w.types.copy(); types[0, 0] = 4
    with pytest.raises(B.TsError, match="TS_ERR_INVALID_ARG"):
        sim.set_geometry(types, w.params, None, 0.0)
    types[0, 0] = 9
    with pytest.raises(B.TsError, match="TS_ERR_INVALID_ARG"):
        sim.set_geometry(types, w.params, None, 0.0)
    # the context still works after rejected calls
    sim.set_geometry(w.types, w.params, w.bank, w.voxel)
    sim.step(inp, out)
    torch.cuda.synchronize()
    assert L.ts_destroy(None) == 0 and L.ts_step(None, None, None, None) == 1


def test_outputs_subset_and_replaced_geometry():
    """NULL outputs are skipped (others unchanged); ts_set_geometry may be called again with another bank."""
    import torch
    w = W.config(3, n_envs=16)
    full = _sim(w)
    part = _sim(w, outputs=("depth", "prox"))
    inp = full.upload(w.inputs(0))
    a, b = full.step(inp), part.step(inp)
    torch.cuda.synchronize()
    assert set(b) == {"depth", "prox"} and torch.equal(a["depth"], b["depth"]) and torch.equal(a["prox"], b["prox"])
    w5 = W.config(5, n_envs=16)
    full2 = _sim(w5)
    full2.set_geometry(w5.types, w5.params, w5.bank * np.float32(1.0), w5.voxel)     # same bank again: same results
    x = full2.upload(w5.inputs(0))
    r1 = {k: v.clone() for k, v in full2.step(x).items()}
    full2.reset()
    full2.set_geometry(w5.types, w5.params, w5.bank + np.float32(1e-3), w5.voxel)    # shifted field: 1 mm less depth
    r2 = full2.step(x)
    torch.cuda.synchronize()
    grid_env = torch.from_numpy(w5.types[:, 0] == 4).cuda()
    touched = (r1["depth"] > 1.2e-3) & grid_env[:, None]
    assert touched.any()
    assert torch.allclose(r2["depth"][touched], r1["depth"][touched] - 1e-3, atol=2e-6)
    assert torch.equal(r2["depth"][~grid_env], r1["depth"][~grid_env])               # primitives are untouched
