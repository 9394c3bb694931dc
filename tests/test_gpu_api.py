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
    # maximum sizes: the state rows use 32-bit element indices, n_envs * 12 * T (rounded up to 32) must stay below 2^32
    w5 = W.config(5, n_envs=8)
    with pytest.raises(B.TsError, match="32-bit element indices"):
        B.TactileSim(w5.patches, w5.T, 350000, w5.L, w5.K, physics=w5.physics, noise=w5.noise, outputs=w5.outputs)
    with pytest.raises(B.TsError, match="32-bit element indices"):          # the read-delay ring has its own bound
        B.TactileSim(w5.patches, w5.T, 200000, w5.L, w5.K, physics=w5.physics, noise=dict(w5.noise, read_delay=8), outputs=w5.outputs)


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


def test_output_mask_contract_and_config_ranges():
    """ts.h: every output declared in output_mask must be given and no other; env_id_base must fit the 32-bit Philox
    counter word; kernel_form must be a TS_FORM_* value."""
    from paper_2606_22332_b200 import binding as B
    w = W.config(2, n_envs=8)
    sim = _sim(w, outputs=("depth", "prox"))
    inp = sim.upload(w.inputs(0))
    out = sim.alloc_outputs()
    L = B.lib()
    si, so = sim._structs(inp, out, host=False)
    so.prox = None                                                          # declared, but not given
    assert L.ts_step(sim.h, C.byref(si), C.byref(so), sim._stream()) == 1 and b"declared in output_mask is NULL" in L.ts_last_error(sim.h)
    si, so = sim._structs(inp, out, host=False)
    so.contact = out["depth"].data_ptr()                                    # given, but not declared
    assert L.ts_step(sim.h, C.byref(si), C.byref(so), sim._stream()) == 1 and b"not declared" in L.ts_last_error(sim.h)
    si, so = sim._structs(inp, out, host=False)
    assert L.ts_step(sim.h, C.byref(si), C.byref(so), sim._stream()) == 0
    for bad in (dict(env_id_base=-1), dict(env_id_base=2 ** 32 - 4), dict(physics=dict(w.physics, kernel_form=3))):
        with pytest.raises(B.TsError, match="TS_ERR_INVALID_ARG"):
            B.TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=bad.get("physics", w.physics), env_id_base=bad.get("env_id_base", 0))
    ok = B.TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=w.physics, env_id_base=2 ** 32 - 8)   # the last admissible base
    ok.close()


def test_two_contexts_with_different_shared_memory_needs():
    """the dynamic shared-memory attribute is per device, not per ctx.  A K = 2 ctx (twice the frames per
    block) created FIRST and a K = 1 ctx created after it must both keep stepping, in either order."""
    import torch
    from paper_2606_22332_b200.binding import TactileSim
    w = W.config(2, n_envs=32)
    w3 = W.config(3, n_envs=1)
    E = w.E
    types2 = np.zeros((E, 2), np.int32); params2 = np.zeros((E, 2, 4), np.float32)
    types2[:, 0] = w.types[:, 0]; params2[:, 0] = w.params[:, 0]
    types2[:, 1] = 1; params2[:, 1, 0] = 0.02
    big = TactileSim(w.patches, w.T, E, w.L, 2, physics=w.physics, outputs=w.outputs)
    big.set_geometry(types2, params2, w3.bank, w3.voxel)
    small = _sim(w)
    ref = _sim(w)
    for s in range(3):
        inp = w.inputs(s)
        two = {k: (np.ascontiguousarray(np.concatenate([v, v + (0.2 if k == "obj_pos" else 0.0)], axis=1)) if k.startswith("obj_") else v)
               for k, v in inp.items()}
        a = big.step(big.upload(two))          # the second object sits 20 cm away: it never wins
        b = small.step(small.upload(inp))
        c = ref.step(ref.upload(inp))
        torch.cuda.synchronize()
        for k in b:
            assert torch.equal(b[k], c[k]), k
        assert torch.allclose(a["depth"], b["depth"], atol=1e-6)


def test_per_step_kernel_times_and_kernel_form():
    import torch
    from paper_2606_22332_b200.binding import TactileSim
    w = W.config(4, n_envs=64)
    outs = {}
    for form, launches in (("fused", 2), ("split", 3)):
        sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=dict(w.physics, kernel_form=form), noise=w.noise, outputs=w.outputs)
        sim.set_geometry(w.types, w.params, w.bank, w.voxel)
        assert sim.launches_per_step() == launches
        sim.kernel_time_ms(2)
        for s in range(4):
            g = sim.step(sim.upload(w.inputs(s)))
        torch.cuda.synchronize()
        t = sim.kernel_times_ms()
        assert t.shape == (4, 4) and (t[:, :2] > 0).all() and ((t[:, 2] > 0).all() if form == "split" else (t[:, 2] < 0.02).all())
        ev = t[:, :3].sum(1)
        assert (t[:, 3] > 0).all() and (np.abs(t[:, 3] - ev) < 0.05 + 0.3 * ev).all()     # device-side clock agrees with the events
        ms, n = sim.kernel_time_ms(False)
        assert n == 4 and abs(ms - ev.mean()) < 0.05
        outs[form] = {k: v.clone() for k, v in g.items()}
        sim.close()
    for k in outs["fused"]:
        assert torch.equal(outs["fused"][k], outs["split"][k]), k      # both forms are bit-identical


def test_outputs_stay_inside_their_buffers():
    """compute-sanitizer is closed on this pool (profiles/r02_sanitizer.md), so the bounds are checked here: every
    output tensor is a window into a larger allocation whose margins hold a canary pattern; after stepping configs with
    ragged groups (240 / 248 slots), fillers, K = 1 and every noise knob, the margins must be untouched and the windows
    fully written (no canary left inside)."""
    import torch
    from paper_2606_22332_b200.binding import TactileSim
    for cid, n_envs, extra in ((5, 33, dict(read_delay=2, read_jitter=1, radius_noise=3e-4)), (2, 17, None), (1, 4, None)):
        w = W.config(cid, n_envs=n_envs)
        noise = dict(w.noise, **extra) if (w.noise and extra) else w.noise
        for form in (("fused", "split") if noise else ("auto",)):
            sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=dict(w.physics, kernel_form=form), noise=noise, outputs=w.outputs)
            sim.set_geometry(w.types, w.params, w.bank, w.voxel)
            sh = sim.out_shapes()
            pad = 4096
            big, out = {}, {}
            for k in sim.outputs:
                shape, dt = sh[k]
                n = int(np.prod(shape))
                canary = 0xA5 if dt == torch.uint8 else float("nan")
                big[k] = torch.full((n + 2 * pad,), canary, dtype=dt, device="cuda")
                out[k] = big[k][pad:pad + n].view(shape)
            for s in range(3):
                sim.step(sim.upload(w.inputs(s)), out)
            torch.cuda.synchronize()
            for k in sim.outputs:
                lo, hi, mid = big[k][:pad], big[k][-pad:], big[k][pad:-pad]
                if big[k].dtype == torch.uint8:
                    assert (lo == 0xA5).all() and (hi == 0xA5).all() and (mid <= 1).all(), (cid, form, k)
                else:
                    assert torch.isnan(lo).all() and torch.isnan(hi).all() and torch.isfinite(mid).all(), (cid, form, k)
            sim.close()


def test_chained_launches_equal_serialised_steps():
    """The frames kernel of step n+1 is launched as a programmatic dependent of step n's kernel and the step kernel as a
    dependent of its frames kernel (include/ts.h, "Programmatic dependent launch"): with steps enqueued back to back the
    blocks of the next grid are resident while the grid in front drains.  The result must equal, bit for bit, the same
    steps with a device synchronise after each one (no overlap possible), at BASELINE size where every SM holds blocks of
    both grids at the hand-over."""
    import torch
    w = W.config(5)
    xs = None
    res = []
    for serialise in (False, True, False):
        sim = _sim(w)
        if xs is None:
            xs = [sim.upload(w.inputs(s)) for s in range(6)]
        torch.cuda.synchronize()
        for s in range(36):
            out = sim.step(xs[s % 6])
            if serialise:
                torch.cuda.synchronize()
        torch.cuda.synchronize()
        res.append({k: v.clone() for k, v in out.items()})
        sim.close()
    for r in res[1:]:
        for k in res[0]:
            assert torch.equal(res[0][k], r[k]), k


def test_checkpoint_resume_is_bit_exact():
    """ts_get_state / ts_set_state: a blob taken after 6 steps (a masked reset among them) restores into a FRESH ctx of
    the same configuration, which then produces the same 6 further steps bit for bit: Schmitt bits, Maxwell hysteresis,
    drift, the read-delay ring, the noisy scalar readouts' state, the shear anchors and every counter travel with it.
    A blob from another configuration is refused and leaves the ctx untouched."""
    import torch
    from paper_2606_22332_b200.binding import TactileSim, TsError
    w = W.config(5, n_envs=48)
    pts, cid = W.point_cloud_bank(w, 500)
    noise = dict(w.noise, hyst_mode="maxwell", beta=0.5, tau=0.05, read_delay=2, read_jitter=1, sigma_white_force=2e-3,
                 radius_noise=3e-4, sigma_rw_depth=1e-5, sigma_white_prox=1e-3, sigma_rw_marker=1e-5, quant_marker=1e-4)
    outs = tuple(w.outputs) + ("depth_noisy", "prox_noisy", "marker_noisy")

    def make():
        s = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=dict(w.physics, shear_enable=1), noise=noise, outputs=outs)
        s.set_geometry(w.types, w.params, w.bank, w.voxel)
        s.set_pointclouds(pts, cid)
        return s

    a = make()
    for s in range(6):
        if s == 3:
            a.reset(torch.from_numpy((np.arange(w.E) % 3 == 0).astype(np.uint8)).cuda())
        a.step(a.upload(w.inputs(s)))
    blob = a.get_state()
    assert blob.nbytes == a.state_bytes() and blob.nbytes > w.E * w.T * 50
    want = []
    for s in range(6, 12):
        want.append({k: v.clone() for k, v in a.step(a.upload(w.inputs(s))).items()})
    b = make()
    b.step(b.upload(w.inputs(0)))                      # some other history first: the blob must overwrite all of it
    b.set_state(blob)
    for i, s in enumerate(range(6, 12)):
        got = b.step(b.upload(w.inputs(s)))
        torch.cuda.synchronize()
        for k in got:
            assert torch.equal(got[k], want[i][k]), (k, s)
    # a ctx with another configuration refuses the blob
    c = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=w.physics, noise=w.noise, outputs=w.outputs)
    c.set_geometry(w.types, w.params, w.bank, w.voxel)
    assert c.state_bytes() != blob.nbytes
    with pytest.raises(TsError):
        c.set_state(blob)
    with pytest.raises(TsError):
        c.set_state(blob[:64])
    a.close(); b.close(); c.close()


def test_meshes_and_pointclouds_on_one_ctx_in_any_order_and_replaced():
    """ts_set_meshes and ts_set_pointclouds own separate buffers: one ctx that gets both (in either order, each of them
    twice) and asks for raycast depth, point-cloud proximity and sheared markers at once equals, bit for bit, contexts
    that were given only what each output needs."""
    import torch
    from paper_2606_22332_b200.binding import TactileSim
    w = W.config(5, n_envs=24)
    pts, cid = W.point_cloud_bank(w, 600)
    meshes, mid = W.mesh_bank(w, 2)
    phys = dict(w.physics, shear_enable=1)
    x = None

    def run(outs, order, physics):
        nonlocal x
        sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=physics, outputs=outs)
        sim.set_geometry(w.types, w.params, w.bank, w.voxel)
        for what in order:
            sim.set_meshes(meshes, mid) if what == "m" else sim.set_pointclouds(pts, cid)
        if x is None:
            x = [sim.upload(w.inputs(s)) for s in range(3)]
        for s in range(3):
            g = sim.step(x[s])
        torch.cuda.synchronize()
        res = {k: v.clone() for k, v in g.items()}
        sim.close()
        return res

    ref_rc = run(("depth", "depth_rc", "nrm_rc"), "m", w.physics)
    ref_pc = run(("depth", "marker", "proxpc"), "p", phys)
    assert ref_rc["depth_rc"].abs().sum() > 0 and ref_pc["proxpc"].abs().sum() > 0
    for order in ("mp", "pm", "mpmp", "ppmm"):
        got = run(("depth", "marker", "proxpc", "depth_rc", "nrm_rc"), order, phys)
        for k in ("depth_rc", "nrm_rc"):
            assert torch.equal(got[k], ref_rc[k]), (order, k)
        for k in ("proxpc", "marker", "depth"):
            assert torch.equal(got[k], ref_pc[k]), (order, k)


def test_two_contexts_on_two_streams_run_concurrently():
    """Contexts are independent: two of them stepped from two CUDA streams at the same time (their chained launches and
    the per-device kernel attributes are shared machinery) give, bit for bit, what each gives when stepped alone."""
    import torch
    wa, wb = W.config(5, n_envs=3000), W.config(4, n_envs=2500)
    xa = xb = None
    res = {}
    for mode in ("alone", "together"):
        a, b = _sim(wa), _sim(wb)
        if xa is None:
            xa = [a.upload(wa.inputs(s)) for s in range(5)]
            xb = [b.upload(wb.inputs(s)) for s in range(5)]
        oa, ob = a.alloc_outputs(), b.alloc_outputs()
        torch.cuda.synchronize()
        if mode == "alone":
            for s in range(15):
                a.step(xa[s % 5], oa)
            torch.cuda.synchronize()
            for s in range(15):
                b.step(xb[s % 5], ob)
        else:
            sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
            for s in range(15):
                with torch.cuda.stream(sa):
                    a.step(xa[s % 5], oa)
                with torch.cuda.stream(sb):
                    b.step(xb[s % 5], ob)
        torch.cuda.synchronize()
        res[mode] = ({k: v.clone() for k, v in oa.items()}, {k: v.clone() for k, v in ob.items()})
        a.close(); b.close()
    for i in (0, 1):
        for k in res["alone"][i]:
            assert torch.equal(res["alone"][i][k], res["together"][i][k]), (i, k)
