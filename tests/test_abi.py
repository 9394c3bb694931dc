"""CPU-side checks of the boundary: the library loads, exports every declared symbol, the layout
builder (host code of the product) agrees with the oracle's own builder, host-side validation."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2606_22332_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2606_22332_b200 import build, binding
    build.build()
    return binding


def test_library_exports_every_declared_symbol(B):
    hdr = open(os.path.join(ROOT, "include", "ts.h")).read()
    declared = set(re.findall(r"\b(ts_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(B.SYMBOLS), declared ^ set(B.SYMBOLS)
    L = B.lib()
    for s in declared:
        assert hasattr(L, s), s
    assert b"sm_100a" in L.ts_version()


def test_struct_sizes_match_header(B):
    # ts_patch_desc: 1+3+3+3+2 floats/ints + 2 + 1 + 2 = 17 x 4 bytes; ts_step_in 8 ptrs; ts_step_out 7 ptrs
    assert C.sizeof(B.PatchDesc) == 17 * 4
    assert C.sizeof(B.StepIn) == 8 * 8 and C.sizeof(B.StepOut) == 13 * 8
    cfg = B.Config()
    B.lib().ts_config_default(C.byref(cfg))
    assert (cfg.k_n, cfg.c_n, cfg.k_t, cfg.k_omega) == (500.0, 1.0, 2.0, 2.0)          # Eq. 10
    assert cfg.alpha == pytest.approx(1.2) and cfg.eta_on == pytest.approx(5e-4)
    assert (cfg.s_d, cfg.lambda_d) == (100.0, 8000.0) and cfg.march_steps == 16
    assert cfg.chi == 0.0 and cfg.output_mask == 31
    assert (cfg.gain_min, cfg.gain_max) == (1.0, 1.0) and cfg.stuck_max_torque == 0.0
    assert cfg.xtalk_sigma == 0.0 and cfg.radius_noise == 0.0 and (cfg.read_delay, cfg.read_jitter) == (0, 0) and C.sizeof(B.Config) % 8 == 0                         # last field lands right


@pytest.mark.parametrize("cid", [1, 2, 3, 4])
def test_layout_builder_matches_oracle_builder(B, cid):
    """two independent implementations of S0 (product C++, oracle C++) give the same fp32 layout"""
    from oracle import oracle as O
    w = W.config(cid, n_envs=1)
    mask = None
    if cid == 3:
        mask = np.ones(w.L, np.uint8); mask[[2, 11]] = 0
    lay = B.Layout(w.patches, w.T, mask, w.L).view()
    o = O.Oracle(w.patches, w.T, w.L, 1, np.arange(1), link_mask=mask)
    ref = o.layout()
    for k in ("pos", "nrm", "radius", "marker_pos", "marker_nrm"):
        np.testing.assert_array_equal(lay[k].astype(np.float64), ref[k], err_msg=k)
    for k in ("link", "patch", "nbr", "marker_patch"):
        np.testing.assert_array_equal(lay[k], ref[k], err_msg=k)
    assert lay["pos"].shape == (w.T, 3) and (lay["radius"] > 0).sum() == sum(
        p["nu"] * p["nv"] for p in w.patches if mask is None or mask[p["link"]])


def test_layout_validation(B):
    L = B.lib()
    ok = dict(link=0, origin=(0, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=0.01, size_v=0.01, nu=4, nv=4,
              radius=0.002)
    for bad in (dict(nu=9, nv=8), dict(nu=0), dict(radius=0.0), dict(u_axis=(1, 1, 0)), dict(v_axis=(1, 0, 0)),
                dict(marker_nu=3, marker_nv=0), dict(marker_nu=9, marker_nv=9), dict(link=-1)):
        with pytest.raises(B.TsError):
            B.Layout([dict(ok, **bad)], 100)
    with pytest.raises(B.TsError):
        B.Layout([ok], 15)                       # fewer slots than the patch needs
    lay = B.Layout([ok], 20)
    assert lay.view()["patch"].tolist() == [0] * 16 + [-1] * 4
    assert L.ts_destroy(None) == 0 and L.ts_layout_destroy(None) == 0
    assert L.ts_step(None, None, None, None) == 1 and L.ts_reset(None, None, None) == 1


def test_create_rejects_bad_config_before_touching_cuda(B):
    lay = B.Layout(W.config(1).patches, 200)
    h = C.c_void_p()
    for bad in (dict(physics=dict(eta_off=6e-4)), dict(physics=dict(march_steps=65)), dict(n_links=3),
                dict(noise=dict(noise_enable=1, p_dead=1.0)), dict(outputs=["ft_noisy"]),
                dict(noise=dict(noise_enable=1, gain_min=0.0)), dict(noise=dict(noise_enable=1, gain_min=1.2, gain_max=1.1)),
                dict(noise=dict(noise_enable=1, quant_force=-1e-3)), dict(noise=dict(noise_enable=1, sigma_white_torque=-1.0)),
                dict(noise=dict(noise_enable=1, stuck_min_force=1.0, stuck_max_force=0.5)),
                dict(noise=dict(noise_enable=1, xtalk_sigma=1.5)), dict(noise=dict(noise_enable=1, xtalk_sigma=-0.1)),
                dict(noise=dict(noise_enable=1, radius_noise=-1e-4)), dict(noise=dict(noise_enable=1, read_delay=-1)),
                dict(noise=dict(noise_enable=1, read_delay=60, read_jitter=5)), dict(noise=dict(noise_enable=1, radius_noise=float("inf")))):
        kw = dict(n_envs=4, n_links=16, objs_per_env=1, layout=lay)
        kw.update(bad)
        cfg = B.make_config(**kw)
        assert B.lib().ts_create(C.byref(cfg), 0, C.byref(h)) == 1, bad
        assert B.lib().ts_last_error(None)
