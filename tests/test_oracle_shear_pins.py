"""Pins for the oracle's elastomer shear history (App. A.7, Eq. 22-23; constants P:304; reading R11).

One tracked point over a flat pad: the anchor is set when the point sinks below -eta_enter (so the first anchored step
shows no shear), the marker under the point then moves by exactly s_s (z_p - e_p)_tangential h_p, markers beside it by
that times exp(-lambda_s r^2), the normal component of the slide is projected out, the anchor survives shallow lifting
up to +eta_exit and is cleared above it (re-anchoring at the new position), a reset clears it, a point beside the pad
never anchors, and the shear sum is added to the dilation output (Eq. 23).
"""
import math

import numpy as np

from oracle import oracle as O

S_S, LAM_S, ENTER, EXIT = (float(np.float32(v)) for v in (100.0, 2000.0, 1e-5, 1e-4))


def _oracle(shear=1):
    # one 20 x 20 mm pad, 4 x 4 taxels, 5 x 5 markers (marker (2, 2) sits at the pad centre), normal +z
    patch = dict(link=0, origin=(0, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=0.02, size_v=0.02, nu=4, nv=4, radius=2e-3,
                 marker_nu=5, marker_nv=5)
    o = O.Oracle([patch], 16, 1, 1, np.arange(1), physics=dict(shear_enable=shear))
    o.set_geometry(np.zeros((1, 1), np.int32), np.zeros((1, 1, 4), np.float32))      # no SDF object: dilation is zero
    o.set_pointclouds(np.zeros((1, 1, 3), np.float32), np.zeros((1, 1), np.int32))   # one tracked point at the object origin
    return o


def _step(o, obj_pos):
    f = lambda v, n: np.asarray(v, np.float32).reshape(1, 1, n)
    inp = dict(link_pos=f((0, 0, 0), 3), link_quat=f((1, 0, 0, 0), 4), link_linvel=f((0, 0, 0), 3), link_angvel=f((0, 0, 0), 3),
               obj_pos=f(obj_pos, 3), obj_quat=f((1, 0, 0, 0), 4), obj_linvel=f((0, 0, 0), 3), obj_angvel=f((0, 0, 0), 3))
    return o.step(inp, want=("marker",))["marker"][0].reshape(5, 5, 3)              # [v, u, xyz]


def test_anchor_enter_slide_exit_sequence():
    o = _oracle()
    h = float(np.float32(0.001))
    assert not _step(o, (0, 0, 0.002)).any()                     # above the pad: nothing
    assert not _step(o, (0, 0, -0.000005)).any()                 # 5 um inside, above -eta_enter = -10 um: no anchor yet
    assert not _step(o, (0, 0, -0.001)).any()                    # sinks to -1 mm: anchor set HERE, z_p - e_p = 0
    dx = float(np.float32(0.0005))
    m = _step(o, (0.0005, 0, -0.001))                            # slides 0.5 mm along +x at constant depth
    # marker (2,2) at the pad centre: r = x_j - z_p = (-dx, 0, .): weight exp(-lambda_s dx^2)
    want_c = S_S * dx * h * math.exp(-LAM_S * dx * dx)
    np.testing.assert_allclose(m[2, 2], [want_c, 0, 0], rtol=1e-12, atol=1e-18)
    # marker (2,3) one pitch (4 mm) further along +u: r = (0.004 - dx, 0)
    xm = float(np.float32(0.004))
    np.testing.assert_allclose(m[2, 3, 0], S_S * dx * h * math.exp(-LAM_S * (xm - dx) ** 2), rtol=1e-7)   # marker x is 0.2 * f32(0.02), rounded
    # slide with a normal component: only the tangential part of z_p - e_p enters (Pi_n); h_p follows the new depth
    m2 = _step(o, (0.0005, 0.0003, -0.0015))
    h2, dy = float(np.float32(0.0015)), float(np.float32(0.0003))
    w2 = S_S * h2 * math.exp(-LAM_S * (dx * dx + dy * dy))
    np.testing.assert_allclose(m2[2, 2], [w2 * dx, w2 * dy, 0], rtol=1e-12, atol=1e-18)
    # lifting to +50 um (below eta_exit = 100 um) keeps the anchor but h_p = 0: no output; sinking again resumes with the OLD anchor
    assert not _step(o, (0.0005, 0, 0.00005)).any()
    m3 = _step(o, (0.001, 0, -0.001))
    dx3 = float(np.float32(0.001))
    np.testing.assert_allclose(m3[2, 2, 0], S_S * dx3 * h * math.exp(-LAM_S * dx3 * dx3), rtol=1e-12)
    # lifting above eta_exit clears it: the next contact anchors at the new place (zero shear on its first step)
    assert not _step(o, (0.001, 0, 0.0002)).any()
    assert not _step(o, (0.001, 0, -0.001)).any()
    m4 = _step(o, (0.0012, 0, -0.001))
    d4 = float(np.float32(0.0012)) - float(np.float32(0.001))
    np.testing.assert_allclose(m4[2, 2, 0], S_S * d4 * h * math.exp(-LAM_S * float(np.float32(0.0012)) ** 2), rtol=1e-9)
    # reset clears the anchors
    o.reset()
    assert not _step(o, (0.0012, 0, -0.001)).any()


def test_point_beside_the_pad_never_anchors_and_switch():
    o = _oracle()
    _step(o, (0.011, 0, -0.001))                                 # 1 mm outside the 20 mm pad laterally
    assert not _step(o, (0.0115, 0, -0.001)).any()
    _step(o, (0.0095, 0, -0.001))                                # now over the pad: anchors
    assert _step(o, (0.009, 0, -0.001)).any()
    off = _oracle(shear=0)
    _step(off, (0, 0, -0.001))
    assert not _step(off, (0.0005, 0, -0.001)).any()             # shear_enable = 0: Eq. 23 keeps the dilation sum only


def test_shear_adds_to_dilation_eq23():
    # a sphere object pressing the pad: marker = dilation (Eq. 21) + shear (Eq. 22); the dilation part equals the run without shear
    patch = dict(link=0, origin=(0, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=0.02, size_v=0.02, nu=8, nv=8, radius=2e-3,
                 marker_nu=7, marker_nv=7)
    rng = np.random.default_rng(5)
    u = rng.normal(size=(1, 400, 3)); u /= np.linalg.norm(u, axis=-1, keepdims=True)
    pts = (0.03 * u).astype(np.float32)                          # tracked points on the r = 30 mm sphere
    outs = []
    for shear in (0, 1):
        o = O.Oracle([patch], 64, 1, 1, np.arange(1), physics=dict(shear_enable=shear))
        o.set_geometry(np.ones((1, 1), np.int32), np.full((1, 1, 4), 0.03, np.float32))
        o.set_pointclouds(pts, np.zeros((1, 1), np.int32))
        seq = []
        for k in range(4):
            seq.append(_step_sphere(o, (0.0004 * k, 0.0, 0.029)))   # sphere centre 29 mm above the pad: 1 mm indentation, sliding along +x
        outs.append(seq)
    d, s = outs
    np.testing.assert_allclose(s[0], d[0], rtol=0, atol=0)       # first contact step: anchors just set
    diff = s[3] - d[3]
    assert np.abs(diff[..., 0]).max() > 3e-4 and np.abs(diff[..., 2]).max() < 1e-15      # shear is tangential, along the slide
    assert (diff[..., 0] >= 0).all()


def _step_sphere(o, obj_pos):
    f = lambda v, n: np.asarray(v, np.float32).reshape(1, 1, n)
    inp = dict(link_pos=f((0, 0, 0), 3), link_quat=f((1, 0, 0, 0), 4), link_linvel=f((0, 0, 0), 3), link_angvel=f((0, 0, 0), 3),
               obj_pos=f(obj_pos, 3), obj_quat=f((1, 0, 0, 0), 4), obj_linvel=f((0, 0, 0), 3), obj_angvel=f((0, 0, 0), 3))
    return o.step(inp, want=("marker",))["marker"][0].copy()
