"""Pins for the oracle's point-cloud ProximityTaxel (App. A.6, Eq. 12-17; constants P:267).

Closed forms: one tracked point on the taxel normal gives f = k rho P a_j and no torque; two points placed
symmetrically about the normal cancel the torque and double the force; a point outside the sensing sphere contributes
nothing and P falls linearly to 0 at the sphere; a sliding object adds k_s rho P v_t along the tangential relative
velocity only; rho = density / N_tracked; the reported channels are R_L^T f^w, R_L^T tau^w (rotating the link rotates
them back); a rigid transform of the whole scene changes nothing; and the sum over a random cloud equals a numpy
evaluation of Eq. 12-17 written out here.
"""
import numpy as np

from oracle import oracle as O

R, KF, KS, DENS = (float(np.float32(v)) for v in (0.01, 300.0, 10.0, 100.0))


def _patch():
    return dict(link=0, origin=(0, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=0.004, size_v=0.004, nu=1, nv=1,
                radius=2e-3, marker_nu=0, marker_nv=0)


def _run(points, link_pos=(0, 0, 0), link_quat=(1, 0, 0, 0), obj_pos=(0, 0, 0), obj_quat=(1, 0, 0, 0), vL=(0, 0, 0), wL=(0, 0, 0),
         vO=(0, 0, 0), wO=(0, 0, 0)):
    pts = np.asarray(points, np.float32).reshape(1, -1, 3)
    o = O.Oracle([_patch()], 1, 1, 1, np.arange(1))
    o.set_geometry(np.zeros((1, 1), np.int32), np.zeros((1, 1, 4), np.float32))      # no SDF object: the cloud is the geometry
    o.set_pointclouds(pts, np.zeros((1, 1), np.int32))
    f = lambda v, n: np.asarray(v, np.float32).reshape(1, 1, n)
    inp = dict(link_pos=f(link_pos, 3), link_quat=f(link_quat, 4), link_linvel=f(vL, 3), link_angvel=f(wL, 3),
               obj_pos=f(obj_pos, 3), obj_quat=f(obj_quat, 4), obj_linvel=f(vO, 3), obj_angvel=f(wO, 3))
    return o.step(inp, want=("proxpc",))["proxpc"][0, 0]


def test_single_point_on_the_normal():
    # taxel at the origin, normal +z; one tracked point 4 mm above it: P = 6 mm, rho = 100 / 1
    out = _run([[0, 0, 0.004]])
    P = R - float(np.float32(0.004))
    np.testing.assert_allclose(out, [0, 0, KF * DENS * P, 0, 0, 0], rtol=1e-12, atol=1e-15)
    assert not _run([[0, 0, 0.0101]]).any()                                # outside the sensing sphere
    np.testing.assert_allclose(_run([[0, 0, 0.0099]])[2], KF * DENS * (R - float(np.float32(0.0099))), rtol=1e-9)   # linear fall-off to 0


def test_symmetric_points_cancel_the_torque_and_density_scale():
    d = float(np.float32(0.003))
    one = _run([[0.003, 0, 0.004]])
    dist = np.hypot(d, float(np.float32(0.004)))
    P = R - dist
    # Eq. 17: tau = k rho P (p - q) x a = k rho P (dx, 0, dz) x (0, 0, 1) = k rho P (0, -dx, 0)
    np.testing.assert_allclose(one, [0, 0, KF * DENS * P, 0, -KF * DENS * P * d, 0], rtol=1e-12, atol=1e-15)
    two = _run([[0.003, 0, 0.004], [-0.003, 0, 0.004]])
    # rho = density / 2 tracked points: the force equals the single-point force, the torque cancels
    np.testing.assert_allclose(two, [0, 0, KF * DENS * P, 0, 0, 0], rtol=1e-12, atol=1e-15)
    # a far-away third tracked point only dilutes rho (N_active counts tracked points, reading Q27)
    three = _run([[0.003, 0, 0.004], [-0.003, 0, 0.004], [0.5, 0.5, 0.5]])
    np.testing.assert_allclose(three, two * 2.0 / 3.0, rtol=1e-12, atol=1e-15)


def test_slip_term_is_tangential_only():
    P = R - float(np.float32(0.004))
    # object slides along +x at 0.2 m/s and approaches along -z at 0.1 m/s: only the tangential part enters (Eq. 14)
    out = _run([[0, 0, 0.004]], vO=(0.2, 0, -0.1))
    np.testing.assert_allclose(out, [KS * DENS * P * float(np.float32(0.2)), 0, KF * DENS * P, 0, 0, 0], rtol=1e-12, atol=1e-15)
    # the taxel's own motion counts with the opposite sign (Eq. 13: v_p - v_tax)
    out2 = _run([[0, 0, 0.004]], vL=(0.2, 0, 0))
    np.testing.assert_allclose(out2[0], -KS * DENS * P * float(np.float32(0.2)), rtol=1e-12)
    # a spinning object: v_p = w_O x (p - p_O), p on the axis -> zero; off the axis -> w x r
    out3 = _run([[0.003, 0, 0.004]], wO=(0, 0, 2.0))
    dist = np.hypot(float(np.float32(0.003)), float(np.float32(0.004)))
    np.testing.assert_allclose(out3[1], KS * DENS * (R - dist) * 2.0 * float(np.float32(0.003)), rtol=1e-12)


def test_link_frame_and_rigid_invariance():
    rng = np.random.default_rng(3)
    pts = rng.normal(0, 0.006, (40, 3))
    base = _run(pts, vO=(0.1, -0.05, 0.02), wO=(0.3, 0.1, -0.2), vL=(0.01, 0.02, 0.0), wL=(0.0, 0.4, 0.1))
    assert np.abs(base[:5]).min() > 0 and base[5] == 0          # tau ~ (p - q) x a has no component along a
    # apply one rigid transform to link and object (and rotate the velocities): every channel is link-frame -> unchanged
    q = np.array([0.3, -0.5, 0.7, 0.4]); q /= np.linalg.norm(q)
    w, x, y, z = q
    Rm = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                   [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                   [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
    t = np.array([0.05, -0.02, 0.03])
    moved = _run(pts, link_pos=t, link_quat=q, obj_pos=t, obj_quat=q, vO=Rm @ [0.1, -0.05, 0.02], wO=Rm @ [0.3, 0.1, -0.2],
                 vL=Rm @ [0.01, 0.02, 0.0], wL=Rm @ [0.0, 0.4, 0.1])
    np.testing.assert_allclose(moved, base, rtol=2e-5, atol=1e-9)        # fp32 rounding of the rotated inputs only


def test_random_cloud_against_eq12_17_written_out():
    rng = np.random.default_rng(11)
    pts = rng.normal(0, 0.007, (300, 3)).astype(np.float32)
    vO, wO, vL, wL = (np.asarray(v, np.float32).astype(np.float64) for v in ((0.1, -0.05, 0.02), (0.3, 0.1, -0.2), (0.01, 0.02, 0.0), (0.0, 0.4, 0.1)))
    pL = np.asarray((0.001, -0.002, 0.0005), np.float32).astype(np.float64)
    out = _run(pts, link_pos=pL, vO=vO, wO=wO, vL=vL, wL=wL)
    p = pts.astype(np.float64); q = pL; a = np.array([0, 0, 1.0])
    dv = p - q
    dist = np.linalg.norm(dv, axis=1)
    m = dist < R
    P = R - dist[m]
    rho = DENS / len(p)
    vp = vO + np.cross(wO, p[m])                      # p_O = 0
    vtax = vL + np.cross(wL, q - pL)
    vr = vp - vtax
    vt = vr - np.outer(vr @ a, a)
    f = KF * rho * P.sum() * a + KS * rho * (P[:, None] * vt).sum(0)
    tau = KF * rho * (P[:, None] * np.cross(dv[m], a)).sum(0)
    assert m.sum() > 50
    np.testing.assert_allclose(out, np.concatenate([f, tau]), rtol=1e-11, atol=1e-14)
