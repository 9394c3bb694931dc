"""Pins for the oracle's raycast depth backend (App. A.1; reading Q28): per triangle a sphere-triangle
closest-point test (penetration R_j - dist) and a ray-triangle test from the probe centre along -a_j (penetration
R_j - hit_distance); the deepest wins; the normal is the winning triangle's face normal.

Pinned against: dense barycentric sampling of the triangle (closest point), the closed form of a ray meeting a plane,
the exact box SDF on a 12-triangle cube mesh (the two backends agree where the nearest feature is a face, edge or
corner of a convex mesh seen from outside), the face normal, and the analytic star surface on a fine star mesh.
"""
import numpy as np

from oracle import oracle as O
from paper_2606_22332_b200 import workloads as W

R_TAX = 2.0e-3


def test_closest_point_triangle_vs_dense_sampling():
    rng = np.random.default_rng(0)
    s = np.linspace(0, 1, 201)
    U, V = np.meshgrid(s, s)
    m = U + V <= 1.0
    U, V = U[m], V[m]
    for _ in range(40):
        a, b, c, p = rng.normal(size=(4, 3))
        cp = O.closest_point_triangle(p, a, b, c)
        S = a + U[:, None] * (b - a) + V[:, None] * (c - a)
        dmin = np.linalg.norm(S - p, axis=1).min()
        d = np.linalg.norm(cp - p)
        assert d <= dmin + 1e-12 and dmin - d < 0.02                      # never worse than any sample; sampling is 1/200 coarse
        # the returned point lies on the triangle: barycentric coordinates in [0, 1]
        Mx = np.stack([b - a, c - a], 1)
        uv, *_ = np.linalg.lstsq(Mx, cp - a, rcond=None)
        assert uv.min() > -1e-9 and uv.sum() < 1 + 1e-9 and np.linalg.norm(Mx @ uv - (cp - a)) < 1e-9
    # hand cases: above the interior, beside an edge, beyond a vertex
    a, b, c = np.array([0, 0, 0.]), np.array([1, 0, 0.]), np.array([0, 1, 0.])
    np.testing.assert_allclose(O.closest_point_triangle([0.2, 0.3, 5], a, b, c), [0.2, 0.3, 0], atol=1e-15)
    np.testing.assert_allclose(O.closest_point_triangle([0.5, -2, 1], a, b, c), [0.5, 0, 0], atol=1e-15)
    np.testing.assert_allclose(O.closest_point_triangle([-1, -1, 3], a, b, c), [0, 0, 0], atol=1e-15)
    np.testing.assert_allclose(O.closest_point_triangle([1, 1, 0], a, b, c), [0.5, 0.5, 0], atol=1e-15)


def test_ray_triangle_closed_forms():
    a, b, c = np.array([0, 0, 0.]), np.array([1, 0, 0.]), np.array([0, 1, 0.])
    d = np.array([0.3, 0.1, -1.0]); d /= np.linalg.norm(d)
    o = np.array([0.1, 0.2, 0.5])
    t = O.ray_triangle(o, d, a, b, c)
    assert abs(t - 0.5 / -d[2]) < 1e-14 and abs((o + t * d)[2]) < 1e-15    # plane z = 0: t = o_z / -d_z
    assert O.ray_triangle(o, -d, a, b, c) == -1.0                           # pointing away
    assert O.ray_triangle([2, 2, 0.5], [0, 0, -1.0], a, b, c) == -1.0       # beside the triangle
    assert abs(O.ray_triangle([0.2, 0.2, -0.5], [0, 0, 1.0], a, b, c) - 0.5) < 1e-15   # back face counts too (Q28)
    assert O.ray_triangle(o, [1.0, 0, 0], a, b, c) == -1.0                  # parallel


def _scene(meshes, mesh_id, link_pos, link_quat=(1, 0, 0, 0)):
    patch = dict(link=0, origin=(0, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=0.01, size_v=0.01, nu=4, nv=4, radius=R_TAX,
                 marker_nu=0, marker_nv=0)
    E = len(link_pos)
    o = O.Oracle([patch], 16, 1, 1, np.arange(E))
    o.set_geometry(np.full((E, 1), 2, np.int32), np.tile(np.array([0.02, 0.03, 0.025, 0], np.float32), (E, 1, 1)))   # the exact box, for the SDF backend
    o.set_meshes(meshes, mesh_id)
    f = lambda v, n: np.ascontiguousarray(np.asarray(v, np.float32).reshape(E, 1, n))
    z3, q0 = np.zeros((E, 3)), np.tile([1.0, 0, 0, 0], (E, 1))
    inp = dict(link_pos=f(link_pos, 3), link_quat=f(np.tile(link_quat, (E, 1)), 4), link_linvel=f(z3, 3), link_angvel=f(z3, 3),
               obj_pos=f(z3, 3), obj_quat=f(q0, 4), obj_linvel=f(z3, 3), obj_angvel=f(z3, 3))
    return o.step(inp, want=("depth", "depth_rc"))   # (aux_phi = the box SDF at the taxel centre)


def test_cube_mesh_agrees_with_the_exact_box_from_outside():
    # taxel spheres approaching the box from outside: the nearest feature of the mesh (face, edge, corner) is the nearest
    # point of the box, so R - dist equals the SDF depth; the ray test (from the centre along -a) never exceeds it (Q28)
    rng = np.random.default_rng(4)
    b = np.array([0.02, 0.03, 0.025])
    E = 200
    u = rng.normal(size=(E, 3)); u /= np.linalg.norm(u, axis=1, keepdims=True)
    pos = u * (np.abs(b / np.abs(u)).min(1, keepdims=True)) + u * rng.uniform(0.0005, 0.003, (E, 1))   # 0.5-3 mm outside the surface
    r = _scene([W.cube_mesh(b)], np.zeros((E, 1), np.int32), pos)
    out = r["aux_phi"] >= 0                                                          # taxel centre outside the box
    assert ((r["depth"] > 0) & out).sum() > 300
    np.testing.assert_allclose(r["depth_rc"][out], r["depth"][out], rtol=0, atol=2e-9)   # fp32 mesh vertices vs fp32 box extents
    # a centre INSIDE the mesh sees the nearest face from behind: R - |phi| instead of the SDF backend's R + |phi| (P:188
    # "the two backends ... differ at sharp features"; here: once the centre has passed the surface)
    ins = r["aux_phi"] < -1e-6
    assert ins.any()
    np.testing.assert_allclose(r["depth_rc"][ins], np.maximum(0.0, R_TAX + r["aux_phi"][ins]), rtol=0, atol=2e-9)
    # the face normal: press the pad flat onto the +z face: every touching taxel reports (0, 0, 1) rotated into the link frame
    qd = np.array([0.0, 1.0, 0.0, 0.0])                                             # link rotated 180 deg about x: link +z = world -z
    r2 = _scene([W.cube_mesh(b)], np.zeros((1, 1), np.int32), [[0, 0, 0.026]], link_quat=qd)
    touch = r2["depth_rc"][0] > 0
    assert touch.all()
    np.testing.assert_allclose(r2["depth_rc"][0], R_TAX - 0.001, atol=1e-9)
    np.testing.assert_allclose(r2["nrm_rc"][0], np.tile([0, 0, -1.0], (16, 1)), atol=1e-12)    # world +z seen from the flipped link
    assert (r2["aux_rc_gap"][0] > 1e-4).all()                                        # the neighbouring faces are far behind
    # no mesh -> zeros
    r3 = _scene([W.cube_mesh(b)], np.full((1, 1), -1, np.int32), [[0, 0, 0.026]], link_quat=qd)
    assert not r3["depth_rc"].any() and not r3["nrm_rc"].any()


def test_star_mesh_depth_vs_analytic_surface():
    # a fine star mesh (5,120 triangles): the raycast depth of probes near the surface agrees with R - (analytic distance
    # estimate f / |grad f|) to the discretisation error of the mesh (chord error ~ edge^2 / 8 r ~ 1e-5 m)
    V, F = W.star_mesh(4)
    assert len(F) == 20 * 4 ** 4
    rng = np.random.default_rng(9)
    E = 64
    u = rng.normal(size=(E, 3)); u /= np.linalg.norm(u, axis=1, keepdims=True)
    rad = W.star_radius(u)
    pos = u * (rad + 0.001)[:, None]                                                 # pad centres 1 mm outside the analytic surface
    patch = dict(link=0, origin=(0, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=0.002, size_v=0.002, nu=1, nv=1, radius=R_TAX,
                 marker_nu=0, marker_nv=0)
    o = O.Oracle([patch], 1, 1, 1, np.arange(E))
    o.set_geometry(np.zeros((E, 1), np.int32), np.zeros((E, 1, 4), np.float32))
    o.set_meshes([(V, F)], np.zeros((E, 1), np.int32))
    f = lambda v, n: np.ascontiguousarray(np.asarray(v, np.float32).reshape(E, 1, n))
    z3, q0 = np.zeros((E, 3)), np.tile([1.0, 0, 0, 0], (E, 1))
    inp = dict(link_pos=f(pos, 3), link_quat=f(q0, 4), link_linvel=f(z3, 3), link_angvel=f(z3, 3), obj_pos=f(z3, 3),
               obj_quat=f(q0, 4), obj_linvel=f(z3, 3), obj_angvel=f(z3, 3))
    d = o.step(inp, want=("depth_rc",))["depth_rc"][:, 0]
    assert (d > 0).all()
    # true distance from a point 1 mm out along the radius to the star surface is <= 1 mm and >= 1 mm * cos(tilt) ~ 0.9 mm
    assert (d >= R_TAX - 0.001 - 6e-5).all() and (d <= R_TAX - 0.0008).all()      # chord sag of the 2.7 mm edges ~ 2-4e-5 m
