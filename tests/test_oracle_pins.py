"""Pins for the oracle (CPU only): closed forms, invariants, known answers and brute force.

Each test is chosen so that a plausible mistake in oracle/oracle.cpp (dropped term, wrong sign
or index, transposed operand) fails it.  P-numbers follow DESIGN.md "Pins".
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2606_22332_b200 import workloads as W

R_TAX = 2.0e-3


def one_patch(nu=1, nv=1, size_u=0.004, size_v=0.004, radius=R_TAX, mnu=0, mnv=0, link=0):
    return dict(link=link, origin=(0, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=size_u, size_v=size_v,
                nu=nu, nv=nv, radius=radius, marker_nu=mnu, marker_nv=mnv)


def scene(patches, T, E=1, L=1, physics=None, noise=None, geom=("sphere", [0.030]), bank=None, voxel=0.0):
    o = O.Oracle(patches, T, L, 1, np.arange(E), physics=physics, noise=noise)
    types = np.full((E, 1), O.GEOM[geom[0]], np.int32)
    params = np.zeros((E, 1, 4), np.float32)
    params[:, 0, :len(geom[1])] = geom[1]
    o.set_geometry(types, params, bank, voxel)
    return o


def inputs(E=1, L=1, link_pos=(0, 0, 0), link_quat=(1, 0, 0, 0), **kw):
    d = dict(link_pos=np.tile(np.asarray(link_pos, np.float32), (E, L, 1)),
             link_quat=np.tile(np.asarray(link_quat, np.float32), (E, L, 1)),
             link_linvel=np.zeros((E, L, 3), np.float32), link_angvel=np.zeros((E, L, 3), np.float32),
             obj_pos=np.zeros((E, 1, 3), np.float32), obj_quat=np.tile(np.array([1, 0, 0, 0], np.float32), (E, 1, 1)),
             obj_linvel=np.zeros((E, 1, 3), np.float32), obj_angvel=np.zeros((E, 1, 3), np.float32))
    for k, v in kw.items():
        d[k] = np.broadcast_to(np.asarray(v, np.float32), d[k].shape).copy()
    return d


# ------------------------------------------------------------------ P15 Philox
def test_philox_known_answers():
    kat = [((0, 0, 0, 0), (0, 0), (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
           ((0xffffffff,) * 4, (0xffffffff,) * 2, (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
           ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0),
            (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1))]
    for ctr, key, ref in kat:   # Random123 kat_vectors, philox4x32 10 rounds
        assert tuple(int(x) for x in O.philox(ctr, key)) == ref


def test_uniform_and_box_muller():
    assert O.uniform(0) == 2.0 ** -24
    assert O.uniform(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert float(np.float32(O.uniform(0x12345678))) == O.uniform(0x12345678)   # exact in fp32
    z = O.box_muller(0x80000000, 0)          # u_a ~ 0.5, u_b ~ 0: z0 = sqrt(2 ln 2), z1 ~ 0
    ua, ub = (2.0 * (0x80000000 >> 9) + 1) / 2 ** 24, 2.0 ** -24
    assert z[0] == pytest.approx(math.sqrt(-2 * math.log(ua)) * math.cos(2 * math.pi * ub), rel=1e-14)
    assert z[1] == pytest.approx(math.sqrt(-2 * math.log(ua)) * math.sin(2 * math.pi * ub), rel=1e-12)
    rng = np.random.default_rng(1)
    w = rng.integers(0, 2 ** 32, size=(20000, 2), dtype=np.uint64)
    zz = np.array([O.box_muller(a, b) for a, b in w]).ravel()
    assert abs(zz.mean()) < 4 / math.sqrt(zz.size)
    assert abs(zz.var() - 1) < 0.03
    assert abs((zz ** 4).mean() - 3) < 0.15
    assert abs((zz[0::2] * zz[1::2]).mean()) < 0.03          # cos / sin legs uncorrelated


# ------------------------------------------------------------------ P1, P5 primitives
def test_sphere_closed_form(golden):
    x = np.array([0.012, -0.02, 0.0205])
    q = O.sdf_query("sphere", [0.03], x)
    assert q["phi"] == pytest.approx(np.linalg.norm(x) - 0.03, abs=1e-15)
    np.testing.assert_allclose(q["grad"], x / np.linalg.norm(x), atol=1e-15)
    assert R_TAX + 0.030 - 0.031 == pytest.approx(golden["depth_sphere_31mm"], rel=1e-12)


def _surface_samples_box(b, n):
    g = np.linspace(-1, 1, n)
    A, B = np.meshgrid(g, g, indexing="ij")
    pts = []
    for ax in range(3):
        for s in (-1, 1):
            p = np.zeros(A.shape + (3,))
            p[..., ax] = s
            p[..., (ax + 1) % 3] = A
            p[..., (ax + 2) % 3] = B
            pts.append(p.reshape(-1, 3) * b)
    return np.concatenate(pts)


def _surface_samples_capsule(r, h, n):
    th = np.linspace(0, 2 * np.pi, n, endpoint=False)
    z = np.linspace(-h, h, n)
    TH, Z = np.meshgrid(th, z, indexing="ij")
    cyl = np.stack([r * np.cos(TH), r * np.sin(TH), Z], -1).reshape(-1, 3)
    ph = np.linspace(0, np.pi / 2, n // 2)
    TH, PH = np.meshgrid(th, ph, indexing="ij")
    cap = np.stack([r * np.cos(TH) * np.cos(PH), r * np.sin(TH) * np.cos(PH), r * np.sin(PH)], -1).reshape(-1, 3)
    top = cap + [0, 0, h]
    bot = cap * [1, 1, -1] - [0, 0, h]
    return np.concatenate([cyl, top, bot])


@pytest.mark.parametrize("kind,params", [("box", [0.02, 0.03, 0.015]), ("capsule", [0.015, 0.03])])
def test_primitive_vs_brute_force(kind, params):
    """|phi| = distance to the nearest of a dense set of surface samples; sign from the inside test."""
    rng = np.random.default_rng(3)
    if kind == "box":
        surf = _surface_samples_box(np.array(params), 400)
        inside = lambda x: np.all(np.abs(x) < params)
    else:
        surf = _surface_samples_capsule(params[0], params[1], 700)
        inside = lambda x: np.linalg.norm(x - [0, 0, np.clip(x[2], -params[1], params[1])]) < params[0]
    for x in rng.uniform(-0.06, 0.06, (60, 3)):
        q = O.sdf_query(kind, params, x)
        dist = np.min(np.linalg.norm(surf - x, axis=1))
        assert abs(q["phi"]) == pytest.approx(dist, abs=2e-4)          # sample spacing ~1.5e-4
        assert (q["phi"] < 0) == inside(x)
        # gradient: unit, and equal to the central difference of phi (independent of the formula for g)
        assert np.linalg.norm(q["grad"]) == pytest.approx(1.0, abs=1e-12)
        h = 1e-7
        fd = np.array([(O.sdf_query(kind, params, x + h * e)["phi"] - O.sdf_query(kind, params, x - h * e)["phi"])
                       / (2 * h) for e in np.eye(3)])
        if q["boxgap"] > 1e-5:                                          # away from the interior medial axis
            np.testing.assert_allclose(q["grad"], fd, atol=1e-5)


def test_box_special_cases():
    b = [0.02, 0.03, 0.015]
    q = O.sdf_query("box", b, [0.05, 0.0, 0.0])                          # face region
    assert q["phi"] == pytest.approx(0.03) and tuple(q["grad"]) == (1.0, 0.0, 0.0)
    q = O.sdf_query("box", b, [-0.05, -0.07, 0.0])                       # edge region
    assert q["phi"] == pytest.approx(math.hypot(0.03, 0.04))
    np.testing.assert_allclose(q["grad"], [-0.6, -0.8, 0.0], atol=1e-12)
    q = O.sdf_query("box", b, [0.0, 0.0, -0.012])                        # interior: nearest face is -z
    assert q["phi"] == pytest.approx(-0.003) and tuple(q["grad"]) == (0.0, 0.0, -1.0)
    q = O.sdf_query("box", b, [0.0, 0.0, 0.0])                           # interior, w = (-.02,-.03,-.015)
    assert q["phi"] == pytest.approx(-0.015) and q["boxgap"] == pytest.approx(0.005)


def test_capsule_special_cases():
    q = O.sdf_query("capsule", [0.015, 0.03], [0.04, 0.0, 0.01])         # cylinder part
    assert q["phi"] == pytest.approx(0.025)
    np.testing.assert_allclose(q["grad"], [1, 0, 0], atol=1e-15)
    q = O.sdf_query("capsule", [0.015, 0.03], [0.0, 0.03, 0.07])         # cap
    assert q["phi"] == pytest.approx(0.05 - 0.015)
    np.testing.assert_allclose(q["grad"], [0, 0.6, 0.8], atol=1e-15)


# ------------------------------------------------------------------ P6, P7, P9 grid
def _affine_grid(N, hv, n, c):
    ax = (np.arange(N) - 0.5 * (N - 1)) * hv
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    return (n[0] * X + n[1] * Y + n[2] * Z + c)


def test_grid_affine_exact():
    """trilinear interpolation reproduces an affine field; gradient == n everywhere (flat-plane check)"""
    N, hv = 16, 0.002
    n = np.array([0.36, -0.48, 0.8])
    g64 = _affine_grid(N, hv, n, 0.004)
    g = g64.astype(np.float32)
    rng = np.random.default_rng(5)
    for x in rng.uniform(-0.0149, 0.0149, (200, 3)):
        q = O.sdf_query("grid", [0], x, grid=g, voxel=hv)
        assert q["phi"] == pytest.approx(n @ x + 0.004, abs=2e-9)        # fp32 storage of the nodes
        np.testing.assert_allclose(q["grad"], n, atol=2e-6)
    # x fastest: a field that depends on x only must give a gradient along x only
    gx = _affine_grid(N, hv, np.array([1.0, 0, 0]), 0.0).astype(np.float32)
    q = O.sdf_query("grid", [0], [0.003, -0.004, 0.005], grid=gx, voxel=hv)
    np.testing.assert_allclose(q["grad"], [1, 0, 0], atol=1e-5)
    assert q["phi"] == pytest.approx(0.003, abs=1e-9)


def test_grid_outside_extension():
    N, hv = 8, 0.002
    g = _affine_grid(N, hv, np.array([0.0, 0.0, 1.0]), 0.0).astype(np.float32)
    half = 0.5 * (N - 1) * hv
    x = np.array([half + 0.003, 0.001, 0.002])                           # 3 mm beyond the +x face
    q = O.sdf_query("grid", [0], x, grid=g, voxel=hv)
    assert q["phi"] == pytest.approx(0.002 + 0.003, abs=1e-9)            # phi_tri(clamped) + distance
    np.testing.assert_allclose(q["grad"], [0, 0, 1], atol=1e-5)           # gradient of the clamped point
    x = np.array([half + 0.003, -half - 0.004, 0.0])                     # beyond an edge
    q = O.sdf_query("grid", [0], x, grid=g, voxel=hv)
    assert q["phi"] == pytest.approx(0.0 + 0.005, abs=1e-9)


def _star_f_and_grad(x):
    """analytic f = |x| - 0.04 (1 + 0.2 Y32(x/|x|)) and its gradient, written out independently"""
    c = 0.25 * math.sqrt(105 / math.pi)
    X, Y, Z = x
    rho = math.sqrt(X * X + Y * Y + Z * Z)
    Yv = c * (X * X - Y * Y) * Z / rho ** 3
    f = rho - 0.04 * (1 + 0.2 * Yv)
    gradY = c * (np.array([2 * X * Z, -2 * Y * Z, X * X - Y * Y]) / rho ** 3 - 3 * (X * X - Y * Y) * Z * x / rho ** 5)
    return f, x / rho - 0.008 * gradY


def test_star_grid_vs_analytic():
    """value error O(h^2 |f''|), gradient error O(h |f''|); |f''| <~ 1/rho + 0.008 * 30/rho^2 ~ 200 1/m here"""
    N, hv = 64, 0.002
    g = W.star_grid(N, hv)
    rng = np.random.default_rng(7)
    n_checked = 0
    for _ in range(400):
        u = rng.standard_normal(3)
        u /= np.linalg.norm(u)
        x = u * rng.uniform(0.030, 0.058)
        f, gf = _star_f_and_grad(x)
        fd = np.array([(_star_f_and_grad(x + 1e-6 * e)[0] - _star_f_and_grad(x - 1e-6 * e)[0]) / 2e-6 for e in np.eye(3)])
        np.testing.assert_allclose(gf, fd, atol=1e-7)                     # the test's own formula is right
        q = O.sdf_query("grid", [0], x, grid=g, voxel=hv)
        assert q["phi"] == pytest.approx(f, abs=0.125 * 3 * hv * hv * 200)   # 3/8 h^2 max|f''|
        np.testing.assert_allclose(q["grad"], gf, atol=3 * hv * 200 * 0.5 + 1e-3)
        n_checked += 1
    assert n_checked == 400


def _point_tri_dist(p, a, b, c):
    """exact point-triangle distance (Ericson, Real-Time Collision Detection 5.1.5), own implementation"""
    ab, ac, ap = b - a, c - a, p - a
    d1, d2 = ab @ ap, ac @ ap
    if d1 <= 0 and d2 <= 0: return np.linalg.norm(p - a)
    bp = p - b
    d3, d4 = ab @ bp, ac @ bp
    if d3 >= 0 and d4 <= d3: return np.linalg.norm(p - b)
    vc = d1 * d4 - d3 * d2
    if vc <= 0 and d1 >= 0 and d3 <= 0: return np.linalg.norm(p - (a + ab * (d1 / (d1 - d3))))
    cp = p - c
    d5, d6 = ab @ cp, ac @ cp
    if d6 >= 0 and d5 <= d6: return np.linalg.norm(p - c)
    vb = d5 * d2 - d1 * d6
    if vb <= 0 and d2 >= 0 and d6 <= 0: return np.linalg.norm(p - (a + ac * (d2 / (d2 - d6))))
    va = d3 * d6 - d5 * d4
    if va <= 0 and (d4 - d3) >= 0 and (d5 - d6) >= 0:
        return np.linalg.norm(p - (b + (c - b) * ((d4 - d3) / ((d4 - d3) + (d5 - d6)))))
    den = 1.0 / (va + vb + vc)
    return np.linalg.norm(p - (a + ab * (vb * den) + ac * (vc * den)))


def _mesh_sdf(p, V, F):
    d = min(_point_tri_dist(p, V[f[0]], V[f[1]], V[f[2]]) for f in F)
    inside = all(np.cross(V[f[1]] - V[f[0]], V[f[2]] - V[f[0]]) @ (p - V[f[0]]) < 0 for f in F)   # convex, CCW out
    return -d if inside else d


def _cube_mesh(b):
    V = np.array([[sx, sy, sz] for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)], float) * b
    F = [(0, 1, 3), (0, 3, 2), (4, 6, 7), (4, 7, 5), (0, 4, 5), (0, 5, 1), (2, 3, 7), (2, 7, 6), (0, 2, 6), (0, 6, 4),
         (1, 5, 7), (1, 7, 3)]
    return V, F


def _tetra_mesh(s):
    V = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], float) * s
    F = [(0, 1, 2), (0, 3, 1), (0, 2, 3), (1, 3, 2)]
    c = V.mean(0)
    F = [f if np.cross(V[f[1]] - V[f[0]], V[f[2]] - V[f[0]]) @ (V[f[0]] - c) > 0 else (f[0], f[2], f[1]) for f in F]
    return V, F


def test_box_vs_cube_mesh_brute_force():
    b = np.array([0.012, 0.009, 0.015])
    V, F = _cube_mesh(b)
    rng = np.random.default_rng(9)
    for x in rng.uniform(-0.03, 0.03, (150, 3)):
        assert O.sdf_query("box", b, x)["phi"] == pytest.approx(_mesh_sdf(x, V, F), abs=1e-12)


@pytest.mark.parametrize("mesh", ["cube", "tetra"])
def test_grid_vs_mesh_brute_force(mesh):
    """brute-force mesh distance -> grid -> oracle lookup vs direct brute force at random points"""
    N, hv = 12, 0.004
    V, F = _cube_mesh(np.array([0.010, 0.008, 0.012])) if mesh == "cube" else _tetra_mesh(0.010)
    ax = (np.arange(N) - 0.5 * (N - 1)) * hv
    g = np.zeros((N, N, N))
    for k in range(N):
        for j in range(N):
            for i in range(N):
                g[k, j, i] = _mesh_sdf(np.array([ax[i], ax[j], ax[k]]), V, F)
    g32 = g.astype(np.float32)
    rng = np.random.default_rng(11)
    exact_hits = 0
    for x in rng.uniform(-0.021, 0.021, (300, 3)):
        q = O.sdf_query("grid", [0], x, grid=g32, voxel=hv)
        ref = _mesh_sdf(x, V, F)
        assert q["phi"] == pytest.approx(ref, abs=0.75 * hv)            # 1-Lipschitz field: |err| <= sqrt(3)/2 h
        # where the cell lies in one face's Voronoi region the field is affine -> lookup is exact
        i0 = np.clip(np.floor((x - ax[0]) / hv).astype(int), 0, N - 2)
        corners = np.array([[ax[i0[0] + a], ax[i0[1] + b_], ax[i0[2] + c_]] for a in (0, 1) for b_ in (0, 1) for c_ in (0, 1)])
        if mesh == "cube":
            bx = np.array([0.010, 0.008, 0.012])
            for axis in range(3):
                o1, o2 = (axis + 1) % 3, (axis + 2) % 3
                if np.all(corners[:, axis] > bx[axis]) and np.all(np.abs(corners[:, o1]) < bx[o1]) and \
                        np.all(np.abs(corners[:, o2]) < bx[o2]):
                    assert q["phi"] == pytest.approx(ref, abs=2e-9)
                    e = np.zeros(3); e[axis] = 1
                    np.testing.assert_allclose(q["grad"], e, atol=1e-5)
                    exact_hits += 1
    if mesh == "cube":
        assert exact_hits > 5


# ------------------------------------------------------------------ P1-P4 depth + kinematic F/T
def test_sphere_depth_and_spring(golden):
    """worked example: R = 2 mm, r = 30 mm, |q - c| = 31 mm, 0.5 mm and 2 mm variants, zero velocity"""
    for dist, name in ((0.031, "spring_1mm"), (0.0315, "spring_0p5mm"), (0.030, "spring_2mm")):
        o = scene([one_patch()], 1)
        out = o.step(inputs(link_pos=(0, 0, -dist)))
        d = float(np.float32(R_TAX)) + float(np.float32(0.030)) - float(np.float32(dist))   # inputs are fp32
        assert out["depth"][0, 0] == pytest.approx(d, abs=1e-12)
        f = out["ft"][0, 0]
        assert np.linalg.norm(f[:3]) == pytest.approx(golden[name], rel=2e-5)   # fp32 rounding of dist
        assert f[2] < 0 and abs(f[0]) < 1e-15 and abs(f[1]) < 1e-15            # pushes the taxel away (-z)
        np.testing.assert_allclose(f[3:], 0, atol=1e-15)                      # x_j = 0 -> no torque
    assert golden["s_at_1mm"] == pytest.approx(1e-3 ** 1.2, rel=1e-7)


def test_kinematic_ft_closed_forms(golden):
    m = np.array([0.0, 0.0, -1.0])
    xj = np.array([0.003, -0.002, 0.0])
    # spring + lever arm
    f = O.kinematic_ft(1e-3, m, xj)
    assert np.linalg.norm(f[:3]) == pytest.approx(golden["spring_1mm"], rel=1e-6)   # alpha is stored as fp32 1.2f
    np.testing.assert_allclose(f[3:], np.cross(xj, f[:3]), atol=1e-18)
    # damping: object approaches the taxel along m with 0.05 (v_rel . m_bar = 0.05)
    f = O.kinematic_ft(1e-3, m, [0, 0, 0], vO=0.05 * m)
    assert np.linalg.norm(f[:3]) == pytest.approx(golden["normal_1mm_v0p05"], rel=1e-6)
    f2 = O.kinematic_ft(1e-3, m, [0, 0, 0], vL=-0.05 * m)             # same relative velocity from the link side
    np.testing.assert_allclose(f, f2, atol=1e-15)
    # tangential, uncapped (mu = inf reproduces Eq. 8): -k_t v_t
    f = O.kinematic_ft(1e-3, m, [0, 0, 0], vO=[0.1, 0, 0], physics=dict(mu=float("inf")))
    assert f[0] == pytest.approx(-golden["tangential_v0p1"], rel=1e-12)
    assert f[2] == pytest.approx(-golden["spring_1mm"], rel=1e-6)   # alpha is stored as fp32 1.2f
    # capped at mu |f_n| (D2): 0.2 > 1.0 * 0.1256
    f = O.kinematic_ft(1e-3, m, [0, 0, 0], vO=[0.1, 0, 0], physics=dict(mu=1.0))
    assert f[0] == pytest.approx(-golden["spring_1mm"], rel=1e-6)   # alpha is stored as fp32 1.2f
    f = O.kinematic_ft(1e-3, m, [0, 0, 0], vO=[0.01, 0, 0], physics=dict(mu=1.0))   # below the cap: untouched
    assert f[0] == pytest.approx(-0.02, rel=1e-12)
    # torsional term -k_w ((w_C - w_L) . m) m_bar
    f = O.kinematic_ft(1e-3, m, [0, 0, 0], wO=[0, 0, 0.3], pO=[0, 0, 0], pL=[0, 0, 0])
    np.testing.assert_allclose(f[3:], -2.0 * (0.3 * m[2]) * m, atol=1e-15)
    f = O.kinematic_ft(1e-3, m, [0, 0, 0], wL=[0, 0, 0.3])
    np.testing.assert_allclose(f[3:], +2.0 * (0.3 * m[2]) * m, atol=1e-15)
    # Eq. 4: omega_C x (q - r_C) enters the point velocity
    f = O.kinematic_ft(1e-3, m, [0, 0, 0], pL=[0.1, 0, 0], wO=[0, 0, 1.0], physics=dict(mu=float("inf")))
    assert f[1] == pytest.approx(-2.0 * 0.1, rel=1e-12)                 # v_C = w x r = (0, 0.1, 0)
    # use_velocity = 0 drops every velocity term
    f = O.kinematic_ft(1e-3, m, xj, vO=[0.1, 0.2, 0.3], wO=[1, 2, 3], physics=dict(use_velocity=0))
    assert np.linalg.norm(f[:3]) == pytest.approx(golden["spring_1mm"], rel=1e-6)   # alpha is stored as fp32 1.2f
    np.testing.assert_allclose(f[3:], np.cross(xj, f[:3]), atol=1e-18)
    # link-frame output: rotate the link by 90 deg about x; world normal (0,0,-1) -> link (0,-1,0)
    qx = [math.sqrt(0.5), math.sqrt(0.5), 0, 0]
    f = O.kinematic_ft(1e-3, m, [0, 0, 0], quat_L=qx)
    np.testing.assert_allclose(f[:3] / np.linalg.norm(f[:3]), [0, -1, 0], atol=1e-7)
    # zero depth -> all zero (Q5)
    assert not O.kinematic_ft(0.0, m, xj, vO=[1, 1, 1], wO=[1, 1, 1]).any()


# ------------------------------------------------------------------ P10 Schmitt
def test_schmitt_sequence():
    seq = [0.0, 3e-4, 6e-4, 3e-4, 1e-4, 3e-4]
    for eta_off, ref in ((2e-4, [0, 0, 1, 1, 0, 0]), (5e-4, [0, 0, 1, 0, 0, 0])):
        o = scene([one_patch()], 1, physics=dict(eta_on=5e-4, eta_off=eta_off))
        got = []
        for d in seq:
            out = o.step(inputs(link_pos=(0, 0, -(0.030 + R_TAX - d))))
            assert out["depth"][0, 0] == pytest.approx(d, abs=2e-9)
            got.append(int(out["contact"][0, 0]))
        assert got == ref
    o.reset()
    assert int(o.step(inputs(link_pos=(0, 0, -(0.032 - 3e-4))))["contact"][0, 0]) == 0   # state cleared


# ------------------------------------------------------------------ P11 marker
def test_marker_single_source(golden):
    rs = golden["r_star"]
    assert rs == pytest.approx(1 / math.sqrt(2 * 8000.0), rel=1e-7)
    # one taxel at the patch centre, two markers at +-size_u/4 = +-r*; taxel 1 mm inside the sphere
    p = one_patch(1, 1, size_u=4 * rs, size_v=0.004, mnu=2, mnv=1)
    o = scene([p], 1)
    out = o.step(inputs(link_pos=(0, 0, -(0.030 - 1e-3))))
    assert out["aux_phi"][0, 0] == pytest.approx(-1e-3, abs=2e-9)
    mk = out["marker"][0]
    assert mk[1, 0] == pytest.approx(golden["marker_ut_1mm"], rel=1e-5)     # pushed away from the source (+x)
    assert mk[0, 0] == pytest.approx(-golden["marker_ut_1mm"], rel=1e-5)
    assert mk[0, 2] == pytest.approx(golden["marker_un_1mm"], rel=1e-5)     # bulge along +n
    assert abs(mk[0, 1]) < 1e-12
    # h = 0 (touching only through the probe radius) -> no marker motion although depth > 0
    out = o.step(inputs(link_pos=(0, 0, -0.031)))
    assert out["depth"][0, 0] > 0 and not out["marker"].any()
    # c = 0: in-plane far field decays like 1/r.  41 x 1 taxels at 2 mm pitch (eps = 2 mm, Q15); a 1.5 mm
    # ball indents only the centre taxel by 0.5 mm; markers sit at +-10.25 mm and +-30.75 mm from it.
    o = scene([one_patch(41, 1, size_u=0.082, size_v=0.004, mnu=4, mnv=1)], 41, physics=dict(c_e=0.0),
              geom=("sphere", [0.0015]))
    out = o.step(inputs(link_pos=(0, 0, -0.001)))
    assert (out["aux_phi"][0] < 0).sum() == 1 and out["aux_phi"][0, 20] == pytest.approx(-5e-4, abs=1e-9)
    mk = out["marker"][0]
    r1, r2, eps, h = 0.01025, 0.03075, 0.002, 5e-4
    ref = lambda r: 100.0 * h * r * (1 / (r * r + eps * eps)) / (1 / (2 * eps))      # s_d r h rho / rho_bar
    assert mk[2, 0] == pytest.approx(ref(r1), rel=1e-5) and mk[3, 0] == pytest.approx(ref(r2), rel=1e-5)
    assert mk[1, 0] == pytest.approx(-ref(r1), rel=1e-5)
    assert mk[2, 0] / mk[3, 0] == pytest.approx(3.0, rel=0.04)                        # ~ r2 / r1


# ------------------------------------------------------------------ P12 march
def test_march_plane_closed_form(golden):
    N, hv, R = 64, 0.002, 0.020
    n = np.array([0.0, 0.0, 1.0])
    g = _affine_grid(N, hv, n, 0.0).astype(np.float32)                      # plane z = 0, phi = z
    D = 0.010
    for th_deg, key in ((0, None), (30, "march_30deg_mm"), (60, "march_60deg_mm"), (75, None)):
        th = math.radians(th_deg)
        a = np.array([math.sin(th), 0.0, -math.cos(th)])
        P = O.march("grid", [0], [0.001, 0.002, D], a, R, 16, grid=g, voxel=hv)
        t_ref = min(D / math.cos(th) * (1 - (1 - math.cos(th)) ** 16), R)
        assert R - P == pytest.approx(t_ref, abs=2e-9)
        if key:
            assert (R - P) * 1e3 == pytest.approx(golden[key], abs=2e-6)
        if th_deg == 0:
            assert O.march("grid", [0], [0.001, 0.002, D], a, R, 1, grid=g, voxel=hv) == pytest.approx(R - D, abs=2e-9)
        if th_deg == 75:
            assert P == 0.0
    # intermediate iterates follow the geometric law
    th = math.radians(60)
    a = np.array([math.sin(th), 0.0, -math.cos(th)])
    for k in (1, 2, 5):
        P = O.march("grid", [0], [0, 0, D], a, R, k, grid=g, voxel=hv)
        assert R - P == pytest.approx(D / 0.5 * (1 - 0.5 ** k), abs=2e-9)


def test_march_sphere_and_limits():
    R = 0.020
    assert O.march("sphere", [0.03], [0, 0, -0.04], [0, 0, 1], R, 16) == pytest.approx(R - 0.010, abs=1e-15)
    assert O.march("sphere", [0.03], [0, 0, -0.04], [0, 0, 1], R, 1) == pytest.approx(R - 0.010, abs=1e-15)
    assert O.march("sphere", [0.03], [0, 0, -0.02], [0, 0, 1], R, 16) == R          # inside: t frozen at 0
    assert O.march("sphere", [0.03], [0, 0, -0.06], [0, 0, 1], R, 16) == 0.0        # phi >= R_prox
    assert O.march("sphere", [0.03], [0, 0, -0.04], [0, 0, -1], R, 16) == 0.0       # looking away


# ------------------------------------------------------------------ P13 hysteresis
def test_hysteresis_closed_forms(golden):
    base = dict(noise_enable=1, seed=1, sigma_rw_force=0.0, sigma_rw_torque=0.0, p_dead=0.0, chi=0.0)
    # Maxwell (Eq. 29-30), step 0 -> X
    o = scene([one_patch()], 1, physics=dict(use_velocity=0),
              noise=dict(base, hyst_mode="maxwell", beta=golden["maxwell_beta"], tau=golden["maxwell_tau"]))
    for k in range(4):
        out = o.step(inputs(link_pos=(0, 0, -0.031)))
        X = out["ft"][0, 0, 2]
        assert out["ft_noisy"][0, 0, 2] / X == pytest.approx(golden["maxwell_k%d" % k], rel=2e-7)
    # falling step: undershoot
    out = o.step(inputs(link_pos=(0, 0, -0.05)))
    assert out["ft"][0, 0, 2] == 0 and out["ft_noisy"][0, 0, 2] * X < 0
    # asymmetric first-order (D3): load with 0.8, unload with 0.5
    o = scene([one_patch()], 1, physics=dict(use_velocity=0),
              noise=dict(base, hyst_mode="asym", alpha_load=0.8, alpha_unload=0.5))
    for k in range(1, 5):
        out = o.step(inputs(link_pos=(0, 0, -0.031)))
        assert out["ft_noisy"][0, 0, 2] / out["ft"][0, 0, 2] == pytest.approx(1 - 0.2 ** k, rel=1e-7)    # alpha_load stored as fp32
    Y = out["ft_noisy"][0, 0, 2]
    for k in range(1, 4):
        out = o.step(inputs(link_pos=(0, 0, -0.05)))
        assert out["ft_noisy"][0, 0, 2] == pytest.approx(Y * 0.5 ** k, rel=1e-7)


# ------------------------------------------------------------------ P14 crosstalk
def test_crosstalk_invariants():
    noise = dict(noise_enable=1, seed=1, sigma_rw_force=0.0, sigma_rw_torque=0.0, p_dead=0.0, chi=0.05, hyst_mode="off")
    # impulse: a 3 mm ball touches only the centre taxel of a 5 x 5 patch (4 mm pitch)
    o = scene([one_patch(5, 5, 0.020, 0.020)], 25, noise=noise, geom=("sphere", [0.003]))
    out = o.step(inputs(link_pos=(0, 0, -0.0045)))
    ft, fn = out["ft"][0], out["ft_noisy"][0]
    assert (np.abs(ft).max(1) > 0).sum() == 1 and np.abs(ft[12]).max() > 0
    np.testing.assert_allclose(fn[12], 0.95 * ft[12], rtol=1e-8)       # chi stored as fp32 0.05f
    for k in (7, 11, 13, 17):
        np.testing.assert_allclose(fn[k], 0.0125 * ft[12], rtol=1e-7)
    assert not fn[[6, 8, 16, 18, 0, 24]].any()
    # patch-sum preservation on a generic field, incl. edges and corners; several patches
    w = W.config(2, n_envs=8)
    o = O.Oracle(w.patches, w.T, w.L, 1, np.arange(8), physics=w.physics, noise=noise)
    o.set_geometry(w.types, w.params)
    out = o.step(w.inputs(0))
    lay = o.layout()
    assert np.abs(out["ft"]).sum() > 0
    for p in range(16):
        sel = lay["patch"] == p
        np.testing.assert_allclose(out["ft_noisy"][:, sel].sum(1), out["ft"][:, sel].sum(1), rtol=1e-10, atol=1e-14)
    assert np.abs(out["ft_noisy"] - out["ft"]).max() > 1e-4
    # constant field is a fixed point: flat plane under a patch with use_velocity = 0
    N, hv = 32, 0.002
    g = _affine_grid(N, hv, np.array([0, 0, -1.0]), 0.0).astype(np.float32)   # solid above z = 0 ... phi = -z
    o = scene([one_patch(4, 3, 0.020, 0.015)], 12, physics=dict(use_velocity=0), noise=noise, geom=("grid", [0]),
              bank=g[None], voxel=hv)
    out = o.step(inputs(link_pos=(0, 0, -0.001), link_quat=(1, 0, 0, 0)))
    assert np.ptp(out["ft"][0, :, 2]) < 1e-12 and abs(out["ft"][0, 0, 2]) > 0.1
    np.testing.assert_allclose(out["ft_noisy"][0, :, 2], out["ft"][0, :, 2], rtol=1e-12)


# ------------------------------------------------------------------ P15 drift, P16 dead
def test_drift_random_walk_moments():
    noise = dict(noise_enable=1, seed=1234, sigma_rw_force=1e-3, sigma_rw_torque=1e-5, p_dead=0.0, chi=0.0,
                 hyst_mode="off")
    E = 256
    o = scene([one_patch(8, 8, 0.02, 0.02)], 64, E=E, noise=noise)
    o.threads = 4
    far = inputs(E=E, link_pos=(0, 0, -0.5))
    prev = None
    for n in range(1, 26):
        out = o.step(far)["ft_noisy"]
        if n == 1:
            first = out.copy()
        prev = out
    assert not o.step(far)["ft"].any()
    assert abs(first[..., :3].std() / 1e-3 - 1) < 0.02 and abs(first[..., 3:].std() / 1e-5 - 1) < 0.02
    assert abs(prev[..., :3].var() / (25 * 1e-6) - 1) < 0.05                 # variance n sigma^2
    assert abs(prev[..., :3].mean()) < 4 * 5e-3 / math.sqrt(prev[..., :3].size)
    # the six channels and neighbouring taxels / envs are independent draws
    c = np.corrcoef(first.reshape(-1, 6).T)
    assert np.abs(c - np.eye(6)).max() < 0.05
    assert abs(np.corrcoef(first[:, :-1, 0].ravel(), first[:, 1:, 0].ravel())[0, 1]) < 0.05
    assert abs(np.corrcoef(first[:-1, :, 0].ravel(), first[1:, :, 0].ravel())[0, 1]) < 0.05
    # keyed by the GLOBAL env id: a context over envs {5, 9} reproduces rows 5 and 9
    o2 = O.Oracle([one_patch(8, 8, 0.02, 0.02)], 64, 1, 1, np.array([5, 9]), noise=noise)
    o2.set_geometry(np.ones((2, 1), np.int32), np.full((2, 1, 4), 0.03, np.float32))
    sub = o2.step({k: v[:2] for k, v in far.items()})["ft_noisy"]
    np.testing.assert_array_equal(sub, first[[5, 9]])


def test_dead_taxels():
    noise = dict(noise_enable=1, seed=77, sigma_rw_force=1e-3, sigma_rw_torque=1e-5, p_dead=0.02, chi=0.05,
                 hyst_mode="asym", alpha_load=0.8, alpha_unload=0.5)
    w = W.config(4, n_envs=32)
    o = O.Oracle(w.patches, w.T, w.L, 1, np.arange(32), physics=w.physics, noise=noise)
    o.set_geometry(w.types, w.params, w.bank, w.voxel)
    masks = []
    for s in range(3):
        out = o.step(w.inputs(s))
        dead = out["dead"].astype(bool)
        masks.append(dead)
        assert not out["ft_noisy"][dead].any() and not out["contact"][dead].any()
        assert np.abs(out["ft_noisy"][~dead]).min() > 0                       # live taxels carry drift
    assert (masks[0] == masks[1]).all() and (masks[1] == masks[2]).all()
    frac, n = masks[0].mean(), masks[0].size
    assert abs(frac - 0.02) < 3 * math.sqrt(0.02 * 0.98 / n)
    o.reset()
    m2 = o.step(w.inputs(0))["dead"].astype(bool)
    assert (m2 != masks[0]).any() and abs(m2.mean() - 0.02) < 3 * math.sqrt(0.02 * 0.98 / n)
    # masked reset: only env 3 changes
    keep = m2.copy()
    mask = np.zeros(32, np.uint8); mask[3] = 1
    o.reset(mask)
    m3 = o.step(w.inputs(0))["dead"].astype(bool)
    assert (m3[np.arange(32) != 3] == keep[np.arange(32) != 3]).all() and (m3[3] != keep[3]).any()


# ------------------------------------------------------------------ P19-P22 remaining knobs of Eq. 25-28
def _contact_scene(noise, E=64, nu=8, nv=8):
    """One 8x8 patch pressed 1 mm into the r = 30 mm sphere (centre taxels touch), clean ft != 0."""
    o = scene([one_patch(nu, nv, 0.02, 0.02)], nu * nv, E=E, noise=dict(dict(noise_enable=1, seed=99, hyst_mode="off"), **noise))
    o.threads = 4
    return o, inputs(E=E, link_pos=(0, 0, -0.031), link_quat=(1, 0, 0, 0))


def test_bias_and_white_noise_eq25():
    # Eq. 25 with drift off: ft_noisy = ft + b + n_t, n_t ~ N(0, sigma^2), fresh every step
    o, x = _contact_scene(dict(bias_force=0.25, bias_torque=-0.003, sigma_white_force=2e-3, sigma_white_torque=1e-5))
    a, b = o.step(x), o.step(x)
    clean = a["ft"]
    assert np.abs(clean).max() > 0.01                                        # the scene really touches
    ra, rb = a["ft_noisy"] - clean, b["ft_noisy"] - clean
    assert abs(ra[..., :3].mean() - 0.25) < 4 * 2e-3 / math.sqrt(ra[..., :3].size)
    assert abs(ra[..., 3:].mean() + 0.003) < 4 * 1e-5 / math.sqrt(ra[..., 3:].size)
    assert abs(ra[..., :3].std() / 2e-3 - 1) < 0.03 and abs(ra[..., 3:].std() / 1e-5 - 1) < 0.03
    assert abs(np.corrcoef(ra[..., 0].ravel(), rb[..., 0].ravel())[0, 1]) < 0.05    # white: no memory
    # with sigma = 0 the shift is exactly the bias
    o2, _ = _contact_scene(dict(bias_force=0.25, bias_torque=-0.003))
    r2 = o2.step(x)
    np.testing.assert_allclose(r2["ft_noisy"][..., :3] - r2["ft"][..., :3], 0.25, rtol=0, atol=1e-7)
    np.testing.assert_allclose(r2["ft_noisy"][..., 3:] - r2["ft"][..., 3:], -0.003, rtol=0, atol=1e-9)
    # white noise and drift use different Philox streams: with both on, the step-1 residual has variance s_w^2 + s_rw^2
    o3, _ = _contact_scene(dict(sigma_white_force=2e-3, sigma_rw_force=1e-3, sigma_white_torque=0.0, sigma_rw_torque=0.0))
    r3 = o3.step(x)
    res = (r3["ft_noisy"] - r3["ft"])[..., :3]
    assert abs(res.var() / (4e-6 + 1e-6) - 1) < 0.05


def test_quantisation_eq25():
    # quantize(y, q) = q rint(y / q): every readout is a multiple of q, within q/2 of the unquantised one
    q_f, q_t = 0.01, 1e-4
    o, x = _contact_scene(dict(quant_force=q_f, quant_torque=q_t))
    ref, _ = _contact_scene(dict())
    yq, y = o.step(x), ref.step(x)["ft_noisy"]
    out = yq["ft_noisy"]
    kf, kt = out[..., :3] / np.float32(q_f), out[..., 3:] / np.float32(q_t)
    assert np.abs(kf - np.rint(kf)).max() < 1e-4 and np.abs(kt - np.rint(kt)).max() < 1e-4
    assert np.abs(out[..., :3] - y[..., :3]).max() <= 0.5 * q_f * (1 + 1e-5)
    assert np.abs(out[..., 3:] - y[..., 3:]).max() <= 0.5 * q_t * (1 + 1e-5)
    assert len(np.unique(np.rint(kf))) > 3                                   # several levels are hit
    # hand values, round half to even: 0.025 -> 0.02, 0.035 -> 0.04 (in fp32: 0.025f/0.01f = 2.5 exactly?  use bias to place y)
    for b, want in ((0.0249, 0.02), (0.0251, 0.03), (-0.0151, -0.02)):
        o2 = scene([one_patch()], 1, noise=dict(noise_enable=1, seed=1, hyst_mode="off", bias_force=b, quant_force=0.01))
        r = o2.step(inputs(link_pos=(0, 0, -0.5)))["ft_noisy"][0, 0, 0]
        assert r == pytest.approx(want, abs=1e-7)
    # the comparator aid reports the distance to the nearest rounding boundary
    assert "aux_quant" in yq and np.isfinite(yq["aux_quant"]).all() and (yq["aux_quant"] >= 0).all()
    assert yq["aux_quant"][..., :3].max() <= 0.5 * q_f * (1 + 1e-5)


def test_gain_eq27():
    # gamma_bj ~ U[0.8, 1.2] once per episode: ft_noisy = gamma ft exactly, the same every step, new after reset
    o, x = _contact_scene(dict(gain_min=0.8, gain_max=1.2))
    a, b = o.step(x), o.step(x)
    touch = np.abs(a["ft"][..., 2]) > 1e-3
    g1 = a["ft_noisy"][..., 2][touch] / a["ft"][..., 2][touch]
    g2 = b["ft_noisy"][..., 2][touch] / b["ft"][..., 2][touch]
    assert g1.min() >= 0.8 and g1.max() <= 1.2 and g1.max() - g1.min() > 0.3
    np.testing.assert_allclose(g1, g2, rtol=1e-12)
    assert abs(g1.mean() - 1.0) < 4 * (0.4 / math.sqrt(12)) / math.sqrt(g1.size)
    assert abs(g1.std() / (0.4 / math.sqrt(12)) - 1) < 0.1                   # uniform, not Gaussian: sd = width / sqrt(12)
    # all six channels of a taxel share the gain
    gx = a["ft_noisy"][..., 4][touch] / a["ft"][..., 4][touch]
    np.testing.assert_allclose(gx, g1, rtol=1e-9)
    o.reset()
    g3 = o.step(x)
    g3 = g3["ft_noisy"][..., 2][touch] / g3["ft"][..., 2][touch]
    assert np.abs(g3 - g1).max() > 0.1
    # gain enters BEFORE the hysteresis (R1): with ASYM loading from rest, y_1 = alpha_load * gamma * x
    o2, _ = _contact_scene(dict(gain_min=0.8, gain_max=1.2, hyst_mode="asym", alpha_load=0.8, alpha_unload=0.5))
    r = o2.step(x)
    np.testing.assert_allclose(r["ft_noisy"][..., 2][touch] / r["ft"][..., 2][touch], float(np.float32(0.8)) * g1, rtol=1e-6)


def test_stuck_value_eq28():
    # dead taxels read z_bj ~ U[l, u] for the whole episode; l = u = 0 is D5
    nz = dict(p_dead=0.2, stuck_min_force=0.5, stuck_max_force=1.5, stuck_min_torque=-0.02, stuck_max_torque=-0.01,
              sigma_rw_force=1e-3, sigma_rw_torque=1e-5)
    o, x = _contact_scene(nz)
    a, b = o.step(x), o.step(x)
    dead = a["dead"].astype(bool)
    assert 0.15 < dead.mean() < 0.25
    za = a["ft_noisy"][dead]
    assert za[:, :3].min() >= 0.5 and za[:, :3].max() <= 1.5 and za[:, 3:].min() >= -0.02 and za[:, 3:].max() <= -0.01
    np.testing.assert_array_equal(za, b["ft_noisy"][dead])                   # stuck: identical every step
    assert abs(za[:, :3].mean() - 1.0) < 0.05 and za[:, 0].std() > 0.2       # spread over the interval
    assert np.abs(np.corrcoef(za[:, 0], za[:, 1])[0, 1]) < 0.1               # channels drawn independently
    assert (a["ft_noisy"][~dead] != b["ft_noisy"][~dead]).any()              # live taxels keep drifting
    o.reset()
    c = o.step(x)
    d2 = c["dead"].astype(bool)
    both = dead & d2
    assert both.any() and (c["ft_noisy"][both] != a["ft_noisy"][both]).any()  # re-drawn at reset


def test_radius_noise_eq26():
    # P24, Eq. 26 (R8): the noisy readout senses with R~_j = max(0, R_j + eps_j), eps_j ~ U[-rho, rho] per
    # (env, taxel, episode); with zero velocities Eq. 10 gives |f| = k_n d^alpha, so d~ can be read back.
    rho, k_n, alpha = float(np.float32(5e-4)), 500.0, float(np.float32(1.2))   # the fp32 images the oracle holds
    o, x = _contact_scene(dict(radius_noise=rho), E=256)
    ref, _ = _contact_scene(dict(), E=256)
    a, b, c0 = o.step(x), o.step(x), ref.step(x)
    for k in ("depth", "ft", "contact", "prox"):                               # clean outputs keep R_j
        np.testing.assert_array_equal(a[k], c0[k])
    phi, d = a["aux_phi"], a["depth"]
    fn = np.linalg.norm(a["ft_noisy"][..., :3], axis=-1)
    dt = (fn / k_n) ** (1.0 / alpha)
    sure = (R_TAX - rho - phi) > 1e-9                                          # touching under every eps
    assert sure.sum() > 2000
    eps = dt[sure] - d[sure]
    assert eps.min() >= -rho * (1 + 1e-6) and eps.max() <= rho * (1 + 1e-6)
    assert abs(eps.mean()) < 4 * rho / math.sqrt(3 * eps.size)                 # U[-rho, rho]: mean 0, var rho^2/3
    assert abs(eps.var() / (rho * rho / 3) - 1) < 0.08
    assert eps.min() < -0.95 * rho and eps.max() > 0.95 * rho
    never = (R_TAX + rho - phi) < -1e-9                                        # out of reach under every eps
    assert never.any() and (a["ft_noisy"][never] == 0).all()
    maybe = ~sure & ~never                                                     # contact only appears / vanishes here
    gained, lost = (fn > 0) & (d == 0), (fn == 0) & (d > 0)
    assert gained.any() and lost.any() and not (gained & ~maybe).any() and not (lost & ~maybe).any()
    # same contact normal: f~ is parallel to f, torque = x_j x f~ keeps the same lever arm
    both = sure & (d > 0)
    f, g = a["ft"][both], a["ft_noisy"][both]
    assert np.abs(np.cross(f[:, :3], g[:, :3])).max() < 1e-9 * np.abs(f[:, :3]).max() * np.abs(g[:, :3]).max() + 1e-15
    np.testing.assert_allclose(g[:, 3:] * np.linalg.norm(f[:, :3], axis=-1)[:, None],
                               f[:, 3:] * np.linalg.norm(g[:, :3], axis=-1)[:, None], rtol=1e-9, atol=1e-15)
    np.testing.assert_array_equal(a["ft_noisy"], b["ft_noisy"])                # fixed for the episode
    # the draw itself: stream 8, n = 0, word 0 of the (env, taxel, episode) counter
    e, j = np.argwhere(sure)[7]
    u = O.uniform(int(O.philox((e, j, 0, (0 << 4) | 8), (99, 0))[0]))
    assert abs((dt[e, j] - d[e, j]) - (-rho + 2 * rho * u)) < 1e-12
    np.testing.assert_allclose(a["aux_rgate"][e, j], abs(float(np.float32(R_TAX)) - rho + 2 * rho * u - phi[e, j]), rtol=0, atol=1e-12)
    o.reset()
    c = o.step(x)
    assert (c["ft_noisy"][sure][:, 2] != a["ft_noisy"][sure][:, 2]).mean() > 0.99          # re-drawn at reset
    # the clamp: rho = 10 R leaves R~ = 0 for ~45 % of the taxels; those read [0 - phi]_+
    big, xb = _contact_scene(dict(radius_noise=10 * R_TAX), E=64)
    r = big.step(xb)
    fz = np.linalg.norm(r["ft_noisy"][..., :3], axis=-1)
    zero = fz == 0
    assert 0.35 < zero.mean() < 0.6 and (r["aux_phi"] > 0).all()               # nothing penetrates: clamped ones read 0
    assert ((fz / k_n) ** (1 / alpha) <= 11 * R_TAX).all()


def _moving_inputs(E, steps):
    """The patch of _contact_scene pressed by a depth that changes every step (and differs per env)."""
    out = []
    for t in range(steps):
        z = -0.0305 - 0.0004 * np.sin(0.9 * t + 0.3 * np.arange(E))
        d = inputs(E=E, link_quat=(1, 0, 0, 0))
        d["link_pos"][:, 0, 2] = z
        out.append(d)
    return out


def test_read_delay_eq25():
    # P25, Eq. 25 (R9): quantize(y_{t - Delta} + b + n_t + d_t, q): the delayed term is the post-crosstalk signal, the
    # additive terms are of the current step.  Pinned by shifting an undelayed run of the same scene.
    E, S, D = 8, 14, 3
    xs = _moving_inputs(E, S)
    base = dict(hyst_mode="asym", alpha_load=0.8, alpha_unload=0.5, chi=0.2)
    ref, _ = _contact_scene(base, E=E)
    c = [ref.step(x)["ft_noisy"] for x in xs]                                 # no additive terms: y_t = c_t
    assert max(np.abs(c[t + 1] - c[t]).max() for t in range(S - 1)) > 1e-3    # the signal really moves
    dly, _ = _contact_scene(dict(base, read_delay=D), E=E)
    for t, x in enumerate(xs):
        y = dly.step(x)["ft_noisy"]
        np.testing.assert_array_equal(y, c[t - D] if t >= D else np.zeros_like(y))
        if t == 8:                                                             # a reset empties the pipe
            dly.reset()
            ref2, _ = _contact_scene(base, E=E)
            c2 = [ref2.step(x2)["ft_noisy"] for x2 in xs[9:]]
            for u, x2 in enumerate(xs[9:]):
                y2 = dly.step(x2)["ft_noisy"]
                np.testing.assert_array_equal(y2, c2[u - D] if u >= D else np.zeros_like(y2))
            break
    # drift, bias and white noise are NOT delayed: y_delay[t] - y_nodelay[t] = c[t - D] - c[t] with the same seed
    add = dict(base, sigma_rw_force=1e-3, sigma_rw_torque=1e-5, bias_force=0.05, sigma_white_force=1e-3)
    a0, _ = _contact_scene(add, E=E)
    a1, _ = _contact_scene(dict(add, read_delay=D), E=E)
    for t, x in enumerate(xs):
        y0, y1 = a0.step(x)["ft_noisy"], a1.step(x)["ft_noisy"]
        want = (c[t - D] if t >= D else 0.0) - c[t]
        np.testing.assert_allclose(y1 - y0, want, rtol=0, atol=1e-12)
    # jitter: one Delta_n in [D - J, D + J] per (env, step), shared by all taxels, every value reached, about uniform
    J, E2, S2 = 2, 64, 40
    xs2 = _moving_inputs(E2, S2)
    r2, _ = _contact_scene(base, E=E2)
    c2 = [r2.step(x)["ft_noisy"] for x in xs2]
    jit, _ = _contact_scene(dict(base, read_delay=D, read_jitter=J), E=E2)
    counts = np.zeros(2 * J + 1, int)
    for t, x in enumerate(xs2):
        y = jit.step(x)["ft_noisy"]
        if t < D + J:
            continue
        for e in range(E2):
            hits = [k for k in range(-J, J + 1) if np.array_equal(y[e], c2[t - D - k][e])]
            assert len(hits) == 1, (t, e, hits)
            counts[hits[0] + J] += 1
    assert counts.min() > 0.7 * counts.sum() / (2 * J + 1), counts
    # the draw itself: stream 9, taxel counter 0xffffffff, step n; k = (((w >> 9) * (2J + 1)) >> 23) - J
    w0 = int(O.philox((5, 0xffffffff, 20, (0 << 4) | 9), (99, 0))[0])
    k = (((w0 >> 9) * (2 * J + 1)) >> 23) - J
    jit2, _ = _contact_scene(dict(base, read_delay=D, read_jitter=J), E=E2)
    for t in range(21):
        y = jit2.step(xs2[t])["ft_noisy"]
    np.testing.assert_array_equal(y[5], c2[20 - D - k][5])
    # jitter larger than the delay clamps at zero delay
    z, _ = _contact_scene(dict(base, read_delay=0, read_jitter=1), E=E2)
    for t, x in enumerate(xs2[:12]):
        y = z.step(x)["ft_noisy"]
        for e in range(E2):
            assert np.array_equal(y[e], c2[t][e]) or (np.array_equal(y[e], c2[t - 1][e]) if t >= 1 else not y[e].any())


def test_gaussian_crosstalk_eq11_vs_scipy():
    # Eq. 11 / 31 (R7): z~ = (1 - chi) z + chi (G_sigma * z); pinned against scipy's zero-padded 2-D convolution of the
    # oracle's own clean ft field with an L1-normalised separable Gaussian (a library routine, not the oracle's loop)
    from scipy.signal import convolve2d
    for nu, nv, sigma, chi in ((8, 8, 0.8, 0.3), (6, 8, 1.2, 0.05), (5, 8, 0.5, 1.0)):
        o, x = _contact_scene(dict(chi=chi, xtalk_sigma=sigma), E=2, nu=nu, nv=nv)
        out = o.step(x)
        ft, got = out["ft"], out["ft_noisy"]
        assert (np.abs(ft[..., 2]) > 1e-3).sum() > 4 and (ft[..., 2] == 0).sum() > 4      # a real, non-constant field
        r = int(math.ceil(3 * np.float32(sigma)))
        g = np.exp(-np.arange(-r, r + 1) ** 2 / (2.0 * float(np.float32(sigma)) ** 2))
        g /= g.sum()
        G = np.outer(g, g)
        assert abs(G.sum() - 1) < 1e-12
        for e in range(2):
            for c in range(6):
                z = ft[e, :, c].reshape(nv, nu)                                        # u fastest
                want = (1 - float(np.float32(chi))) * z + float(np.float32(chi)) * convolve2d(z, G, mode="same", boundary="fill")
                np.testing.assert_allclose(got[e, :, c].reshape(nv, nu), want, rtol=2e-6, atol=1e-9)
    # sigma -> 0: the kernel collapses to the identity (r = 1, g[+-1] = exp(-50))
    o, x = _contact_scene(dict(chi=0.5, xtalk_sigma=0.1), E=1)
    out = o.step(x)
    np.testing.assert_allclose(out["ft_noisy"], out["ft"], rtol=1e-6, atol=1e-12)
    # interior impulse: a single loaded taxel spreads as chi * G around it and keeps (1 - chi) + chi G[0,0] itself
    o = scene([one_patch(8, 8, 0.0008, 0.0008, radius=1e-4)], 64, noise=dict(noise_enable=1, seed=3, hyst_mode="off", chi=0.4, xtalk_sigma=0.7))
    # tiny patch (0.1 mm pitch) under a box face: uniform depth -> constant field; interior taxels stay fixed
    o.set_geometry(np.full((1, 1), O.GEOM["box"], np.int32), np.array([[[0.05, 0.05, 0.05, 0]]], np.float32))
    out = o.step(inputs(link_pos=(0, 0, -0.05005)))
    f = out["ft"][0, :, 2].reshape(8, 8)
    assert np.ptp(f) < 1e-9 * abs(f).max() and abs(f).max() > 0
    n = out["ft_noisy"][0, :, 2].reshape(8, 8)
    rr = int(math.ceil(3 * 0.7))
    np.testing.assert_allclose(n[rr:-rr, rr:-rr], f[rr:-rr, rr:-rr], rtol=1e-6)     # constants are a fixed point away from the border
    assert abs(n[0, 0]) < abs(f[0, 0])                                             # zero padding loses mass at the border


# ------------------------------------------------------------------ P8, P17 whole path
def test_no_contact_and_fillers():
    w = W.config(2, n_envs=4)
    o = O.Oracle(w.patches, w.T, w.L, 1, np.arange(4), physics=w.physics)
    o.set_geometry(w.types, w.params)
    inp = w.inputs(0)
    inp["obj_pos"] = inp["obj_pos"] + np.float32(1.0)                          # object 1.7 m away
    out = o.step(inp)
    for k in ("contact", "depth", "ft", "marker", "prox"):
        assert not out[k].any()
    out = o.step(w.inputs(0))
    lay = o.layout()
    fill = lay["radius"] == 0
    assert fill.sum() == 8 and (lay["patch"][fill] == -1).all()                # Q18: 192 active + 8 fillers
    for k in ("contact", "depth", "ft", "prox"):
        assert not out[k][:, fill].any() and out[k][:, ~fill].any()


def test_link_filter_makes_fillers():
    w = W.config(2, n_envs=2)
    mask = np.ones(16, np.uint8); mask[[3, 7]] = 0
    o = O.Oracle(w.patches, w.T, w.L, 1, np.arange(2), physics=w.physics, link_mask=mask)
    o.set_geometry(w.types, w.params)
    out = o.step(w.inputs(0))
    lay = o.layout()
    off = np.isin(lay["link"], [3, 7]) & (lay["patch"] >= 0)
    assert (lay["radius"][off] == 0).all() and off.sum() == 24
    assert not out["depth"][:, off].any() and not out["prox"][:, off].any()
    assert not out["marker"][:, np.isin(lay["marker_patch"], [3, 7])].any()


def _rigid(inp, q, t):
    from paper_2606_22332_b200.workloads import _qmul, _qrot
    q = np.asarray(q, np.float64)
    out = {}
    for b in ("link", "obj"):
        out[b + "_pos"] = _qrot(q, inp[b + "_pos"].astype(np.float64)) + t
        out[b + "_quat"] = _qmul(q, inp[b + "_quat"].astype(np.float64))
        out[b + "_linvel"] = _qrot(q, inp[b + "_linvel"].astype(np.float64))
        out[b + "_angvel"] = _qrot(q, inp[b + "_angvel"].astype(np.float64))
    return {k: v.astype(np.float32) for k, v in out.items()}


@pytest.mark.parametrize("cid", [2, 3])
def test_frame_invariance(cid):
    """one rigid transform applied to every pose (velocities rotated) leaves all outputs unchanged"""
    w = W.config(cid, n_envs=6)
    outs = []
    g = np.array([0.5, -0.5, 0.5, 0.5])
    for moved in (False, True):
        o = O.Oracle(w.patches, w.T, w.L, 1, np.arange(6), physics=w.physics)
        o.set_geometry(w.types, w.params, w.bank, w.voxel)
        inp = w.inputs(1)
        if moved:
            inp = _rigid(inp, g, np.array([0.02, -0.01, 0.015]))
        outs.append(o.step(inp))
    a, b = outs
    # inputs are re-rounded to fp32 after the transform: ~1e-8 m position noise, amplified by k_n alpha d^(alpha-1)
    face_ok = (a["aux_face"] > 1e-3) & (a["aux_boxgap"] > 1e-5) & (np.abs(a["depth"] - 5e-4) > 1e-6) & \
              (np.abs(R_TAX - a["aux_phi"]) > 1e-6)
    assert (a["contact"][face_ok] == b["contact"][face_ok]).all()
    np.testing.assert_allclose(b["depth"], a["depth"], atol=1e-7)
    np.testing.assert_allclose(b["prox"], a["prox"], atol=1e-6)
    np.testing.assert_allclose(b["marker"], a["marker"], atol=2e-5)
    np.testing.assert_allclose(b["ft"][face_ok], a["ft"][face_ok], rtol=1e-3, atol=1e-4)
    assert np.abs(a["ft"]).max() > 0.1 and np.abs(a["marker"]).max() > 0.01


def test_layout_grid_positions():
    p = dict(link=2, origin=(0.01, 0.0, 0.002), u_axis=(0, 1, 0), v_axis=(0, 0, 1), size_u=0.020, size_v=0.015,
             nu=4, nv=3, radius=R_TAX, marker_nu=2, marker_nv=2)
    o = O.Oracle([p], 14, 3, 1, np.arange(1))
    lay = o.layout()
    # Q19: cell-centred, u fastest: taxel (iu, iv) at origin + ((iu+.5)/nu-.5) size_u u + ((iv+.5)/nv-.5) size_v v
    np.testing.assert_allclose(lay["pos"][0], [0.01, -0.0075, 0.002 - 0.005], atol=1e-9)
    np.testing.assert_allclose(lay["pos"][1], [0.01, -0.0025, 0.002 - 0.005], atol=1e-9)
    np.testing.assert_allclose(lay["pos"][4], [0.01, -0.0075, 0.002], atol=1e-9)
    np.testing.assert_allclose(lay["nrm"][:12], np.tile([1.0, 0, 0], (12, 1)), atol=1e-12)   # u x v
    assert (lay["link"][:12] == 2).all() and (lay["radius"][12:] == 0).all()
    assert list(lay["nbr"][0]) == [-1, 1, -1, 4] and list(lay["nbr"][5]) == [4, 6, 1, 9]
    assert list(lay["nbr"][11]) == [10, -1, 7, -1]
    np.testing.assert_allclose(lay["marker_pos"][0], [0.01, -0.005, 0.002 - 0.00375], atol=1e-9)
    assert o.M == 4


def test_transform_eq1():
    """Eq. 1: q = p_L + R_L x_j, a = R_L n_j, with a rotated link and an off-centre taxel"""
    s = math.sqrt(0.5)
    p = dict(link=0, origin=(0.01, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=0.004, size_v=0.004, nu=1, nv=1,
             radius=R_TAX, marker_nu=0, marker_nv=0)
    o = scene([p], 1, geom=("sphere", [0.005]))
    # link rotated +90 deg about z: x_j = (0.01,0,0) -> world offset (0,0.01,0); normal stays +z
    pL = np.array([0.02, -0.03, 0.0])
    out = o.step(inputs(link_pos=pL, link_quat=(s, 0, 0, s), obj_pos=pL + [0, 0.01, 0.0065]))
    # taxel sits 6.5 mm below the ball centre: phi = 1.5 mm, depth 0.5 mm, march along +z hits after 1.5 mm
    assert out["aux_phi"][0, 0] == pytest.approx(0.0015, abs=3e-9)
    assert out["depth"][0, 0] == pytest.approx(0.0005, abs=3e-9)
    assert out["prox"][0, 0] == pytest.approx(0.020 - 0.0015, abs=3e-9)
    f = out["ft"][0, 0]
    assert f[2] < 0 and abs(f[0]) < 1e-7 and abs(f[1]) < 1e-7     # quaternion is fp32
    np.testing.assert_allclose(f[3:], np.cross([0.01, 0, 0], f[:3]), atol=1e-12)   # lever arm is x_j (link frame)
    # the wrong rotation sense would put the taxel at (0,-0.01,0): no contact there
    out = o.step(inputs(link_pos=pL, link_quat=(s, 0, 0, s), obj_pos=pL + [0, -0.01, 0.0065]))
    assert out["depth"][0, 0] == 0
