"""Seeded synthetic workloads shaped like the paper's (BASELINE.json configs 1-5; recipe in DESIGN.md).

This module serves BOTH the CUDA path and the oracle and holds none of the method's
arithmetic: it only draws scenes (patch descriptors, object parameters, poses, velocities,
star-surface voxel grids) with numpy.  It evaluates no signed-distance query, no force law,
no noise model.  Surfaces are located with each shape's *radial* function rho(u) (distance
from the object origin to its surface along a unit direction), which exists in closed form
because every shape used here is star-shaped about its origin.

The paper measures on Genesis scenes (pyramid of cubes, XHand1 / Sharpa hands)
that are not available here; these inputs stand in for them (hundreds to a thousand taxels
over 16-20 links, Table 11; up to 20,480 envs P:10).
"""
import math

import numpy as np

DT = 0.005          # 200 Hz physics
TAXEL_RADIUS = 2.0e-3   # Q1
T_PERIOD = 40       # trajectory period in steps (configs 4-5)

GEOM_SPHERE, GEOM_BOX, GEOM_CAPSULE, GEOM_GRID = 1, 2, 3, 4


# --------------------------------------------------------------------------- quaternions
def _qmul(a, b):
    aw, ax, ay, az = a[..., 0], a[..., 1], a[..., 2], a[..., 3]
    bw, bx, by, bz = b[..., 0], b[..., 1], b[..., 2], b[..., 3]
    return np.stack([aw * bw - ax * bx - ay * by - az * bz,
                     aw * bx + ax * bw + ay * bz - az * by,
                     aw * by - ax * bz + ay * bw + az * bx,
                     aw * bz + ax * by - ay * bx + az * bw], axis=-1)


def _qrot(q, v):
    """rotate v by unit quaternion q (w,x,y,z)"""
    w = q[..., :1]
    u = q[..., 1:]
    t = 2.0 * np.cross(u, v)
    return v + w * t + np.cross(u, t)


def _qnorm(q):
    return q / np.linalg.norm(q, axis=-1, keepdims=True)


def _rand_quat(rng, shape):
    return _qnorm(rng.standard_normal(shape + (4,)))


def _rand_dir(rng, shape):
    v = rng.standard_normal(shape + (3,))
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _axis_angle(axis, ang):
    h = 0.5 * ang[..., None]
    return np.concatenate([np.cos(h), np.sin(h) * axis], axis=-1)


def _rotvec_quat(rv):
    ang = np.linalg.norm(rv, axis=-1)
    safe = np.where(ang > 1e-300, ang, 1.0)
    axis = rv / safe[..., None]
    return _axis_angle(axis, ang)


def _align_z_to(d):
    """shortest-arc quaternion taking +z to unit vector d"""
    z = np.zeros_like(d)
    z[..., 2] = 1.0
    w = 1.0 + d[..., 2]
    xyz = np.cross(z, d)
    q = np.concatenate([w[..., None], xyz], axis=-1)
    bad = w < 1e-9
    q[bad] = np.array([0.0, 1.0, 0.0, 0.0])
    return _qnorm(q)


# --------------------------------------------------------------------------- shapes
def y32(xhat):
    """real spherical harmonic Y_3^2 on unit vectors: 1/4 sqrt(105/pi) (x^2-y^2) z"""
    c = 0.25 * math.sqrt(105.0 / math.pi)
    return c * (xhat[..., 0] ** 2 - xhat[..., 1] ** 2) * xhat[..., 2]


def star_radius(xhat, scale=1.0, rot=None):
    """r(theta,phi) = 40 mm (1 + 0.2 Y_3^2), optionally rotated (rot: 3x3, columns = body axes) and scaled"""
    if rot is not None:
        xhat = xhat @ rot          # rot^T xhat
    return 0.040 * scale * (1.0 + 0.2 * y32(xhat))


def star_grid(N, voxel, scale=1.0, rot=None):
    """f(x) = |x| - r(x/|x|) sampled on N^3 nodes, node i at (i - (N-1)/2) voxel; index [k,j,i], x fastest."""
    ax = (np.arange(N, dtype=np.float64) - 0.5 * (N - 1)) * voxel
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    P = np.stack([X, Y, Z], axis=-1)
    r = np.linalg.norm(P, axis=-1)
    xhat = P / np.where(r > 0, r, 1.0)[..., None]
    return (r - star_radius(xhat, scale, rot)).astype(np.float32)


def _radial(types, params, u, stars=None):
    """surface distance from the object origin along unit directions u [E,L,3] (object frame)"""
    E = types.shape[0]
    rho = np.zeros(u.shape[:-1])
    for e_sel, kind in ((types == GEOM_SPHERE, GEOM_SPHERE), (types == GEOM_BOX, GEOM_BOX),
                        (types == GEOM_CAPSULE, GEOM_CAPSULE), (types == GEOM_GRID, GEOM_GRID)):
        idx = np.nonzero(e_sel)[0]
        if idx.size == 0:
            continue
        uu = u[idx]
        p = params[idx].astype(np.float64)
        if kind == GEOM_SPHERE:
            rho[idx] = p[:, None, 0]
        elif kind == GEOM_BOX:
            with np.errstate(divide="ignore"):
                rho[idx] = np.min(p[:, None, :3] / np.abs(uu), axis=-1)
        elif kind == GEOM_CAPSULE:
            r, h = p[:, None, 0], p[:, None, 1]
            rad = np.sqrt(uu[..., 0] ** 2 + uu[..., 1] ** 2)
            with np.errstate(divide="ignore"):
                t_cyl = r / rad
            uc = np.abs(uu[..., 2]) * h
            t_cap = uc + np.sqrt(np.maximum(uc * uc - h * h + r * r, 0.0))
            rho[idx] = np.where(np.abs(t_cyl * uu[..., 2]) <= h, t_cyl, t_cap)
        else:
            for e in idx:
                s = stars[int(params[e, 0])]
                rho[e] = star_radius(u[e], s["scale"], s["rot"])
    assert E == rho.shape[0]
    return rho


# --------------------------------------------------------------------------- layouts
def _patch(link, nu, nv, size_u, size_v, markers):
    return dict(link=link, origin=(0.0, 0.0, 0.0), u_axis=(1.0, 0.0, 0.0), v_axis=(0.0, 1.0, 0.0),
                size_u=size_u, size_v=size_v, nu=nu, nv=nv, radius=TAXEL_RADIUS,
                marker_nu=markers, marker_nv=markers)


def _hand_patches(cid):
    if cid in (1, 2):      # 16 links x (4 x 3) on 20 x 15 mm (Q19)
        return [_patch(l, 4, 3, 0.020, 0.015, 0 if cid == 1 else 7) for l in range(16)]
    if cid == 3:           # 20 links x (5 x 5)
        return [_patch(l, 5, 5, 0.020, 0.020, 7) for l in range(20)]
    out = []               # Q20: 5 x (8x8) + 10 x (6x8) + 5 x (5x8), 2.5 mm pitch
    for l in range(20):
        nu = 8 if l < 5 else (6 if l < 15 else 5)
        out.append(_patch(l, nu, 8, 0.0025 * nu, 0.020, 7))
    return out


class Workload:
    """A scene family: static layout + geometry, and per-step pose/velocity inputs (all fp32)."""

    def __init__(self, cid, n_envs=None, seed=0, delta_range=(-0.003, 0.022)):
        assert cid in (1, 2, 3, 4, 5)
        full = {1: 4, 2: 4096, 3: 8192, 4: 16384, 5: 20480}[cid]
        self.cid, self.seed = cid, seed
        self.E = int(n_envs) if n_envs else full
        self.K = 1
        self.patches = _hand_patches(cid)
        self.L = len(self.patches)
        self.T = {1: 200, 2: 200, 3: 500, 4: 1000, 5: 1000}[cid]
        self.steps = {1: 10, 2: 10, 3: 10, 4: 100, 5: 200}[cid]
        self.delta_range = delta_range
        self.name = {1: "tiny", 2: "primitives", 3: "sdf", 4: "noise", 5: "stress"}[cid]
        self.physics = dict(mu=1.0, eta_on=5e-4, eta_off=5e-4 if cid <= 3 else 2e-4, r_prox=0.020, march_steps=16,
                            dt=DT)
        self.noise = None
        if cid >= 4:
            self.noise = dict(noise_enable=1, seed=0x5EED0000 + seed, sigma_rw_force=1e-3, sigma_rw_torque=1e-5,
                              hyst_mode="asym", alpha_load=0.8, alpha_unload=0.5, beta=0.5, tau=0.05, p_dead=0.02,
                              chi=0.05)
        self.outputs = ("contact", "depth", "ft") if cid == 1 else ("contact", "depth", "ft", "marker", "prox")
        if cid >= 4:
            self.outputs += ("ft_noisy", "dead")
        self._static()

    # ---- static scene: object types / parameters / grids, trajectory base
    def _static(self):
        rng = np.random.default_rng([self.seed, self.cid, 0])
        E, cid = self.E, self.cid
        self.bank, self.voxel, self.stars = None, 0.0, None
        types = np.zeros(E, np.int32)
        params = np.zeros((E, 4), np.float32)
        if cid == 1:
            types[:] = GEOM_SPHERE
            params[:, 0] = 0.030
        elif cid in (2, 5):
            if cid == 2:
                cls = rng.integers(0, 3, size=E)
                grid_id = np.zeros(E, np.int64)
            else:
                m = np.arange(E) % 16
                cls = np.where(m < 8, 3, np.where(m < 10, 0, np.where(m < 13, 1, 2)))
                grid_id = m
            r_s = rng.uniform(0.020, 0.040, size=E)
            b = rng.uniform(0.015, 0.035, size=(E, 3))
            hl = rng.uniform(0.020, 0.040, size=E)
            for e in range(E):
                if cls[e] == 0:
                    types[e] = GEOM_SPHERE; params[e, 0] = r_s[e]
                elif cls[e] == 1:
                    types[e] = GEOM_BOX; params[e, :3] = b[e]
                elif cls[e] == 2:
                    types[e] = GEOM_CAPSULE; params[e, 0] = 0.015; params[e, 1] = hl[e]
                else:
                    types[e] = GEOM_GRID; params[e, 0] = float(grid_id[e])
        elif cid == 3:
            types[:] = GEOM_GRID
        else:
            types[:] = GEOM_GRID
            params[:, 0] = rng.integers(0, 8, size=E).astype(np.float32)
        if cid >= 3:
            n_grids = 1 if cid == 3 else 8
            N = 96 if cid == 5 else 64
            self.voxel = 0.128 / N          # Q21: same 128 mm extent
            srng = np.random.default_rng([self.seed, 777, cid])
            self.stars = []
            for k in range(n_grids):
                if cid == 3:
                    self.stars.append(dict(scale=1.0, rot=None))
                else:
                    q = _rand_quat(srng, ())
                    rot = np.stack([_qrot(q, np.eye(3)[i]) for i in range(3)], axis=1)
                    self.stars.append(dict(scale=float(srng.uniform(0.85, 1.15)), rot=rot))
            self.bank = np.stack([star_grid(N, self.voxel, s["scale"], s["rot"]) for s in self.stars])
        self.types = types.reshape(E, 1)
        self.params = params.reshape(E, 1, 4)
        if cid >= 4:   # coherent trajectory: base pose + sinusoid (DESIGN.md input recipe)
            self._base = self._near_surface(rng)
            L = self.L
            self._v = dict(link_lin=rng.normal(0, 0.1, (E, L, 3)), link_ang=rng.normal(0, 0.5, (E, L, 3)),
                           obj_lin=rng.normal(0, 0.1, (E, 1, 3)), obj_ang=rng.normal(0, 0.5, (E, 1, 3)))

    # ---- near-surface recipe: link origins at signed radial offset delta from the surface
    def _near_surface(self, rng):
        E, L = self.E, self.L
        obj_pos = rng.uniform(-0.01, 0.01, (E, 1, 3))
        obj_quat = _rand_quat(rng, (E, 1))
        u = _rand_dir(rng, (E, L))
        rho = _radial(self.types[:, 0], self.params[:, 0], u, self.stars)
        delta = rng.uniform(self.delta_range[0], self.delta_range[1], (E, L))
        p_obj = (rho + delta)[..., None] * u                     # link origin, object frame
        q_align = _align_z_to(-u)                                # link +z towards the object
        roll = _axis_angle(np.broadcast_to(np.array([0.0, 0.0, 1.0]), (E, L, 3)), rng.uniform(0, 2 * np.pi, (E, L)))
        phi = rng.uniform(0, 2 * np.pi, (E, L))
        tilt_axis = np.stack([np.cos(phi), np.sin(phi), np.zeros_like(phi)], axis=-1)
        tilt = _axis_angle(tilt_axis, rng.normal(0, np.deg2rad(10.0), (E, L)))
        q_lo = _qmul(_qmul(q_align, roll), tilt)
        link_quat = _qnorm(_qmul(obj_quat, q_lo))
        link_pos = obj_pos + _qrot(obj_quat, p_obj)
        return dict(link_pos=link_pos, link_quat=link_quat, obj_pos=obj_pos, obj_quat=obj_quat)

    # ---- per-step inputs
    def inputs(self, step):
        E, L, cid = self.E, self.L, self.cid
        rng = np.random.default_rng([self.seed, cid, 1000 + step])
        if cid == 1:
            d = dict(link_pos=rng.uniform(-0.05, 0.05, (E, L, 3)), link_quat=_rand_quat(rng, (E, L)),
                     obj_pos=np.zeros((E, 1, 3)), obj_quat=np.tile(np.array([1.0, 0, 0, 0]), (E, 1, 1)),
                     link_linvel=rng.normal(0, 0.05, (E, L, 3)), link_angvel=rng.normal(0, 0.5, (E, L, 3)),
                     obj_linvel=rng.normal(0, 0.05, (E, 1, 3)), obj_angvel=rng.normal(0, 0.5, (E, 1, 3)))
        elif cid in (2, 3):
            d = self._near_surface(rng)
            d.update(link_linvel=rng.normal(0, 0.1, (E, L, 3)), link_angvel=rng.normal(0, 0.5, (E, L, 3)),
                     obj_linvel=rng.normal(0, 0.1, (E, 1, 3)), obj_angvel=rng.normal(0, 0.5, (E, 1, 3)))
        else:
            amp = DT * T_PERIOD / (2 * np.pi)
            s, c = math.sin(2 * np.pi * step / T_PERIOD), math.cos(2 * np.pi * step / T_PERIOD)
            b, v = self._base, self._v
            d = {}
            for body, lin, ang in (("link", "link_lin", "link_ang"), ("obj", "obj_lin", "obj_ang")):
                q = _qnorm(_qmul(b[body + "_quat"], _rotvec_quat(v[ang] * (amp * s))))
                d[body + "_pos"] = b[body + "_pos"] + v[lin] * (amp * s)
                d[body + "_quat"] = q
                d[body + "_linvel"] = v[lin] * c
                d[body + "_angvel"] = _qrot(q, v[ang]) * c
        return {k: np.ascontiguousarray(a, dtype=np.float32) for k, a in d.items()}

    def parity_envs(self):
        """env ids whose outputs the oracle recomputes at full size"""
        E, cid = self.E, self.cid
        if cid == 3:
            ids = np.arange(0, E, 16)
        elif cid == 4:
            ids = np.arange(0, E, 128)
        elif cid == 5:
            ids = np.array([1281 * k for k in range(16) if 1281 * k < E])
        else:
            ids = np.arange(E)
        return ids.astype(np.int64)

    def subset(self, inp, ids):
        return {k: a[ids] for k, a in inp.items()}


def star_point_cloud(n_points, scale=1.0, rot=None, seed=0):
    """n_points surface samples of the star r(u) = 40 mm (1 + 0.2 Y_3^2(u)) (scaled / rotated like star_grid), object
    frame, fp32: uniform random directions times the closed-form radius (the paper samples tracked links into surface
    point clouds at reset; N_pc = 5,000 P:267)."""
    rng = np.random.default_rng([seed, 4242, n_points])
    u = _rand_dir(rng, (n_points,))
    return (star_radius(u, scale, rot)[:, None] * u).astype(np.float32)


def point_cloud_bank(w, n_points=5000):
    """Tracked point clouds for a grid-object workload (configs 3-5): cloud k samples star k of the SDF bank; envs whose
    object is a primitive get cloud_id -1 (not tracked).  Returns (points [G, N, 3], cloud_id [E, 1])."""
    pts = np.stack([star_point_cloud(n_points, s["scale"], s["rot"], seed=k) for k, s in enumerate(w.stars)])
    cid = np.where(w.types[:, 0] == GEOM_GRID, w.params[:, 0, 0].astype(np.int32), -1).astype(np.int32)
    return pts, cid.reshape(-1, 1)


def cube_mesh(b):
    """12-triangle box with half-extents b (outward winding): (verts [8,3] fp32, tris [12,3] int32)."""
    b = np.asarray(b, np.float64)
    v = np.array([[sx, sy, sz] for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)], np.float64) * b
    quads = [(0, 1, 3, 2), (4, 6, 7, 5), (0, 4, 5, 1), (2, 3, 7, 6), (0, 2, 6, 4), (1, 5, 7, 3)]   # -x, +x, -y, +y, -z, +z
    tris = [t for a, b_, c, d in quads for t in ((a, b_, c), (a, c, d))]
    return v.astype(np.float32), np.asarray(tris, np.int32)


def star_mesh(level=3, scale=1.0, rot=None):
    """Triangle mesh of the star surface r(u) = 40 mm (1 + 0.2 Y_3^2(u)): an icosahedron subdivided `level` times
    (20 * 4^level triangles, outward winding), vertices pushed to the star radius.  Object frame, fp32."""
    t = (1.0 + math.sqrt(5.0)) / 2.0
    v = [(-1, t, 0), (1, t, 0), (-1, -t, 0), (1, -t, 0), (0, -1, t), (0, 1, t), (0, -1, -t), (0, 1, -t), (t, 0, -1), (t, 0, 1),
         (-t, 0, -1), (-t, 0, 1)]
    f = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11), (1, 5, 9), (5, 11, 4), (11, 10, 2), (10, 7, 6), (7, 1, 8),
         (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8), (3, 8, 9), (4, 9, 5), (2, 4, 11), (6, 2, 10), (8, 6, 7), (9, 8, 1)]
    v = [np.asarray(x, np.float64) / np.linalg.norm(x) for x in v]
    for _ in range(level):
        cache, nf = {}, []

        def mid(i, j):
            key = (min(i, j), max(i, j))
            if key not in cache:
                m = v[i] + v[j]
                v.append(m / np.linalg.norm(m))
                cache[key] = len(v) - 1
            return cache[key]
        for a, b, c in f:
            ab, bc, ca = mid(a, b), mid(b, c), mid(c, a)
            nf += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
        f = nf
    u = np.asarray(v)
    return (star_radius(u, scale, rot)[:, None] * u).astype(np.float32), np.asarray(f, np.int32)


def mesh_bank(w, level=3):
    """Triangle meshes for a grid-object workload (configs 3-5): mesh k triangulates star k of the SDF bank; envs whose
    object is a primitive get mesh_id -1.  Returns (list of (verts, tris), mesh_id [E, 1])."""
    meshes = [star_mesh(level, s["scale"], s["rot"]) for s in w.stars]
    mid = np.where(w.types[:, 0] == GEOM_GRID, w.params[:, 0, 0].astype(np.int32), -1).astype(np.int32)
    return meshes, mid.reshape(-1, 1)


def config(cid, n_envs=None, seed=0):
    return Workload(cid, n_envs=n_envs, seed=seed)
