"""ORACLE -- TEST INFRASTRUCTURE ONLY (see oracle.cpp header).

ctypes wrapper around liboracle.so.  Argument marshalling only; every formula lives in
oracle.cpp.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module; the product package never does.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "oracle.cpp")


def build(force=False):
    """g++ -O2 -fopenmp oracle.cpp -> liboracle.so (rebuilt when the source is newer)."""
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(_SRC):
        return _SO
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", _SRC, "-o", _SO]
    subprocess.run(cmd, check=True)
    return _SO


class OrcPatch(C.Structure):
    _fields_ = [("link", C.c_int32), ("origin", C.c_float * 3), ("u_axis", C.c_float * 3), ("v_axis", C.c_float * 3),
                ("size_u", C.c_float), ("size_v", C.c_float), ("nu", C.c_int32), ("nv", C.c_int32),
                ("radius", C.c_float), ("marker_nu", C.c_int32), ("marker_nv", C.c_int32)]


class OrcParams(C.Structure):
    _fields_ = [("k_n", C.c_float), ("c_n", C.c_float), ("alpha", C.c_float), ("k_t", C.c_float),
                ("k_omega", C.c_float), ("mu", C.c_float), ("eta_on", C.c_float), ("eta_off", C.c_float),
                ("use_velocity", C.c_int32),
                ("s_d", C.c_float), ("lambda_d", C.c_float), ("alpha_e", C.c_float), ("c_e", C.c_float),
                ("r_prox", C.c_float), ("march_steps", C.c_int32), ("dt", C.c_float),
                ("noise_enable", C.c_int32), ("seed_lo", C.c_uint32), ("seed_hi", C.c_uint32),
                ("sigma_rw_force", C.c_float), ("sigma_rw_torque", C.c_float), ("hyst_mode", C.c_int32),
                ("beta", C.c_float), ("tau", C.c_float), ("alpha_load", C.c_float), ("alpha_unload", C.c_float),
                ("p_dead", C.c_float), ("chi", C.c_float),
                ("sigma_white_force", C.c_float), ("sigma_white_torque", C.c_float),
                ("bias_force", C.c_float), ("bias_torque", C.c_float),
                ("quant_force", C.c_float), ("quant_torque", C.c_float),
                ("gain_min", C.c_float), ("gain_max", C.c_float),
                ("stuck_min_force", C.c_float), ("stuck_max_force", C.c_float),
                ("stuck_min_torque", C.c_float), ("stuck_max_torque", C.c_float), ("xtalk_sigma", C.c_float),
                ("radius_noise", C.c_float), ("read_delay", C.c_int32), ("read_jitter", C.c_int32),
                ("sn_sigma_white", C.c_float * 3), ("sn_sigma_rw", C.c_float * 3), ("sn_bias", C.c_float * 3),
                ("sn_quant", C.c_float * 3), ("sn_stuck_min", C.c_float * 3), ("sn_stuck_max", C.c_float * 3),
                ("pc_radius", C.c_float), ("pc_k", C.c_float), ("pc_ks", C.c_float), ("pc_density", C.c_float),
                ("shear_enable", C.c_int32), ("s_s", C.c_float), ("lambda_s", C.c_float), ("eta_enter", C.c_float),
                ("eta_exit", C.c_float)]

SN_CLASS = {"depth": 0, "prox": 1, "marker": 2}          # noisy scalar readouts (R10)
SN_KNOBS = ("sigma_white", "sigma_rw", "bias", "quant", "stuck_min", "stuck_max")


HYST = {"off": 0, "maxwell": 1, "asym": 2}
GEOM = {"none": 0, "sphere": 1, "box": 2, "capsule": 3, "grid": 4}

_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(OrcParams), C.POINTER(OrcPatch), C.c_int, C.c_int, C.c_void_p, C.c_int,
                                 C.c_void_p, C.c_int, C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_n_markers.argtypes = [C.c_void_p]
        L.orc_get_layout.argtypes = [C.c_void_p] + [C.c_void_p] * 9
        L.orc_set_geometry.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_float, C.c_void_p]
        L.orc_reset.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_step.argtypes = [C.c_void_p] + [C.c_void_p] * 19 + [C.c_int]
        L.orc_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_uniform.restype = C.c_double
        L.orc_uniform.argtypes = [C.c_uint32]
        L.orc_box_muller.argtypes = [C.c_uint32, C.c_uint32, C.c_void_p]
        L.orc_sdf_query.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_kinematic_ft.argtypes = [C.POINTER(OrcParams), C.c_double] + [C.c_void_p] * 10
        L.orc_march.restype = C.c_double
        L.orc_march.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_void_p, C.c_void_p,
                                C.c_double, C.c_int]
        L.orc_set_aux_quant.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_set_aux_rgate.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_set_aux_wingap.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_set_scalar_noisy.argtypes = [C.c_void_p] + [C.c_void_p] * 7
        L.orc_set_pointclouds.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_set_proxpc.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_set_meshes.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 5
        L.orc_set_raycast_out.argtypes = [C.c_void_p] + [C.c_void_p] * 3
        L.orc_closest_point_triangle.argtypes = [C.c_void_p] * 5
        L.orc_ray_triangle.restype = C.c_double
        L.orc_ray_triangle.argtypes = [C.c_void_p] * 5
        L.orc_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def make_params(physics=None, noise=None):
    """Defaults = paper constants (Eq. 10) with the DESIGN.md readings."""
    d = dict(k_n=500.0, c_n=1.0, alpha=1.2, k_t=2.0, k_omega=2.0, mu=1.0, eta_on=5e-4, eta_off=5e-4, use_velocity=1,
             s_d=100.0, lambda_d=8000.0, alpha_e=1.2, c_e=1.0, r_prox=0.020, march_steps=16, dt=0.005,
             noise_enable=0, seed=0, sigma_rw_force=0.0, sigma_rw_torque=0.0, hyst_mode=0, beta=0.0, tau=0.05,
             alpha_load=1.0, alpha_unload=1.0, p_dead=0.0, chi=0.0,
             sigma_white_force=0.0, sigma_white_torque=0.0, bias_force=0.0, bias_torque=0.0, quant_force=0.0,
             quant_torque=0.0, gain_min=1.0, gain_max=1.0, stuck_min_force=0.0, stuck_max_force=0.0,
             stuck_min_torque=0.0, stuck_max_torque=0.0, xtalk_sigma=0.0, radius_noise=0.0, read_delay=0, read_jitter=0,
             pc_radius=0.01, pc_k=300.0, pc_ks=10.0, pc_density=100.0,          # A.6 constants
             shear_enable=0, s_s=100.0, lambda_s=2000.0, eta_enter=1e-5, eta_exit=1e-4)   # A.7 shear constants
    sn = {}
    for src in (physics, noise):
        if src:
            for k, v in src.items():
                knob, _, cls = k.rpartition("_")
                if knob in SN_KNOBS and cls in SN_CLASS:     # e.g. sigma_white_depth, quant_marker
                    sn[(knob, cls)] = float(v)
                    continue
                if k not in d:
                    raise KeyError(k)
                d[k] = v
    seed = int(d.pop("seed"))
    hm = d["hyst_mode"]
    d["hyst_mode"] = HYST[hm] if isinstance(hm, str) else int(hm)
    p = OrcParams()
    for k, v in d.items():
        setattr(p, k, v)
    p.seed_lo = seed & 0xFFFFFFFF
    p.seed_hi = (seed >> 32) & 0xFFFFFFFF
    for (knob, cls), v in sn.items():
        getattr(p, "sn_" + knob)[SN_CLASS[cls]] = v
    return p


def make_patches(patches):
    arr = (OrcPatch * len(patches))()
    for i, d in enumerate(patches):
        a = arr[i]
        a.link = int(d["link"])
        a.origin[:] = [float(x) for x in d["origin"]]
        a.u_axis[:] = [float(x) for x in d["u_axis"]]
        a.v_axis[:] = [float(x) for x in d["v_axis"]]
        a.size_u, a.size_v = float(d["size_u"]), float(d["size_v"])
        a.nu, a.nv = int(d["nu"]), int(d["nv"])
        a.radius = float(d["radius"])
        a.marker_nu, a.marker_nv = int(d.get("marker_nu", 0)), int(d.get("marker_nv", 0))
    return arr


class Oracle:
    """One oracle context over `env_ids` (global env numbers; Philox counters use them)."""

    def __init__(self, patches, n_taxels, n_links, objs_per_env, env_ids, physics=None, noise=None, link_mask=None,
                 threads=1):
        self.L = lib()
        self.env_ids = np.ascontiguousarray(env_ids, dtype=np.int64)
        self.E, self.T, self.nl, self.K = len(self.env_ids), int(n_taxels), int(n_links), int(objs_per_env)
        self.params = make_params(physics, noise)
        self._patches = make_patches(patches)
        lm = None if link_mask is None else np.ascontiguousarray(link_mask, dtype=np.uint8)
        self.h = self.L.orc_create(C.byref(self.params), self._patches, len(patches), self.T, _p(lm), self.E,
                                   _p(self.env_ids), self.nl, self.K)
        if not self.h:
            raise ValueError("orc_create failed (patches need more taxels than n_taxels?)")
        self.M = self.L.orc_n_markers(self.h)
        self.threads = int(threads)

    def close(self):
        if self.h:
            self.L.orc_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def layout(self):
        T, M = self.T, self.M
        out = dict(pos=np.zeros((T, 3)), nrm=np.zeros((T, 3)), radius=np.zeros(T), link=np.zeros(T, np.int32),
                   patch=np.zeros(T, np.int32), nbr=np.zeros((T, 4), np.int32), marker_pos=np.zeros((M, 3)),
                   marker_nrm=np.zeros((M, 3)), marker_patch=np.zeros(M, np.int32))
        self.L.orc_get_layout(self.h, *[_p(out[k]) for k in ("pos", "nrm", "radius", "link", "patch", "nbr",
                                                              "marker_pos", "marker_nrm", "marker_patch")])
        return out

    def set_geometry(self, types, params, bank=None, voxel=0.0):
        types = np.ascontiguousarray(types, dtype=np.int32).reshape(self.E, self.K)
        params = _f32(params).reshape(self.E, self.K, 4)
        if bank is None:
            bank = np.zeros((0, 2, 2, 2), np.float32)
        bank = _f32(bank)
        n, N = bank.shape[0], bank.shape[1]
        rc = self.L.orc_set_geometry(self.h, _p(types), _p(params), n, N, float(voxel), _p(bank))
        if rc:
            raise ValueError("orc_set_geometry: grid id out of range")

    def set_pointclouds(self, points, cloud_id):
        """A.6: points [G, N, 3] fp32 (object frame); cloud_id [E, K] int32 (-1 = object not tracked)."""
        pts = _f32(points)
        cid = np.ascontiguousarray(cloud_id, dtype=np.int32).reshape(self.E, self.K)
        self._pc = True
        if self.L.orc_set_pointclouds(self.h, pts.shape[0], pts.shape[1], _p(pts), _p(cid)):
            raise ValueError("orc_set_pointclouds: cloud id out of range")

    def set_meshes(self, meshes, mesh_id):
        """A.1 raycast backend: meshes = list of (verts [V,3] fp32, tris [F,3] int32) in the object frame;
        mesh_id [E, K] int32 (-1 = object has no mesh)."""
        voff = np.cumsum([0] + [len(v) for v, _ in meshes]).astype(np.int32)
        toff = np.cumsum([0] + [len(t) for _, t in meshes]).astype(np.int32)
        verts = _f32(np.concatenate([v for v, _ in meshes]))
        tris = np.ascontiguousarray(np.concatenate([t for _, t in meshes]), dtype=np.int32)
        mid = np.ascontiguousarray(mesh_id, dtype=np.int32).reshape(self.E, self.K)
        if self.L.orc_set_meshes(self.h, len(meshes), _p(voff), _p(toff), _p(verts), _p(tris), _p(mid)):
            raise ValueError("orc_set_meshes: mesh id out of range")

    def reset(self, env_mask=None):
        m = None if env_mask is None else np.ascontiguousarray(env_mask, dtype=np.uint8)
        self.L.orc_reset(self.h, _p(m))

    def step(self, inp, want=("contact", "depth", "ft", "marker", "prox", "ft_noisy", "dead"), aux=True):
        """inp: dict with link_pos/link_quat/link_linvel/link_angvel [E,L,*], obj_* [E,K,*] (fp32)."""
        E, T, M = self.E, self.T, self.M
        a = {k: _f32(inp[k]) for k in ("link_pos", "link_quat", "link_linvel", "link_angvel", "obj_pos", "obj_quat",
                                       "obj_linvel", "obj_angvel")}
        assert a["link_pos"].shape == (E, self.nl, 3) and a["obj_quat"].shape == (E, self.K, 4)
        out = {}
        if "contact" in want: out["contact"] = np.zeros((E, T), np.uint8)
        if "depth" in want: out["depth"] = np.zeros((E, T))
        if "ft" in want: out["ft"] = np.zeros((E, T, 6))
        if "marker" in want and M > 0: out["marker"] = np.zeros((E, M, 3))
        if "prox" in want: out["prox"] = np.zeros((E, T))
        if "proxpc" in want: out["proxpc"] = np.zeros((E, T, 6))
        if "depth_rc" in want:
            out["depth_rc"] = np.zeros((E, T)); out["nrm_rc"] = np.zeros((E, T, 3)); out["aux_rc_gap"] = np.zeros((E, T))
        if self.params.noise_enable:
            if "ft_noisy" in want: out["ft_noisy"] = np.zeros((E, T, 6))
            if "dead" in want: out["dead"] = np.zeros((E, T), np.uint8)
            # noisy scalar readouts (R10); each needs its clean input computed too
            if "depth_noisy" in want: out["depth_noisy"] = np.zeros((E, T))
            if "prox_noisy" in want:
                out["prox_noisy"] = np.zeros((E, T)); out.setdefault("prox", np.zeros((E, T)))
            if "marker_noisy" in want and M > 0:
                out["marker_noisy"] = np.zeros((E, M, 3)); out.setdefault("marker", np.zeros((E, M, 3)))
        if aux:
            out["aux_phi"] = np.zeros((E, T))
            out["aux_face"] = np.zeros((E, T))
            out["aux_boxgap"] = np.zeros((E, T))
            if self.K > 1:
                out["aux_wingap"] = np.zeros((E, T))
            if self.params.noise_enable:
                out["aux_asym"] = np.zeros((E, T, 6))
                if self.params.quant_force > 0 or self.params.quant_torque > 0:
                    out["aux_quant"] = np.zeros((E, T, 6))
                if self.params.radius_noise != 0:
                    out["aux_rgate"] = np.zeros((E, T))
                if "depth_noisy" in out: out["aux_sq_depth"] = np.zeros((E, T))
                if "prox_noisy" in out: out["aux_sq_prox"] = np.zeros((E, T))
                if "marker_noisy" in out:
                    out["aux_sq_marker"] = np.zeros((E, M, 3)); out["aux_sasym_marker"] = np.zeros((E, M, 3))
        g = out.get
        self.L.orc_set_aux_quant(self.h, _p(g("aux_quant")))
        self.L.orc_set_aux_rgate(self.h, _p(g("aux_rgate")))
        self.L.orc_set_aux_wingap(self.h, _p(g("aux_wingap")))
        self.L.orc_set_proxpc(self.h, _p(g("proxpc")))
        self.L.orc_set_raycast_out(self.h, _p(g("depth_rc")), _p(g("nrm_rc")), _p(g("aux_rc_gap")))
        self.L.orc_set_scalar_noisy(self.h, _p(g("depth_noisy")), _p(g("prox_noisy")), _p(g("marker_noisy")), _p(g("aux_sq_depth")),
                                    _p(g("aux_sq_prox")), _p(g("aux_sq_marker")), _p(g("aux_sasym_marker")))
        self.L.orc_step(self.h, _p(a["link_pos"]), _p(a["link_quat"]), _p(a["link_linvel"]), _p(a["link_angvel"]),
                        _p(a["obj_pos"]), _p(a["obj_quat"]), _p(a["obj_linvel"]), _p(a["obj_angvel"]),
                        _p(g("contact")), _p(g("depth")), _p(g("ft")), _p(g("marker")), _p(g("prox")),
                        _p(g("ft_noisy")), _p(g("dead")), _p(g("aux_phi")), _p(g("aux_face")), _p(g("aux_boxgap")),
                        _p(g("aux_asym")), self.threads)
        return out


# ---- stand-alone pieces (pins) ------------------------------------------------------

def philox(ctr, key):
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    o = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(c), _p(k), _p(o))
    return o


def uniform(word):
    return lib().orc_uniform(int(word))


def box_muller(wa, wb):
    z = np.zeros(2)
    lib().orc_box_muller(int(wa), int(wb), _p(z))
    return z


def sdf_query(kind, params, x, grid=None, voxel=0.0):
    """-> dict(phi, grad (unnormalised, object frame), face, boxgap)."""
    pr = np.zeros(4)
    pr[:len(params)] = params
    x = _f64(x)
    o = np.zeros(6)
    N = 0
    gp = None
    if grid is not None:
        grid = _f32(grid)
        N = grid.shape[0]
        gp = grid
    lib().orc_sdf_query(GEOM[kind], _p(pr), _p(gp), N, float(voxel), _p(x), _p(o))
    return dict(phi=o[0], grad=o[1:4].copy(), face=o[4], boxgap=o[5])


def kinematic_ft(d, m_world, x_j, quat_L=(1, 0, 0, 0), pL=(0, 0, 0), vL=(0, 0, 0), wL=(0, 0, 0), pO=(0, 0, 0),
                 vO=(0, 0, 0), wO=(0, 0, 0), physics=None):
    pr = make_params(physics)
    out = np.zeros(6)
    args = [_f64(m_world), _f64(x_j), _f32(quat_L), _f64(pL), _f64(vL), _f64(wL), _f64(pO), _f64(vO), _f64(wO)]
    lib().orc_kinematic_ft(C.byref(pr), float(d), *[_p(a) for a in args], _p(out))
    return out


def march(kind, params, x0, a, r_prox, steps, grid=None, voxel=0.0):
    pr = np.zeros(4)
    pr[:len(params)] = params
    N = 0
    gp = None
    if grid is not None:
        gp = _f32(grid)
        N = gp.shape[0]
    x0, a = _f64(x0), _f64(a)
    return lib().orc_march(GEOM[kind], _p(pr), _p(gp), N, float(voxel), _p(x0), _p(a), float(r_prox), int(steps))


def closest_point_triangle(p, a, b, c):
    o = np.zeros(3)
    lib().orc_closest_point_triangle(_p(_f64(p)), _p(_f64(a)), _p(_f64(b)), _p(_f64(c)), _p(o))
    return o


def ray_triangle(orig, d, a, b, c):
    return lib().orc_ray_triangle(_p(_f64(orig)), _p(_f64(d)), _p(_f64(a)), _p(_f64(b)), _p(_f64(c)))


def max_threads():
    return lib().orc_max_threads()
