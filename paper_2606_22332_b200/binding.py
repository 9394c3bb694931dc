"""Thin Python binding of include/ts.h (ctypes).  Argument marshalling only: every step of the
path runs in the CUDA kernels of libts.so.  PyTorch supplies device memory and streams.

There is no CPU fallback: importing is cheap, but any call raises if libts.so is missing.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libts.so")

TS_OK = 0
TS_ERR_INVALID_ARG = 1
STATUS = {0: "TS_OK", 1: "TS_ERR_INVALID_ARG", 2: "TS_ERR_CUDA", 3: "TS_ERR_OOM", 4: "TS_ERR_STATE",
          5: "TS_ERR_UNSUPPORTED"}
HYST = {"off": 0, "maxwell": 1, "asym": 2}
FORM = {"auto": 0, "fused": 1, "split": 2}
GEOM = {"none": 0, "sphere": 1, "box": 2, "capsule": 3, "sdf": 4, "grid": 4}
OUT_BITS = {"contact": 1, "depth": 2, "ft": 4, "marker": 8, "prox": 16, "ft_noisy": 32, "dead": 64,
            "depth_noisy": 128, "prox_noisy": 256, "marker_noisy": 512, "proxpc": 1024, "depth_rc": 2048, "nrm_rc": 4096}
SN_CLASS = {"depth": 0, "prox": 1, "marker": 2}          # noisy scalar readouts (ts_config.sn_*[3])
SN_KNOBS = ("sigma_white", "sigma_rw", "bias", "quant", "stuck_min", "stuck_max")

# every symbol include/ts.h declares (tests check that the library exports them all)
SYMBOLS = ["ts_layout_create", "ts_layout_add_patch", "ts_layout_filter_links", "ts_layout_finalize", "ts_layout_get",
           "ts_layout_destroy", "ts_config_default", "ts_create", "ts_set_geometry", "ts_set_pointclouds", "ts_set_meshes", "ts_step", "ts_step_host",
           "ts_reset", "ts_destroy", "ts_last_error", "ts_n_taxels", "ts_n_markers", "ts_launches_per_step",
           "ts_kernel_time_ms", "ts_kernel_times_ms", "ts_first_kernel_time_ms", "ts_version",
           "ts_state_bytes", "ts_get_state", "ts_set_state", "ts_depth_static"]
STATIC_SCRATCH_BYTES = 8 << 20                      # include/ts.h TS_STATIC_SCRATCH_BYTES
STATIC_MAX_FRAMES = STATIC_SCRATCH_BYTES // 96      # TS_STATIC_MAX_FRAMES


class TsError(RuntimeError):
    pass


class PatchDesc(C.Structure):
    _fields_ = [("link", C.c_int32), ("origin", C.c_float * 3), ("u_axis", C.c_float * 3), ("v_axis", C.c_float * 3),
                ("size_u", C.c_float), ("size_v", C.c_float), ("nu", C.c_int32), ("nv", C.c_int32),
                ("radius", C.c_float), ("marker_nu", C.c_int32), ("marker_nv", C.c_int32)]


class LayoutView(C.Structure):
    _fields_ = [("n_taxels", C.c_int32), ("n_patches", C.c_int32), ("n_markers", C.c_int32),
                ("pos", C.POINTER(C.c_float)), ("nrm", C.POINTER(C.c_float)), ("radius", C.POINTER(C.c_float)),
                ("link", C.POINTER(C.c_int32)), ("patch", C.POINTER(C.c_int32)), ("nbr", C.POINTER(C.c_int32)),
                ("patch_start", C.POINTER(C.c_int32)), ("patch_nu", C.POINTER(C.c_int32)),
                ("patch_nv", C.POINTER(C.c_int32)), ("patch_link", C.POINTER(C.c_int32)),
                ("marker_start", C.POINTER(C.c_int32)), ("marker_count", C.POINTER(C.c_int32)),
                ("marker_pos", C.POINTER(C.c_float)), ("marker_nrm", C.POINTER(C.c_float)),
                ("marker_patch", C.POINTER(C.c_int32))]


class Config(C.Structure):
    _fields_ = [("n_envs", C.c_int32), ("n_links", C.c_int32), ("objs_per_env", C.c_int32),
                ("env_id_base", C.c_int64), ("layout", C.c_void_p),
                ("k_n", C.c_float), ("c_n", C.c_float), ("alpha", C.c_float), ("k_t", C.c_float),
                ("k_omega", C.c_float), ("mu", C.c_float), ("use_velocity", C.c_int32),
                ("eta_on", C.c_float), ("eta_off", C.c_float),
                ("s_d", C.c_float), ("lambda_d", C.c_float), ("alpha_e", C.c_float), ("c_e", C.c_float),
                ("r_prox", C.c_float), ("march_steps", C.c_int32), ("dt", C.c_float),
                ("noise_enable", C.c_int32), ("seed", C.c_uint64),
                ("sigma_rw_force", C.c_float), ("sigma_rw_torque", C.c_float), ("hyst_mode", C.c_int32),
                ("beta", C.c_float), ("tau", C.c_float), ("alpha_load", C.c_float), ("alpha_unload", C.c_float),
                ("p_dead", C.c_float), ("chi", C.c_float), ("output_mask", C.c_uint32),
                ("sigma_white_force", C.c_float), ("sigma_white_torque", C.c_float),
                ("bias_force", C.c_float), ("bias_torque", C.c_float),
                ("quant_force", C.c_float), ("quant_torque", C.c_float),
                ("gain_min", C.c_float), ("gain_max", C.c_float),
                ("stuck_min_force", C.c_float), ("stuck_max_force", C.c_float),
                ("stuck_min_torque", C.c_float), ("stuck_max_torque", C.c_float), ("xtalk_sigma", C.c_float),
                ("radius_noise", C.c_float), ("read_delay", C.c_int32), ("read_jitter", C.c_int32),
                ("kernel_form", C.c_int32),
                ("sn_sigma_white", C.c_float * 3), ("sn_sigma_rw", C.c_float * 3), ("sn_bias", C.c_float * 3),
                ("sn_quant", C.c_float * 3), ("sn_stuck_min", C.c_float * 3), ("sn_stuck_max", C.c_float * 3),
                ("pc_radius", C.c_float), ("pc_k", C.c_float), ("pc_ks", C.c_float), ("pc_density", C.c_float),
                ("shear_enable", C.c_int32), ("s_s", C.c_float), ("lambda_s", C.c_float), ("eta_enter", C.c_float),
                ("eta_exit", C.c_float)]


class Meshes(C.Structure):
    _fields_ = [("n_meshes", C.c_int32), ("vert_off", C.c_void_p), ("tri_off", C.c_void_p), ("verts", C.c_void_p),
                ("tris", C.c_void_p), ("mesh_id", C.c_void_p)]


class PointClouds(C.Structure):
    _fields_ = [("n_clouds", C.c_int32), ("n_points", C.c_int32), ("points", C.c_void_p), ("cloud_id", C.c_void_p)]


class Geometry(C.Structure):
    _fields_ = [("type", C.c_void_p), ("params", C.c_void_p), ("n_grids", C.c_int32), ("grid_n", C.c_int32),
                ("voxel", C.c_float), ("grids", C.c_void_p)]


class StepIn(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("link_pos", "link_quat", "link_linvel", "link_angvel", "obj_pos", "obj_quat",
                                          "obj_linvel", "obj_angvel")]


class StepOut(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("contact", "depth", "ft", "marker", "prox", "ft_noisy", "dead", "depth_noisy",
                                          "prox_noisy", "marker_noisy", "proxpc", "depth_rc", "nrm_rc")]


IN_KEYS = [k for k, _ in StepIn._fields_]
OUT_KEYS = [k for k, _ in StepOut._fields_]
_lib = None


def lib():
    """Loads libts.so (built in-tree by paper_2606_22332_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise TsError("libts.so not found at %s: build it with `python -m paper_2606_22332_b200.build` "
                          "(there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp, i32 = C.c_void_p, C.c_int32
        L.ts_layout_create.argtypes = [C.POINTER(vp)]
        L.ts_layout_add_patch.argtypes = [vp, C.POINTER(PatchDesc)]
        L.ts_layout_filter_links.argtypes = [vp, vp, i32]
        L.ts_layout_finalize.argtypes = [vp, i32]
        L.ts_layout_get.argtypes = [vp, C.POINTER(LayoutView)]
        L.ts_layout_destroy.argtypes = [vp]
        L.ts_config_default.argtypes = [C.POINTER(Config)]
        L.ts_config_default.restype = None
        L.ts_create.argtypes = [C.POINTER(Config), C.c_int, C.POINTER(vp)]
        L.ts_set_geometry.argtypes = [vp, C.POINTER(Geometry), vp]
        L.ts_set_pointclouds.argtypes = [vp, C.POINTER(PointClouds), vp]
        L.ts_set_meshes.argtypes = [vp, C.POINTER(Meshes), vp]
        L.ts_step.argtypes = [vp, C.POINTER(StepIn), C.POINTER(StepOut), vp]
        L.ts_step_host.argtypes = [vp, C.POINTER(StepIn), C.POINTER(StepOut), vp]
        L.ts_reset.argtypes = [vp, vp, vp]
        L.ts_destroy.argtypes = [vp]
        L.ts_last_error.argtypes = [vp]
        L.ts_last_error.restype = C.c_char_p
        L.ts_n_taxels.argtypes = [vp]
        L.ts_n_markers.argtypes = [vp]
        L.ts_launches_per_step.argtypes = [vp]
        L.ts_kernel_time_ms.argtypes = [vp, i32, C.POINTER(C.c_float), C.POINTER(i32)]
        L.ts_kernel_times_ms.argtypes = [vp, vp, i32, C.POINTER(i32)]
        L.ts_first_kernel_time_ms.argtypes = [vp]
        L.ts_state_bytes.argtypes = [vp, C.POINTER(C.c_uint64)]
        L.ts_get_state.argtypes = [vp, vp, C.c_uint64, vp]
        L.ts_set_state.argtypes = [vp, vp, C.c_uint64, vp]
        L.ts_depth_static.argtypes = [i32, i32, i32] + [vp] * 11
        L.ts_first_kernel_time_ms.restype = C.c_float
        L.ts_version.restype = C.c_char_p
        _lib = L
    return _lib


def _check(rc, ctx=None, what=""):
    if rc != TS_OK:
        msg = lib().ts_last_error(ctx)
        raise TsError("%s: %s (%s)" % (what, STATUS.get(rc, rc), msg.decode() if msg else ""))


class Layout:
    """ts_layout_* : the taxel-layout builder (S0)."""

    def __init__(self, patches, n_taxels, link_mask=None, n_links=None):
        L = lib()
        self.h = C.c_void_p()
        _check(L.ts_layout_create(C.byref(self.h)), None, "ts_layout_create")
        for d in patches:
            pd = PatchDesc()
            pd.link = int(d["link"])
            pd.origin[:] = [float(x) for x in d["origin"]]
            pd.u_axis[:] = [float(x) for x in d["u_axis"]]
            pd.v_axis[:] = [float(x) for x in d["v_axis"]]
            pd.size_u, pd.size_v = float(d["size_u"]), float(d["size_v"])
            pd.nu, pd.nv = int(d["nu"]), int(d["nv"])
            pd.radius = float(d["radius"])
            pd.marker_nu, pd.marker_nv = int(d.get("marker_nu", 0)), int(d.get("marker_nv", 0))
            _check(L.ts_layout_add_patch(self.h, C.byref(pd)), None, "ts_layout_add_patch")
        if link_mask is not None:
            m = np.ascontiguousarray(link_mask, dtype=np.uint8)
            _check(L.ts_layout_filter_links(self.h, m.ctypes.data_as(C.c_void_p), int(n_links or len(m))), None,
                   "ts_layout_filter_links")
        _check(L.ts_layout_finalize(self.h, int(n_taxels)), None, "ts_layout_finalize")

    def view(self):
        v = LayoutView()
        _check(lib().ts_layout_get(self.h, C.byref(v)), None, "ts_layout_get")
        T, P, M = v.n_taxels, v.n_patches, v.n_markers

        def arr(ptr, shape):
            n = int(np.prod(shape))
            return np.ctypeslib.as_array(ptr, shape=(n,)).reshape(shape).copy() if n else np.zeros(shape)
        return dict(pos=arr(v.pos, (T, 3)), nrm=arr(v.nrm, (T, 3)), radius=arr(v.radius, (T,)), link=arr(v.link, (T,)),
                    patch=arr(v.patch, (T,)), nbr=arr(v.nbr, (T, 4)), patch_start=arr(v.patch_start, (P,)),
                    patch_nu=arr(v.patch_nu, (P,)), patch_nv=arr(v.patch_nv, (P,)), patch_link=arr(v.patch_link, (P,)),
                    marker_start=arr(v.marker_start, (P,)), marker_count=arr(v.marker_count, (P,)),
                    marker_pos=arr(v.marker_pos, (M, 3)), marker_nrm=arr(v.marker_nrm, (M, 3)),
                    marker_patch=arr(v.marker_patch, (M,)))

    def close(self):
        if self.h:
            lib().ts_layout_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def make_config(n_envs, n_links, objs_per_env, layout, physics=None, noise=None, outputs=None, env_id_base=0):
    cfg = Config()
    lib().ts_config_default(C.byref(cfg))
    cfg.n_envs, cfg.n_links, cfg.objs_per_env = int(n_envs), int(n_links), int(objs_per_env)
    cfg.env_id_base = int(env_id_base)
    cfg.layout = layout.h
    names = {f for f, _ in Config._fields_}
    for src in (physics, noise):
        for k, v in (src or {}).items():
            knob, _, cls = k.rpartition("_")
            if knob in SN_KNOBS and cls in SN_CLASS:         # e.g. sigma_white_depth, quant_marker -> sn_*[class]
                getattr(cfg, "sn_" + knob)[SN_CLASS[cls]] = float(v)
                continue
            if k not in names:
                raise KeyError(k)
            if k == "hyst_mode" and isinstance(v, str):
                v = HYST[v]
            if k == "kernel_form" and isinstance(v, str):
                v = FORM[v]
            setattr(cfg, k, v)
    # test override only: TS_SPLIT=0 / 1 in the environment forces the fused / two-kernel form when the caller left
    # kernel_form on AUTO (the C library itself reads no environment variable)
    if cfg.kernel_form == 0 and os.environ.get("TS_SPLIT") in ("0", "1"):
        cfg.kernel_form = FORM["split"] if os.environ["TS_SPLIT"] == "1" else FORM["fused"]
    if outputs is not None:
        cfg.output_mask = sum(OUT_BITS[o] for o in outputs)
    return cfg


def depth_static(n_envs, n_links, n_taxels, taxel_pos, taxel_radius, taxel_link, link_pos, link_quat, obj_pos, obj_quat,
                 geom_type, geom_params, depth, stream=None):
    """ts_depth_static on device tensors (anything with data_ptr(); fp32 / int32, contiguous): the allocation-free contact
    depth against one primitive per env, on the current device.  Marshalling only; `stream` is a raw cudaStream_t or None."""
    ptr = lambda t: C.c_void_p(t.data_ptr() if t is not None else 0)
    st = lib().ts_depth_static(int(n_envs), int(n_links), int(n_taxels), ptr(taxel_pos), ptr(taxel_radius), ptr(taxel_link),
                               ptr(link_pos), ptr(link_quat), ptr(obj_pos), ptr(obj_quat), ptr(geom_type), ptr(geom_params),
                               ptr(depth), C.c_void_p(stream or 0))
    _check(st, None, "ts_depth_static")


class TactileSim:
    """ts_create / ts_set_geometry / ts_step / ts_reset / ts_destroy on torch device tensors."""

    def __init__(self, patches, n_taxels, n_envs, n_links, objs_per_env=1, physics=None, noise=None, outputs=None,
                 link_mask=None, env_id_base=0, device=0):
        import torch
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.layout = Layout(patches, n_taxels, link_mask, n_links)
        self.noise_on = bool((noise or {}).get("noise_enable", 0))
        if outputs is None:
            outputs = ["contact", "depth", "ft", "prox"] + (["ft_noisy", "dead"] if self.noise_on else [])
            if any(int(p.get("marker_nu", 0)) > 0 for p in patches):
                outputs.append("marker")
        self.outputs = tuple(outputs)
        self.cfg = make_config(n_envs, n_links, objs_per_env, self.layout, physics, noise, self.outputs, env_id_base)
        self.h = C.c_void_p()
        _check(lib().ts_create(C.byref(self.cfg), int(device), C.byref(self.h)), None, "ts_create")
        self.E, self.L, self.K = int(n_envs), int(n_links), int(objs_per_env)
        self.T, self.M = lib().ts_n_taxels(self.h), lib().ts_n_markers(self.h)

    # -- helpers
    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def out_shapes(self):
        E, T, M = self.E, self.T, self.M
        t = self.torch
        return dict(contact=((E, T), t.uint8), depth=((E, T), t.float32), ft=((E, T, 6), t.float32),
                    marker=((E, M, 3), t.float32), prox=((E, T), t.float32), ft_noisy=((E, T, 6), t.float32),
                    dead=((E, T), t.uint8), depth_noisy=((E, T), t.float32), prox_noisy=((E, T), t.float32),
                    marker_noisy=((E, M, 3), t.float32), proxpc=((E, T, 6), t.float32),
                    depth_rc=((E, T), t.float32), nrm_rc=((E, T, 3), t.float32))

    def in_shapes(self):
        E, L, K = self.E, self.L, self.K
        return dict(link_pos=(E, L, 3), link_quat=(E, L, 4), link_linvel=(E, L, 3), link_angvel=(E, L, 3),
                    obj_pos=(E, K, 3), obj_quat=(E, K, 4), obj_linvel=(E, K, 3), obj_angvel=(E, K, 3))

    def alloc_outputs(self, pinned_host=False):
        sh = self.out_shapes()
        if pinned_host:
            return {k: self.torch.empty(sh[k][0], dtype=sh[k][1], pin_memory=True) for k in self.outputs}
        return {k: self.torch.empty(sh[k][0], dtype=sh[k][1], device=self.device) for k in self.outputs}

    def upload(self, inp):
        t = self.torch
        return {k: t.from_numpy(np.ascontiguousarray(inp[k], dtype=np.float32)).to(self.device) for k in IN_KEYS}

    # -- C-ABI calls
    def set_geometry(self, types, params, bank=None, voxel=0.0):
        types = np.ascontiguousarray(types, dtype=np.int32).reshape(self.E, self.K)
        params = np.ascontiguousarray(params, dtype=np.float32).reshape(self.E, self.K, 4)
        g = Geometry()
        g.type = types.ctypes.data_as(C.c_void_p)
        g.params = params.ctypes.data_as(C.c_void_p)
        if bank is not None and len(bank):
            bank = np.ascontiguousarray(bank, dtype=np.float32)
            g.n_grids, g.grid_n, g.voxel = bank.shape[0], bank.shape[1], float(voxel)
            g.grids = bank.ctypes.data_as(C.c_void_p)
        with self.torch.cuda.device(self.device):
            _check(lib().ts_set_geometry(self.h, C.byref(g), self._stream()), self.h, "ts_set_geometry")

    def set_meshes(self, meshes, mesh_id):
        """App. A.1 raycast backend: meshes = list of (verts [V,3] fp32, tris [F,3] int32) in the object frame;
        mesh_id [E, K] int32 (-1 = object has no mesh)."""
        voff = np.cumsum([0] + [len(v) for v, _ in meshes]).astype(np.int32)
        toff = np.cumsum([0] + [len(t) for _, t in meshes]).astype(np.int32)
        verts = np.ascontiguousarray(np.concatenate([v for v, _ in meshes]), dtype=np.float32)
        tris = np.ascontiguousarray(np.concatenate([t for _, t in meshes]), dtype=np.int32)
        mid = np.ascontiguousarray(mesh_id, dtype=np.int32).reshape(self.E, self.K)
        vp = lambda a: a.ctypes.data_as(C.c_void_p)
        m = Meshes(len(meshes), vp(voff), vp(toff), vp(verts), vp(tris), vp(mid))
        with self.torch.cuda.device(self.device):
            _check(lib().ts_set_meshes(self.h, C.byref(m), self._stream()), self.h, "ts_set_meshes")

    def set_pointclouds(self, points, cloud_id):
        """App. A.6: points [G, N, 3] fp32 in the object frame; cloud_id [E, K] int32 (-1 = object not tracked)."""
        pts = np.ascontiguousarray(points, dtype=np.float32)
        cid = np.ascontiguousarray(cloud_id, dtype=np.int32).reshape(self.E, self.K)
        pc = PointClouds(pts.shape[0], pts.shape[1], pts.ctypes.data_as(C.c_void_p), cid.ctypes.data_as(C.c_void_p))
        with self.torch.cuda.device(self.device):
            _check(lib().ts_set_pointclouds(self.h, C.byref(pc), self._stream()), self.h, "ts_set_pointclouds")

    def _structs(self, inp, out, host):
        si, so = StepIn(), StepOut()
        ish, osh = self.in_shapes(), self.out_shapes()
        for k in IN_KEYS:
            a = inp[k]
            assert tuple(a.shape) == ish[k] and a.dtype == self.torch.float32 and a.is_contiguous(), k
            assert a.is_cuda != host, k
            setattr(si, k, a.data_ptr())
        for k, a in out.items():
            assert tuple(a.shape) == osh[k][0] and a.dtype == osh[k][1] and a.is_contiguous(), k
            assert a.is_cuda != host, k
            setattr(so, k, a.data_ptr())
        return si, so

    def step(self, inp, out=None):
        """inp: dict of CUDA fp32 tensors (IN_KEYS); out: dict of CUDA tensors (allocated if None).  Asynchronous."""
        if out is None:
            out = self.alloc_outputs()
        si, so = self._structs(inp, out, host=False)
        _check(lib().ts_step(self.h, C.byref(si), C.byref(so), self._stream()), self.h, "ts_step")
        return out

    def step_host(self, inp, out):
        """Same step on HOST tensors (pinned recommended): H2D, kernels, D2H, all enqueued on the current stream."""
        si, so = self._structs(inp, out, host=True)
        _check(lib().ts_step_host(self.h, C.byref(si), C.byref(so), self._stream()), self.h, "ts_step_host")
        return out

    def reset(self, env_mask=None):
        ptr = None
        if env_mask is not None:
            assert env_mask.is_cuda and env_mask.dtype == self.torch.uint8 and env_mask.numel() == self.E
            ptr = C.c_void_p(env_mask.data_ptr())
        _check(lib().ts_reset(self.h, ptr, self._stream()), self.h, "ts_reset")

    def kernel_time_ms(self, enable=True):
        """enable: False / 0 = off, True / 1 = events around the whole step, 2 = events between its kernels too."""
        ms, n = C.c_float(), C.c_int32()
        _check(lib().ts_kernel_time_ms(self.h, int(enable), C.byref(ms), C.byref(n)), self.h, "ts_kernel_time_ms")
        return ms.value, n.value

    def kernel_times_ms(self):
        """Per-step durations [n, 4] recorded since recording was switched on: frames, step, noise kernel (CUDA events)
        and the step's span on the device-side clock (%globaltimer, first block start to last block end), in ms."""
        n = C.c_int32()
        _check(lib().ts_kernel_times_ms(self.h, None, 0, C.byref(n)), self.h, "ts_kernel_times_ms")
        out = np.zeros((max(n.value, 1), 4), np.float32)
        _check(lib().ts_kernel_times_ms(self.h, out.ctypes.data_as(C.c_void_p), n.value, C.byref(n)), self.h, "ts_kernel_times_ms")
        return out[:n.value]

    def state_bytes(self):
        n = C.c_uint64()
        _check(lib().ts_state_bytes(self.h, C.byref(n)), self.h, "ts_state_bytes")
        return int(n.value)

    def get_state(self):
        """The ctx's step-to-step state as one host blob (uint8 array): checkpoint."""
        blob = np.empty(self.state_bytes(), np.uint8)
        _check(lib().ts_get_state(self.h, blob.ctypes.data_as(C.c_void_p), blob.nbytes, self._stream()), self.h, "ts_get_state")
        return blob

    def set_state(self, blob):
        """Restore a blob taken by get_state() from a ctx with the same layout and configuration: resume."""
        blob = np.ascontiguousarray(blob, np.uint8)
        _check(lib().ts_set_state(self.h, blob.ctypes.data_as(C.c_void_p), blob.nbytes, self._stream()), self.h, "ts_set_state")

    def first_kernel_time_ms(self):
        return float(lib().ts_first_kernel_time_ms(self.h))

    def launches_per_step(self):
        return lib().ts_launches_per_step(self.h)

    def close(self):
        if getattr(self, "h", None):
            lib().ts_destroy(self.h)
            self.h = None
        if getattr(self, "layout", None):
            self.layout.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
