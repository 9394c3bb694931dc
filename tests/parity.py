"""Comparator: CUDA path vs oracle, element by element, with the band accounting of DESIGN.md.

Tolerances (BASELINE.json north_star): floats |gpu - ref| <= 1e-6 + 1e-4 |ref|; contact / dead
bit-exact outside a 1e-6 m band around the thresholds.  A band only EXEMPTS an element (and is
counted and reported); tolerances are never loosened.
"""
import numpy as np

import math

ATOL, RTOL, BAND = 1e-6, 1e-4, 1e-6
FACE_BAND = 1e-4        # voxels: trilinear gradient jumps across cell faces
NOISY_TAINT_STEPS = 100  # default hysteresis memory of an exempted ft value (Maxwell, tau = 0.05 s: 0.905^100 < 1e-4)


def taint_steps(noise):
    """Steps until an exempted ft value has left the hysteresis state (its weight has decayed below RTOL):
    Maxwell xi decays by exp(-dt / tau) per step (Eq. 29), ASYM y by (1 - min(alpha_load, alpha_unload)) (D3);
    without hysteresis the chain has no memory of past ft values (drift and white noise do not depend on ft).
    A read delay of Delta + J steps (R9) shows the value that much later."""
    if not noise:
        return NOISY_TAINT_STEPS
    hm = noise.get("hyst_mode", "off")
    delay = int(noise.get("read_delay", 0)) + int(noise.get("read_jitter", 0))
    if hm in ("maxwell", 1):
        r = math.exp(-float(noise.get("dt", 0.005)) / float(noise.get("tau", 0.05)))
    elif hm in ("asym", 2):
        r = 1.0 - min(float(noise.get("alpha_load", 1.0)), float(noise.get("alpha_unload", 1.0)))
    else:
        return 1 + delay
    if r <= 0.0:
        return 1 + delay
    return min(NOISY_TAINT_STEPS, 1 + int(math.ceil(math.log(RTOL) / math.log(r)))) + delay


class Comparator:
    def __init__(self, layout, physics, noise_on, radius, noise=None):
        self.nbr = np.asarray(layout["nbr"])
        self.taint_steps = taint_steps(noise)
        sg = float((noise or {}).get("xtalk_sigma", 0.0))
        self.xt_radius = int(math.ceil(3.0 * sg)) if sg > 0 else 0   # R7: Gaussian support, else the 4-neighbour stencil
        self.eta_on = float(np.float32(physics.get("eta_on", 5e-4)))
        self.eta_off = float(np.float32(physics.get("eta_off", 5e-4)))
        self.radius = np.asarray(radius, np.float64)
        self.noise_on = noise_on
        self.quant = (0.0, 0.0)   # Eq. 25 steps (force, torque); set by the caller when quantisation is on
        self.sn_quant = tuple(float(np.float32((noise or {}).get("quant_" + c, 0.0))) for c in ("depth", "prox", "marker"))
        self.sn_taint = {}
        self.contact_taint = None
        self.noisy_taint = None
        self.stats = dict(steps=0, contact_band=0, contact_tainted=0, ft_exempt=0, noisy_exempt=0, quant_exempt=0,
                          win_tie=0, checked=0, taxel_steps=0, noisy_taxel_steps=0, max_ratio={})
        self.failures = []

    def _tol_ratio(self, g, r):
        return np.abs(g.astype(np.float64) - r) / (ATOL + RTOL * np.abs(r))

    def step(self, gpu, ref):
        st = self.stats
        st["steps"] += 1
        d = ref["depth"]
        E, T = d.shape
        if self.contact_taint is None:
            self.contact_taint = np.zeros((E, T), bool)
            self.noisy_taint = np.zeros((E, T), np.int32)
        # ---- contact: Schmitt band + taint
        band = (np.abs(d - self.eta_on) < BAND) | (np.abs(d - self.eta_off) < BAND)
        decisive = (d > self.eta_on + BAND) | (d < self.eta_off - BAND)
        self.contact_taint = (self.contact_taint | band) & ~decisive
        st["contact_band"] += int(band.sum())
        st["contact_tainted"] += int(self.contact_taint.sum())
        if "contact" in gpu:
            bad = (gpu["contact"] != ref["contact"]) & ~self.contact_taint
            if bad.any():
                self.failures.append(("contact", st["steps"] - 1, int(bad.sum()), np.argwhere(bad)[:4].tolist()))
        if "dead" in gpu:
            bad = gpu["dead"] != ref["dead"]
            if bad.any():
                self.failures.append(("dead", st["steps"] - 1, int(bad.sum()), np.argwhere(bad)[:4].tolist()))
        # ---- scalar float outputs
        for k in ("depth", "prox"):
            if k in gpu:
                self._check(k, gpu[k], ref[k], None)
        if "marker" in gpu:
            self._check("marker", gpu["marker"], ref["marker"], None)
        # ---- noisy scalar readouts (R10): continuous in their inputs; only a quantisation flip (one step q while the
        # pre-quantisation value sits within the tolerance of a rounding boundary) or, for the signed marker channels, an
        # ASYM load/unload tie can legitimately differ; such elements are exempted, counted, and taint the hysteresis state
        for k, cls in (("depth_noisy", 0), ("prox_noisy", 1), ("marker_noisy", 2)):
            if k not in gpu:
                continue
            r = ref[k]
            ex = np.zeros(r.shape, bool)
            tol = ATOL + RTOL * np.abs(r)
            q = self.sn_quant[cls]
            if q > 0:
                diff = np.abs(gpu[k].astype(np.float64) - r)
                aq = ref["aux_sq_" + k.split("_")[0]]
                ex |= (np.abs(diff - q) <= 1e-6 * np.maximum(np.abs(r), q)) & (aq < tol)
            if k == "marker_noisy" and "aux_sasym_marker" in ref:
                ex |= np.abs(ref["aux_sasym_marker"]) < BAND
            t = self.sn_taint.setdefault(k, np.zeros(r.shape, np.int32))
            t[:] = np.maximum(t - 1, 0)
            t[ex] = self.taint_steps
            exn = t > 0
            st["sn_exempt"] = st.get("sn_exempt", 0) + int(exn.sum())
            st["sn_checked"] = st.get("sn_checked", 0) + exn.size
            self._check(k, gpu[k], r, exn)
        # ---- ft: exempt discontinuities of the normal / the d > 0 gate
        phi = ref["aux_phi"]
        active = self.radius[None, :] > 0
        gate = np.abs(self.radius[None, :] - phi) < BAND
        face = (ref["aux_face"] < FACE_BAND) & (d > 0)
        box = (ref["aux_boxgap"] < BAND) & (d > 0)
        ex = (gate | face | box) & active
        if "aux_wingap" in ref:                    # K > 1: two objects within 1e-6 of the winning phi: g* (and the normal) may differ
            tie = (ref["aux_wingap"] < BAND) & (d > 0) & active
            st["win_tie"] += int(tie.sum())
            ex = ex | tie
        st["ft_exempt"] += int(ex.sum())
        st["taxel_steps"] += int(active.sum()) * E
        if "ft" in gpu:
            self._check("ft", gpu["ft"], ref["ft"], ex)
        if "ft_noisy" in gpu:
            asym = np.zeros((E, T), bool)
            if "aux_asym" in ref:
                asym = (np.abs(ref["aux_asym"]) < BAND).any(-1)
            src = ex | asym
            if "aux_rgate" in ref:                 # Eq. 26: the noisy readout's own d~ > 0 gate sits at R~_j, not R_j
                src = src | ((ref["aux_rgate"] < BAND) & active)
            self.noisy_taint = np.maximum(self.noisy_taint - 1, 0)
            self.noisy_taint[src] = self.taint_steps
            t = self.noisy_taint > 0
            spread = self._spread(t)               # crosstalk carries a tainted value over its support
            st["noisy_exempt"] += int(spread.sum())
            st["noisy_taxel_steps"] += int(active.sum()) * E
            ex6 = np.broadcast_to(spread[..., None], ref["ft_noisy"].shape)
            if "aux_quant" in ref:
                # Eq. 25 quantize(): a readout whose pre-quantisation value lies within the float tolerance of a
                # rounding boundary may legitimately land exactly one step away.  Only elements that DO differ by
                # one step (to fp32 rounding) AND sit in that band are exempted and counted; nothing is loosened.
                r = ref["ft_noisy"]
                tol = ATOL + RTOL * np.abs(r)
                q = np.array([self.quant[0]] * 3 + [self.quant[1]] * 3, np.float64)
                diff = np.abs(gpu["ft_noisy"].astype(np.float64) - r)
                one_step = (q > 0) & (np.abs(diff - q) <= 1e-6 * np.maximum(np.abs(r), q))
                qflip = one_step & (ref["aux_quant"] < tol)
                st["quant_exempt"] += int((qflip & ~ex6).sum())
                ex6 = ex6 | qflip
            self._check("ft_noisy", gpu["ft_noisy"], ref["ft_noisy"], ex6)

    def _spread(self, t):
        """Taxels whose crosstalk support (Eq. 31) contains a tainted taxel: the 4 neighbours (D4), or the
        (2r+1) x (2r+1) square of the Gaussian kernel (R7), within the patch."""
        def dilate(m, cols):
            out = m.copy()
            for a in cols:
                nb = self.nbr[:, a]
                ok = nb >= 0
                out[:, ok] |= m[:, nb[ok]]
            return out
        if self.xt_radius == 0:
            return dilate(t, (0, 1, 2, 3))
        s = t
        for _ in range(self.xt_radius):
            s = dilate(s, (0, 1))                  # along u
        for _ in range(self.xt_radius):
            s = dilate(s, (2, 3))                  # along v
        return s

    def _check(self, name, g, r, exempt):
        ratio = self._tol_ratio(g, r)
        if not np.isfinite(g).all():
            self.failures.append((name, self.stats["steps"] - 1, "non-finite", []))
            return
        if exempt is not None:
            ex = exempt[..., None] if (ratio.ndim == 3 and exempt.ndim == 2) else exempt
            ratio = np.where(ex, 0.0, ratio)
        self.stats["checked"] += ratio.size
        m = float(ratio.max()) if ratio.size else 0.0
        self.stats["max_ratio"][name] = max(self.stats["max_ratio"].get(name, 0.0), m)
        if m > 1.0:
            idx = np.unravel_index(np.argmax(ratio), ratio.shape)
            self.failures.append((name, self.stats["steps"] - 1, int((ratio > 1).sum()),
                                  [list(map(int, idx)), float(g[idx]), float(r[idx])]))

    def report(self):
        s = dict(self.stats)
        s["failures"] = self.failures[:10]
        s["ft_exempt_frac"] = s["ft_exempt"] / max(s["taxel_steps"], 1)
        s["noisy_exempt_frac"] = s["noisy_exempt"] / max(s["noisy_taxel_steps"], 1)
        s["taint_steps"] = self.taint_steps
        return s


def run_parity(workload, sim_factory, oracle_factory, env_ids=None, steps=None, outputs=None, threads=8, quant=(0.0, 0.0),
               noise="workload"):
    """Steps the CUDA path over ALL envs of `workload` and the oracle over `env_ids`, comparing each step."""
    import torch
    w = workload
    ids = np.arange(w.E) if env_ids is None else np.asarray(env_ids)
    sim = sim_factory(w)
    orc = oracle_factory(w, ids, threads)
    lay = sim.layout.view()
    nz = w.noise if noise == "workload" else noise
    cmp_ = Comparator(lay, w.physics, nz is not None, lay["radius"], noise=nz)
    cmp_.quant = quant
    outs = outputs or w.outputs
    for s in range(steps or w.steps):
        inp = w.inputs(s)
        g = sim.step(sim.upload(inp))
        torch.cuda.synchronize()
        gpu = {k: v[torch.as_tensor(ids, device=v.device)].cpu().numpy() for k, v in g.items() if k in outs}
        ref = orc.step(w.subset(inp, ids), want=outs)
        cmp_.step(gpu, ref)
    sim.close()
    orc.close()
    return cmp_.report()
