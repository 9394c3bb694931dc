"""Comparator: CUDA path vs oracle, element by element, with the band accounting of DESIGN.md.

Tolerances (BASELINE.json north_star): floats |gpu - ref| <= 1e-6 + 1e-4 |ref|; contact / dead
bit-exact outside a 1e-6 m band around the thresholds.  A band only EXEMPTS an element (and is
counted and reported); tolerances are never loosened.
"""
import numpy as np

ATOL, RTOL, BAND = 1e-6, 1e-4, 1e-6
FACE_BAND = 1e-4        # voxels: trilinear gradient jumps across cell faces
NOISY_TAINT_STEPS = 100  # hysteresis memory of an exempted ft value (0.905^100 < 1e-4)


class Comparator:
    def __init__(self, layout, physics, noise_on, radius):
        self.nbr = np.asarray(layout["nbr"])
        self.eta_on = float(np.float32(physics.get("eta_on", 5e-4)))
        self.eta_off = float(np.float32(physics.get("eta_off", 5e-4)))
        self.radius = np.asarray(radius, np.float64)
        self.noise_on = noise_on
        self.quant = (0.0, 0.0)   # Eq. 25 steps (force, torque); set by the caller when quantisation is on
        self.contact_taint = None
        self.noisy_taint = None
        self.stats = dict(steps=0, contact_band=0, contact_tainted=0, ft_exempt=0, noisy_exempt=0, quant_exempt=0,
                          checked=0, max_ratio={})
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
        # ---- ft: exempt discontinuities of the normal / the d > 0 gate
        phi = ref["aux_phi"]
        active = self.radius[None, :] > 0
        gate = np.abs(self.radius[None, :] - phi) < BAND
        face = (ref["aux_face"] < FACE_BAND) & (d > 0)
        box = (ref["aux_boxgap"] < BAND) & (d > 0)
        ex = (gate | face | box) & active
        st["ft_exempt"] += int(ex.sum())
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
            self.noisy_taint[src] = NOISY_TAINT_STEPS
            t = self.noisy_taint > 0
            spread = t.copy()                      # crosstalk carries a tainted value to its 4 neighbours
            for a in range(4):
                nb = self.nbr[:, a]
                ok = nb >= 0
                spread[:, ok] |= t[:, nb[ok]]
            st["noisy_exempt"] += int(spread.sum())
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
        return s


def run_parity(workload, sim_factory, oracle_factory, env_ids=None, steps=None, outputs=None, threads=8, quant=(0.0, 0.0)):
    """Steps the CUDA path over ALL envs of `workload` and the oracle over `env_ids`, comparing each step."""
    import torch
    w = workload
    ids = np.arange(w.E) if env_ids is None else np.asarray(env_ids)
    sim = sim_factory(w)
    orc = oracle_factory(w, ids, threads)
    lay = sim.layout.view()
    cmp_ = Comparator(lay, w.physics, w.noise is not None, lay["radius"])
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
