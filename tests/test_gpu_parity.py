"""-m gpu: the CUDA path (through the C ABI) against the oracle, element by element."""
import json
import os

import numpy as np
import pytest

from paper_2606_22332_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _sim(w, **kw):
    from paper_2606_22332_b200.binding import TactileSim
    sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=kw.get("physics", w.physics), noise=kw.get("noise", w.noise),
                     outputs=kw.get("outputs", w.outputs))
    sim.set_geometry(w.types, w.params, w.bank, w.voxel)
    return sim


def _orc(w, ids, threads, **kw):
    from oracle import oracle as O
    o = O.Oracle(w.patches, w.T, w.L, w.K, ids, physics=kw.get("physics", w.physics), noise=kw.get("noise", w.noise),
                 threads=threads)
    o.set_geometry(w.types[ids], w.params[ids], w.bank, w.voxel)
    return o


def _assert_ok(rep, max_band_frac=1e-3, max_noisy_frac=0.03):
    """No element outside the tolerance, and the exemptions (bands) stay a small, stated share:
    ft / contact / quantisation bands <= max_band_frac of the checked elements; ft_noisy taxel-steps exempted through
    hysteresis memory and crosstalk spread <= max_noisy_frac of the ft_noisy taxel-steps (printed either way)."""
    print(json.dumps({k: v for k, v in rep.items()}, default=str))
    assert not rep["failures"], rep["failures"]
    n = max(rep["checked"], 1)
    assert rep["ft_exempt"] + rep["contact_tainted"] + rep.get("quant_exempt", 0) <= max(20, max_band_frac * n), rep
    assert rep["noisy_exempt"] <= max(50, max_noisy_frac * rep["noisy_taxel_steps"]), \
        ("noisy_exempt_frac", rep["noisy_exempt_frac"], rep)


def _parity(w, ids=None, steps=None, **kw):
    from parity import run_parity
    nz = kw.get("noise") or {}
    return run_parity(w, lambda ww: _sim(ww, **kw), lambda ww, i, t: _orc(ww, i, t, **kw), ids, steps,
                      kw.get("outputs"), threads=os.cpu_count() or 1,
                      quant=(float(np.float32(nz.get("quant_force", 0.0))), float(np.float32(nz.get("quant_torque", 0.0)))),
                      noise=kw.get("noise", w.noise))


def test_config1_tiny():
    _assert_ok(_parity(W.config(1)))


def test_config2_primitives_small():
    _assert_ok(_parity(W.config(2, n_envs=192)))          # every primitive class, ragged last block


def test_config2_full_size_all_envs():
    """SURVEY 8(d) parity set of config 2: all 4,096 envs x 10 steps, element by element."""
    _assert_ok(_parity(W.config(2)))


def test_config3_sdf_small():
    _assert_ok(_parity(W.config(3, n_envs=96)))


def test_config4_noise_small():
    _assert_ok(_parity(W.config(4, n_envs=48), steps=60))


def test_config4_maxwell_small():
    w = W.config(4, n_envs=32)
    noise = dict(w.noise, hyst_mode="maxwell", beta=0.5, tau=0.05)
    _assert_ok(_parity(w, steps=40, noise=noise))


def test_config5_stress_small():
    _assert_ok(_parity(W.config(5, n_envs=64), steps=50))


def test_uncapped_and_no_velocity():
    w = W.config(2, n_envs=64)
    _assert_ok(_parity(w, steps=3, physics=dict(w.physics, mu=float("inf"))))
    _assert_ok(_parity(w, steps=3, physics=dict(w.physics, use_velocity=0)))
    _assert_ok(_parity(w, steps=3, physics=dict(w.physics, c_e=0.3, march_steps=5, r_prox=0.01)))


def test_config5_full_size_sampled():
    """SURVEY 8(d) parity set of config 5 -- BASELINE size, the launch configuration bench.py times: 20,480 envs x
    1,000 taxels x 200 steps (state carries over: drift grows, hysteresis and Schmitt state evolve over five
    trajectory periods); the oracle recomputes the 16 parity envs {1281 k} (every object class once) element by element."""
    w = W.config(5)
    rep = _parity(w, ids=w.parity_envs(), steps=200)
    _assert_ok(rep)
    assert rep["steps"] == 200 and rep["checked"] > 5e7


def test_config4_full_size_sampled():
    """SURVEY 8(d) parity set of config 4: 16,384 envs x 1,000 taxels x 100 steps, 128 envs (stride 128) recomputed by the
    oracle; ASYM hysteresis as timed, then a second pass with the paper's Maxwell loop (Eq. 29-30, Table 12 values)."""
    w = W.config(4)
    ids = w.parity_envs()
    assert len(ids) == 128
    _assert_ok(_parity(w, ids=ids, steps=100))
    _assert_ok(_parity(w, ids=ids, steps=100, noise=dict(w.noise, hyst_mode="maxwell", beta=0.5, tau=0.05)), max_noisy_frac=0.15)


def test_config5_full_size_optional_knobs_sampled(monkeypatch):
    """BASELINE size with the optional App. A.8 knobs (Table 12 force row + radius noise + a 2 +- 1 step read delay +
    quantisation): the default two-kernel form against the oracle on the 16 parity envs, then fused against two-kernel
    bit for bit on every env (both forms run the same chain code on the same fp32 force/torque values)."""
    import torch
    w = W.config(5)
    noise = dict(w.noise, hyst_mode="maxwell", beta=0.5, tau=0.05, p_dead=0.05, gain_min=0.85, gain_max=1.15,
                 sigma_white_force=5e-3, sigma_white_torque=5e-5, radius_noise=3e-4, read_delay=2, read_jitter=1,
                 quant_force=1e-3, quant_torque=1e-5)
    rep = _parity(w, ids=w.parity_envs(), steps=8, noise=noise)
    _assert_ok(rep, max_band_frac=3e-3)
    outs = {}
    for split in ("0", "1"):
        monkeypatch.setenv("TS_SPLIT", split)
        sim = _sim(w, noise=noise)
        assert sim.launches_per_step() == (3 if split == "1" else 2)   # frames kernel + step kernel (+ noise kernel)
        for s in range(5):
            g = sim.step(sim.upload(w.inputs(s)))
        torch.cuda.synchronize()
        outs[split] = {k: v.clone() for k, v in g.items()}
        sim.close()
    for k in outs["0"]:
        assert torch.equal(outs["0"][k], outs["1"][k]), k


def test_config3_full_size_sampled():
    """SURVEY 8(d) parity set of config 3: 8,192 envs x 500 taxels x 10 steps, 512 envs (stride 16) recomputed."""
    w = W.config(3)
    assert len(w.parity_envs()) == 512
    _assert_ok(_parity(w, ids=w.parity_envs(), steps=10))


def test_more_than_65535_envs():
    """Maximum-size edge: beyond 65,535 envs the step kernel's grid folds the env index over blockIdx.y / blockIdx.z (and
    every other kernel runs a 1-D grid over more than 2^16 envs).  Config 4 (noise on) at 66,000 envs and config 2 (no
    noise) at 70,000 envs; the oracle recomputes the envs around the fold and the last one."""
    w = W.config(4, n_envs=66000)
    ids = np.array([0, 1, 65534, 65535, 65536, 65537, 65999])
    _assert_ok(_parity(w, ids=ids, steps=4))
    w = W.config(2, n_envs=70000)
    ids = np.array([0, 65534, 65535, 65536, 69999])
    _assert_ok(_parity(w, ids=ids, steps=2))


def test_near_the_maximum_env_count():
    """Maximum-size edge: config 5 at 340,000 envs x 1,000 taxels, just under the 32-bit state-index limit of ts_create
    (n_envs * 12 * 1,024 < 2^32, i.e. 349,525 envs; about 45 GB of outputs and state).  Every 32-bit offset in the kernels
    is at its largest here; the oracle recomputes envs at the start, the middle and the very end."""
    w = W.config(5, n_envs=340000)
    ids = np.array([0, 1281, 169999, 170000, 339984, 339999])
    _assert_ok(_parity(w, ids=ids, steps=3))


def test_env_shards_are_bit_identical_to_the_full_run():
    """two contexts over env halves with env_id_base = 0 / E/2 reproduce the full run."""
    import torch
    from paper_2606_22332_b200.sharding import shard_inputs, shard_range
    w = W.config(5, n_envs=32)
    full = _sim(w)
    halves = []
    for r in range(2):
        first, cnt = shard_range(w.E, 2, r)
        from paper_2606_22332_b200.binding import TactileSim
        s = TactileSim(w.patches, w.T, cnt, w.L, w.K, physics=w.physics, noise=w.noise, outputs=w.outputs,
                       env_id_base=first)
        s.set_geometry(w.types[first:first + cnt], w.params[first:first + cnt], w.bank, w.voxel)
        halves.append((first, cnt, s))
    for step in range(4):
        inp = w.inputs(step)
        ref = full.step(full.upload(inp))
        parts = [s.step(s.upload(shard_inputs(inp, first, cnt))) for first, cnt, s in halves]
        torch.cuda.synchronize()
        for k in ref:
            got = torch.cat([p[k] for p in parts])
            assert torch.equal(got, ref[k]), (k, step)


def test_reset_redraws_dead_mask_and_zeroes_state():
    import torch
    w = W.config(4, n_envs=16)
    sim = _sim(w)
    inp = sim.upload(w.inputs(0))
    a = {k: v.clone() for k, v in sim.step(inp).items()}
    for s in range(1, 4):
        sim.step(sim.upload(w.inputs(s)))
    mask = torch.zeros(w.E, dtype=torch.uint8, device="cuda")
    mask[::2] = 1
    sim.reset(mask)
    # a fresh context stepped to the same global step count has the same counters for the untouched envs
    b = sim.step(inp)
    torch.cuda.synchronize()
    dead_a, dead_b = a["dead"].bool(), b["dead"].bool()
    assert torch.equal(dead_a[1::2], dead_b[1::2])            # untouched envs keep their episode's mask
    assert not torch.equal(dead_a[::2], dead_b[::2])           # reset envs drew a new one (episode + 1)
    frac = dead_b.float().mean().item()
    assert 0.01 < frac < 0.03
    assert torch.all(b["ft_noisy"][dead_b] == 0) and torch.all(b["contact"][dead_b] == 0)
    # reset envs restart from zero state: with the same inputs the clean outputs equal step 0's
    assert torch.equal(a["ft"][::2], b["ft"][::2]) and torch.equal(a["depth"], b["depth"])


def test_edge_shapes():
    """One env; a layout that is all fillers; march_steps = 0; outputs subset."""
    import torch
    from paper_2606_22332_b200.binding import TactileSim
    w = W.config(2, n_envs=1)
    _assert_ok(_parity(w, steps=2))
    sim = TactileSim(w.patches, w.T, 1, w.L, 1, physics=dict(w.physics, march_steps=0), outputs=("prox", "depth"),
                     link_mask=np.zeros(w.L, np.uint8))
    sim.set_geometry(w.types, w.params)
    out = sim.step(sim.upload(w.inputs(0)))
    torch.cuda.synchronize()
    assert torch.all(out["prox"] == 0) and torch.all(out["depth"] == 0)   # every taxel filtered out: fillers are 0
    sim2 = TactileSim(w.patches, w.T, 1, w.L, 1, physics=dict(w.physics, march_steps=0), outputs=("prox",))
    sim2.set_geometry(w.types, w.params)
    out2 = sim2.step(sim2.upload(w.inputs(0)))
    torch.cuda.synchronize()
    act = torch.from_numpy(sim2.layout.view()["radius"] > 0).cuda()
    assert torch.allclose(out2["prox"][0][act], torch.full_like(out2["prox"][0][act], 0.02))  # K_m = 0: t = 0, P = r_prox


def test_remaining_noise_knobs(monkeypatch):
    """App. A.8 knobs beyond the four of configs 4-5 (R1-R4): bias, white noise, quantisation (Eq. 25),
    per-episode gain (Eq. 27), stuck readout of dead taxels (Eq. 28), with both hysteresis modes and over a reset.
    With such a knob set the ctx defaults to the two-kernel form; TS_SPLIT=0 forces the fused variant (tested first)."""
    w = W.config(5, n_envs=48)
    monkeypatch.setenv("TS_SPLIT", "0")
    ext = dict(sigma_white_force=2e-3, sigma_white_torque=2e-5, bias_force=0.02, bias_torque=-3e-4, gain_min=0.9,
               gain_max=1.1, stuck_min_force=-0.5, stuck_max_force=0.5, stuck_min_torque=-5e-3, stuck_max_torque=5e-3,
               p_dead=0.05)
    _assert_ok(_parity(w, steps=30, noise=dict(w.noise, **ext)))
    _assert_ok(_parity(w, steps=20, noise=dict(w.noise, hyst_mode="maxwell", beta=0.5, tau=0.05, **ext)))
    # quantisation: 1 mN / 10 uN m steps; boundary hits are exempted and counted by the comparator
    rep = _parity(w, steps=20, noise=dict(w.noise, quant_force=1e-3, quant_torque=1e-5, **ext))
    _assert_ok(rep, max_band_frac=3e-3)
    assert rep["quant_exempt"] < 3e-3 * rep["checked"]
    # each knob alone (the others off), in the default (two-kernel) form
    monkeypatch.delenv("TS_SPLIT")
    for one in (dict(bias_force=0.1), dict(sigma_white_force=1e-3), dict(gain_min=0.5, gain_max=0.6),
                dict(stuck_min_force=1.0, stuck_max_force=1.0), dict(quant_torque=1e-5)):
        _assert_ok(_parity(w, steps=6, noise=dict(w.noise, **one)), max_band_frac=3e-3)


def test_remaining_noise_knobs_reset_and_split(monkeypatch):
    """Gain and stuck values are per episode: the same context after ts_reset must follow the oracle after reset;
    the split (geometry + noise kernel) variant computes the same."""
    import torch
    from oracle import oracle as O
    from parity import Comparator
    w = W.config(4, n_envs=24)
    noise = dict(w.noise, gain_min=0.8, gain_max=1.2, stuck_min_force=0.2, stuck_max_force=0.4, bias_torque=1e-4, p_dead=0.1)
    for split in ("0", "1"):
        monkeypatch.setenv("TS_SPLIT", split)
        sim = _sim(w, noise=noise)
        orc = _orc(w, np.arange(w.E), os.cpu_count() or 1, noise=noise)
        lay = sim.layout.view()
        cmp_ = Comparator(lay, w.physics, True, lay["radius"], noise=noise)
        for s in range(12):
            if s == 6:
                sim.reset()
                orc.reset()
            inp = w.inputs(s)
            g = sim.step(sim.upload(inp))
            torch.cuda.synchronize()
            cmp_.step({k: v.cpu().numpy() for k, v in g.items()}, orc.step(inp, want=w.outputs))
        rep = cmp_.report()
        _assert_ok(rep)
        assert sim.launches_per_step() == (3 if split == "1" else 2)   # frames kernel + step kernel (+ noise kernel)
        sim.close()


def test_radius_noise(monkeypatch):
    """Eq. 26 (R8): ft_noisy starts from the readout at the perturbed radius; the clean outputs keep R_j.
    rho = 0.5 mm of R = 2 mm, and rho = 3 mm (exercises the max(0, .) clamp); alone, with the other knobs, over a
    reset, and in the two-kernel variant."""
    import torch
    from parity import Comparator
    w = W.config(5, n_envs=48)
    _assert_ok(_parity(w, steps=20, noise=dict(w.noise, radius_noise=5e-4)))
    _assert_ok(_parity(w, steps=10, noise=dict(w.noise, radius_noise=3e-3, hyst_mode="maxwell", beta=0.5, tau=0.05)))
    # Gaussian crosstalk spreads an exempted taxel over its 7 x 7 support instead of 5 taxels: larger exempt share
    _assert_ok(_parity(w, steps=10, noise=dict(w.noise, radius_noise=5e-4, gain_min=0.9, gain_max=1.1, bias_force=0.01,
                                               xtalk_sigma=0.8, chi=0.3)), max_noisy_frac=0.10)
    _assert_ok(_parity(W.config(2, n_envs=96), steps=8, noise=dict(noise_enable=1, seed=5, radius_noise=1e-3)))
    for split in ("0", "1"):
        monkeypatch.setenv("TS_SPLIT", split)
        for outputs in (w.outputs, [o for o in w.outputs if o != "ft"]):
            noise = dict(w.noise, radius_noise=5e-4)
            sim = _sim(w, noise=noise, outputs=outputs)
            orc = _orc(w, np.arange(w.E), os.cpu_count() or 1, noise=noise)
            lay = sim.layout.view()
            cmp_ = Comparator(lay, w.physics, True, lay["radius"], noise=noise)
            for s in range(8):
                if s == 4:
                    sim.reset()
                    orc.reset()
                inp = w.inputs(s)
                g = sim.step(sim.upload(inp))
                torch.cuda.synchronize()
                cmp_.step({k: v.cpu().numpy() for k, v in g.items() if k in outputs}, orc.step(inp, want=outputs))
            _assert_ok(cmp_.report())
            sim.close()


def test_read_delay(monkeypatch):
    """Eq. 25 read delay with jitter (R9): ring of past post-crosstalk fields, per-env step counters
    (a partial reset puts the envs at different ring positions), both hysteresis modes, fused and two-kernel."""
    import torch
    from parity import Comparator
    w = W.config(5, n_envs=48)
    _assert_ok(_parity(w, steps=16, noise=dict(w.noise, read_delay=3)))
    _assert_ok(_parity(w, steps=24, noise=dict(w.noise, read_delay=2, read_jitter=2, hyst_mode="maxwell", beta=0.5, tau=0.05,
                                               bias_force=0.01, radius_noise=3e-4)))
    _assert_ok(_parity(w, steps=10, noise=dict(w.noise, read_delay=0, read_jitter=1)))
    mask = (np.arange(w.E) % 3 == 0).astype(np.uint8)
    for split in ("0", "1"):
        monkeypatch.setenv("TS_SPLIT", split)
        noise = dict(w.noise, read_delay=2, read_jitter=1)
        sim = _sim(w, noise=noise)
        orc = _orc(w, np.arange(w.E), os.cpu_count() or 1, noise=noise)
        lay = sim.layout.view()
        cmp_ = Comparator(lay, w.physics, True, lay["radius"], noise=noise)
        for s in range(14):
            if s == 5:
                sim.reset(torch.from_numpy(mask).cuda())
                orc.reset(mask)
            if s == 9:
                sim.reset()
                orc.reset()
            inp = w.inputs(s)
            g = sim.step(sim.upload(inp))
            torch.cuda.synchronize()
            cmp_.step({k: v.cpu().numpy() for k, v in g.items()}, orc.step(inp, want=w.outputs))
        _assert_ok(cmp_.report())
        sim.close()


def test_table12_force_row():
    """The paper's "noisy condition" for force / force_torque probes (Table 12): sigma = 5e-3 N white noise,
    p_dead = 0.05, gain in [0.85, 1.15], Maxwell hysteresis (0.5, 0.05 s); plus the table's probe-radius noise of the
    depth row (3e-4 m) and the Schmitt release threshold 2e-4 m of the bool row."""
    w = W.config(4, n_envs=48)
    noise = dict(noise_enable=1, seed=2606, hyst_mode="maxwell", beta=0.5, tau=0.05, p_dead=0.05, gain_min=0.85, gain_max=1.15,
                 sigma_white_force=5e-3, sigma_white_torque=5e-5, radius_noise=3e-4)
    assert abs(w.physics["eta_off"] - 2e-4) < 1e-12
    _assert_ok(_parity(w, steps=40, noise=noise))


def test_gaussian_crosstalk(monkeypatch):
    """Eq. 11 / 31 with the paper's Gaussian kernel G_sigma (R7) instead of the 4-neighbour stencil, on the
    8x8 / 6x8 / 5x8 patches of config 5 (borders matter), alone and with the other knobs, fused and split."""
    w = W.config(5, n_envs=48)
    monkeypatch.setenv("TS_SPLIT", "0")
    # the taint of an exempted taxel covers the kernel's (2r+1)^2 support (r = ceil(3 sigma)): larger exempt share
    _assert_ok(_parity(w, steps=20, noise=dict(w.noise, chi=0.3, xtalk_sigma=0.8)), max_noisy_frac=0.10)
    _assert_ok(_parity(w, steps=10, noise=dict(w.noise, chi=1.0, xtalk_sigma=1.3, hyst_mode="maxwell", beta=0.5, tau=0.05)),
               max_noisy_frac=0.20)
    _assert_ok(_parity(w, steps=10, noise=dict(w.noise, chi=0.05, xtalk_sigma=0.3, bias_force=0.01, gain_min=0.9, gain_max=1.1)),
               max_noisy_frac=0.05)
    monkeypatch.setenv("TS_SPLIT", "1")
    _assert_ok(_parity(w, steps=10, noise=dict(w.noise, chi=0.3, xtalk_sigma=0.8)), max_noisy_frac=0.10)


def test_two_objects_per_env():
    """K = 2 (Eq. 2's max over geometries, Q3): every env holds its config-2 primitive plus a second object (a sphere
    or an SDF star grid) a few centimetres away, so some links touch one, some the other; exercises the K > 1 kernels
    (frames per (patch, object), winner selection, march over min_k phi_k) against the oracle."""
    import torch
    from paper_2606_22332_b200.binding import TactileSim
    from oracle import oracle as O
    from parity import Comparator
    w = W.config(2, n_envs=96)
    w3 = W.config(3, n_envs=1)                                  # its 64^3 star grid serves as the bank
    E, K = w.E, 2
    rng = np.random.default_rng(5)
    types = np.zeros((E, K), np.int32); params = np.zeros((E, K, 4), np.float32)
    types[:, 0] = w.types[:, 0]; params[:, 0] = w.params[:, 0]
    types[:, 1] = np.where(np.arange(E) % 2 == 0, 1, 4)         # sphere / grid 0
    params[np.arange(E) % 2 == 0, 1, 0] = 0.025
    noise = dict(noise_enable=1, seed=11, sigma_rw_force=1e-3, sigma_rw_torque=1e-5, hyst_mode="asym", alpha_load=0.8,
                 alpha_unload=0.5, p_dead=0.02, chi=0.05)
    outs = ("contact", "depth", "ft", "marker", "prox", "ft_noisy", "dead")
    sim = TactileSim(w.patches, w.T, E, w.L, K, physics=w.physics, noise=noise, outputs=outs)
    sim.set_geometry(types, params, w3.bank, w3.voxel)
    orc = O.Oracle(w.patches, w.T, w.L, K, np.arange(E), physics=w.physics, noise=noise, threads=os.cpu_count() or 1)
    orc.set_geometry(types, params, w3.bank, w3.voxel)
    lay = sim.layout.view()
    cmp_ = Comparator(lay, w.physics, True, lay["radius"], noise=noise)
    off = rng.uniform(-0.03, 0.03, (E, 1, 3)).astype(np.float32)
    win = np.zeros(2, np.int64)
    for s in range(6):
        base = w.inputs(s)
        inp = dict(base)
        for k in ("obj_pos", "obj_quat", "obj_linvel", "obj_angvel"):
            second = base[k].copy()
            if k == "obj_pos":
                second = second + off                          # the second object sits a few cm from the first
            if k == "obj_linvel":
                second = -second
            inp[k] = np.ascontiguousarray(np.concatenate([base[k], second], axis=1))
        g = sim.step(sim.upload(inp))
        torch.cuda.synchronize()
        ref = orc.step(inp, want=outs)
        cmp_.step({k: v.cpu().numpy() for k, v in g.items()}, ref)
    rep = cmp_.report()
    _assert_ok(rep)                                             # winner ties (|phi_k - phi_k'| < 1e-6) are a counted band
    assert rep["max_ratio"]["prox"] <= 1.0 and rep["checked"] > 1e6


def test_noisy_scalar_readouts():
    """SURVEY 8(f-1) / DESIGN.md R10: noisy depth, prox and marker readouts (Table 3 P:346-359 gives them every knob of
    App. A.8 except crosstalk) with the Table 12 values and beyond: white noise, drift, bias, quantisation,
    gain, dead probes with stuck values, both hysteresis modes, the Eq. 26 radius for the depth readout, the read delay
    with jitter, over a reset, with and without the clean outputs requested next to them."""
    import torch
    from oracle import oracle as O
    from parity import Comparator
    from paper_2606_22332_b200.binding import TactileSim
    w = W.config(5, n_envs=48)
    t12 = dict(sigma_white_depth=2e-4, sigma_white_prox=1e-2, sigma_rw_prox=1e-3, quant_prox=1e-2, sigma_white_marker=1e-4,
               sigma_rw_marker=1e-5, quant_marker=1e-4, p_dead=0.05, gain_min=0.85, gain_max=1.15, radius_noise=3e-4)
    more = dict(sigma_rw_depth=1e-5, bias_depth=1e-4, bias_prox=-1e-3, bias_marker=2e-3, quant_depth=5e-5, stuck_min_depth=1e-3,
                stuck_max_depth=2e-3, stuck_min_prox=0.0, stuck_max_prox=0.02, stuck_min_marker=-0.1, stuck_max_marker=0.1)
    full = w.outputs + ("depth_noisy", "prox_noisy", "marker_noisy")
    only = ("contact", "ft", "ft_noisy", "dead", "depth_noisy", "prox_noisy", "marker_noisy")   # clean inputs from scratch buffers
    cases = ((dict(w.noise, hyst_mode="maxwell", beta=0.5, tau=0.05, **t12), full),
             (dict(w.noise, **t12, **more), full),
             (dict(w.noise, hyst_mode="off", **more), only),
             # Eq. 25 read delay with jitter on every readout (Table 3): rings of 3 slots, delays 0..3 steps
             (dict(w.noise, read_delay=2, read_jitter=1, **t12, **more), full),
             (dict(w.noise, hyst_mode="maxwell", beta=0.5, tau=0.05, read_delay=1, read_jitter=1, **t12), only))
    for noise, outs in cases:
        sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=w.physics, noise=noise, outputs=outs)
        sim.set_geometry(w.types, w.params, w.bank, w.voxel)
        assert sim.launches_per_step() in (3, 4)
        orc = O.Oracle(w.patches, w.T, w.L, w.K, np.arange(w.E), physics=w.physics, noise=noise, threads=os.cpu_count() or 1)
        orc.set_geometry(w.types, w.params, w.bank, w.voxel)
        lay = sim.layout.view()
        cmp_ = Comparator(lay, w.physics, True, lay["radius"], noise=noise)
        cmp_.quant = (float(np.float32(noise.get("quant_force", 0.0))), float(np.float32(noise.get("quant_torque", 0.0))))
        for s in range(24):
            if s == 12:
                mask = (np.arange(w.E) % 3 == 0).astype(np.uint8)
                sim.reset(torch.from_numpy(mask).cuda())
                orc.reset(mask)
            inp = w.inputs(s)
            g = sim.step(sim.upload(inp))
            torch.cuda.synchronize()
            cmp_.step({k: v.cpu().numpy() for k, v in g.items()}, orc.step(inp, want=tuple(outs) + ("depth",)))   # the bands need depth
        rep = cmp_.report()
        _assert_ok(rep, max_band_frac=3e-3, max_noisy_frac=0.05)
        assert rep["sn_checked"] > 1e6 and rep["sn_exempt"] <= 5e-3 * rep["sn_checked"], rep
        for k in ("depth_noisy", "prox_noisy", "marker_noisy"):
            assert rep["max_ratio"][k] <= 1.0
        sim.close()


def test_point_cloud_proximity_taxel():
    """the paper's ProximityTaxel (App. A.6, Eq. 12-17) on tracked surface point clouds (N_pc = 5,000 per
    object, R_j = 10 mm, k = 300, k_s = 10, density 100): uniform-grid neighbour query on the GPU against the
    oracle's brute-force sum over every point.  Config-5 scene: star objects are tracked, primitives are not (zeros)."""
    import torch
    from oracle import oracle as O
    from paper_2606_22332_b200.binding import TactileSim
    from parity import ATOL, RTOL
    w = W.config(5, n_envs=32)
    pts, cid = W.point_cloud_bank(w, 5000)
    outs = ("depth", "proxpc")
    sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=w.physics, outputs=outs)
    sim.set_geometry(w.types, w.params, w.bank, w.voxel)
    sim.set_pointclouds(pts, cid)
    orc = O.Oracle(w.patches, w.T, w.L, w.K, np.arange(w.E), physics=w.physics, threads=os.cpu_count() or 1)
    orc.set_geometry(w.types, w.params, w.bank, w.voxel)
    orc.set_pointclouds(pts, cid)
    worst, nz = 0.0, 0
    for s in (0, 7, 19):
        inp = w.inputs(s)
        g = sim.step(sim.upload(inp))["proxpc"].cpu().numpy().astype(np.float64)
        r = orc.step(inp, want=outs, aux=False)["proxpc"]
        ratio = np.abs(g - r) / (ATOL + RTOL * np.abs(r))
        worst = max(worst, float(ratio.max()))
        nz += int((np.abs(r[..., 2]) > 1e-3).sum())
        assert not g[cid[:, 0] < 0].any()                                    # untracked objects: exactly zero
    print(json.dumps({"proxpc_max_ratio": worst, "taxels_with_force": nz}))
    assert worst <= 1.0 and nz > 20000
    sim.close()


def test_elastomer_shear_history():
    """ElastomerTaxel shear history (App. A.7 Eq. 22-23, constants P:304, N_pc = 1,000 tracked points per
    object): anchors per (env, patch, tracked point) carried over 40 steps of the config-5 trajectories (objects slide
    over the pads), a masked reset in the middle, shear added to the dilation markers; element-wise against the oracle."""
    import torch
    from oracle import oracle as O
    from parity import Comparator
    from paper_2606_22332_b200.binding import TactileSim
    w = W.config(5, n_envs=32)
    pts, cid = W.point_cloud_bank(w, 1000)
    phys = dict(w.physics, shear_enable=1)
    outs = ("contact", "depth", "ft", "marker", "prox")
    sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=phys, outputs=outs)
    sim.set_geometry(w.types, w.params, w.bank, w.voxel)
    sim.set_pointclouds(pts, cid)
    plain = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=w.physics, outputs=outs)
    plain.set_geometry(w.types, w.params, w.bank, w.voxel)
    orc = O.Oracle(w.patches, w.T, w.L, w.K, np.arange(w.E), physics=phys, threads=os.cpu_count() or 1)
    orc.set_geometry(w.types, w.params, w.bank, w.voxel)
    orc.set_pointclouds(pts, cid)
    lay = sim.layout.view()
    cmp_ = Comparator(lay, phys, False, lay["radius"])
    moved = 0
    for s in range(40):
        if s == 20:
            mask = (np.arange(w.E) % 2 == 0).astype(np.uint8)
            sim.reset(torch.from_numpy(mask).cuda())
            orc.reset(mask)
        inp = w.inputs(s)
        x = sim.upload(inp)
        g = sim.step(x)
        d = plain.step(x)
        torch.cuda.synchronize()
        cmp_.step({k: v.cpu().numpy() for k, v in g.items()}, orc.step(inp, want=outs))
        moved += int(((g["marker"] - d["marker"]).abs() > 1e-4).sum().item())
    rep = cmp_.report()
    _assert_ok(rep)
    assert rep["max_ratio"]["marker"] <= 1.0 and moved > 5000, (rep["max_ratio"], moved)    # the shear term really acts
    sim.close(); plain.close()


def test_shear_dense_contact_drains_the_queue():
    """A flat, densely sampled face (4,000 tracked points over one 20 x 20 mm pad, all anchored and penetrating) is far more
    than the shear kernel's 512-entry shared-memory queue holds at once: the kernel must drain it in passes and still
    equal the oracle's plain sum over every anchored point (Eq. 22)."""
    import torch
    from oracle import oracle as O
    from paper_2606_22332_b200.binding import TactileSim
    from parity import ATOL, RTOL
    patch = dict(link=0, origin=(0, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=0.02, size_v=0.02, nu=8, nv=8, radius=2e-3,
                 marker_nu=7, marker_nv=7)
    E, N = 3, 4000
    rng = np.random.default_rng(77)
    pts = np.zeros((1, N, 3), np.float32)
    pts[0, :, :2] = rng.uniform(-0.012, 0.012, (N, 2))          # a flat face a little wider than the pad
    cid = np.zeros((E, 1), np.int32)
    phys = dict(shear_enable=1)
    sim = TactileSim([patch], 64, E, 1, 1, physics=phys, outputs=("marker",))
    sim.set_geometry(np.zeros((E, 1), np.int32), np.zeros((E, 1, 4), np.float32))
    sim.set_pointclouds(pts, cid)
    orc = O.Oracle([patch], 64, 1, 1, np.arange(E), physics=phys)
    orc.set_geometry(np.zeros((E, 1), np.int32), np.zeros((E, 1, 4), np.float32))
    orc.set_pointclouds(pts, cid)
    z = lambda n: np.zeros((E, 1, n), np.float32)
    q = z(4); q[..., 0] = 1
    worst, peak = 0.0, 0.0
    for s in range(4):
        op = z(3)
        op[:, 0, 2] = -0.001                                    # 1 mm into the pad
        op[:, 0, 0] = 0.0003 * s * (1 + np.arange(E))           # each env slides at its own rate
        inp = dict(link_pos=z(3), link_quat=q, link_linvel=z(3), link_angvel=z(3), obj_pos=op, obj_quat=q, obj_linvel=z(3), obj_angvel=z(3))
        g = sim.step(sim.upload(inp))["marker"].cpu().numpy().astype(np.float64)
        r = orc.step(inp, want=("marker",), aux=False)["marker"]
        worst = max(worst, float((np.abs(g - r) / (ATOL + RTOL * np.abs(r))).max()))
        peak = max(peak, float(np.abs(r).max()))
    print(json.dumps({"shear_dense_max_ratio": worst, "peak_marker_m": peak}))
    assert worst <= 1.0 and peak > 1e-2                         # thousands of anchored points really contribute
    sim.close()


def test_raycast_depth_backend():
    """the raycast contact-depth backend (App. A.1) on triangle meshes: BVH walk on the GPU against
    the oracle's brute force over every triangle.  Config-5 scene with 1,280-triangle star meshes; depth element-wise,
    the face normal wherever the winning triangle is unique (margin to the best triangle with another normal > 1e-6 m;
    two triangles sharing the closest edge tie exactly and either normal is valid)."""
    import torch
    from oracle import oracle as O
    from paper_2606_22332_b200.binding import TactileSim
    from parity import ATOL, RTOL
    w = W.config(5, n_envs=32)
    meshes, mid = W.mesh_bank(w, 3)
    outs = ("depth", "depth_rc", "nrm_rc")
    sim = TactileSim(w.patches, w.T, w.E, w.L, w.K, physics=w.physics, outputs=outs)
    sim.set_geometry(w.types, w.params, w.bank, w.voxel)
    sim.set_meshes(meshes, mid)
    orc = O.Oracle(w.patches, w.T, w.L, w.K, np.arange(w.E), physics=w.physics, threads=os.cpu_count() or 1)
    orc.set_geometry(w.types, w.params, w.bank, w.voxel)
    orc.set_meshes(meshes, mid)
    n_touch = n_nrm = 0
    for s in (0, 11):
        inp = w.inputs(s)
        g = sim.step(sim.upload(inp))
        torch.cuda.synchronize()
        r = orc.step(inp, want=outs, aux=False)
        gd, gn = g["depth_rc"].cpu().numpy().astype(np.float64), g["nrm_rc"].cpu().numpy().astype(np.float64)
        ratio = np.abs(gd - r["depth_rc"]) / (ATOL + RTOL * np.abs(r["depth_rc"]))
        assert ratio.max() <= 1.0, ratio.max()
        unique = (r["depth_rc"] > 2e-6) & (r["aux_rc_gap"] > 2e-6)
        assert np.abs(gn[unique] - r["nrm_rc"][unique]).max() < 2e-5
        touch = r["depth_rc"] > 0
        # where the normal is not unique it must still be a unit vector (some triangle's face normal)
        assert np.abs(np.linalg.norm(gn[gd > 0], axis=-1) - 1).max() < 1e-5 and not gn[gd == 0].any()
        assert not gd[mid[:, 0] < 0].any()
        n_touch += int(touch.sum()); n_nrm += int(unique.sum())
        # the two backends agree to the mesh's chord error where the probe centre is outside ("equivalent depths
        # to leading order for smooth meshes")
        sdf = g["depth"].cpu().numpy()
        both = touch & (sdf > 0) & (sdf < 1.5e-3)
        assert np.abs(gd[both] - sdf[both]).max() < 4e-4
    print(json.dumps({"raycast_touching": n_touch, "normals_checked": n_nrm}))
    assert n_touch > 3000 and n_nrm > 0.8 * n_touch
    sim.close()
