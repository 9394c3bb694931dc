"""Pins for the oracle's noisy readouts of the scalar sensors (reading R10; Table 3, Eq. 25-30
P:310-338): ContactDepth -> depth_noisy, Proximity -> prox_noisy, Elastomer markers -> marker_noisy.

Chain per channel: x = gamma * clean -> hysteresis (Eq. 29-30 / ASYM) -> y = h + b + sigma_w z_w + D, D <- D + sigma_rw z_rw
-> quantize(y, q) -> dead probes read their stuck value.  No crosstalk (Table 3).  Draw layout:
  taxel j:   stream 10, step n: Box-Muller(words 0,1) -> (z_rw, z_w) of depth, (words 2,3) -> (z_rw, z_w) of prox;
             stream 11, n = 0: word 0 / 1 -> stuck value of depth / prox; gain and dead are the taxel's (streams 3 / 2)
  marker m:  probe word 0x80000000 + m; stream 0, step n: (0,1) -> z_rw of channels 0, 1; (2,3) -> z_rw of channel 2 and
             z_w of channel 0; stream 1: (0,1) -> z_w of channels 1, 2; stream 2 dead, 3 gain, 4 stuck (words 0-2), n = 0
Every draw is rebuilt here from `O.philox` (pinned by the Random123 vectors) with the uniform / Box-Muller rule written
out, and the chain by its closed forms (exact bias shift, Maxwell step response, quantisation lattice, Eq. 26 depth).
"""
import math

import numpy as np

from oracle import oracle as O

SEED = 0x0123456789ABCDEF
KEY = (SEED & 0xFFFFFFFF, SEED >> 32)
ENVS = np.array([3, 70001])
R_TAX = 2.0e-3


def _patch(nu, nv, m=0):
    return dict(link=0, origin=(0, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=0.0025 * nu, size_v=0.0025 * nv, nu=nu,
                nv=nv, radius=R_TAX, marker_nu=m, marker_nv=m)


def _oracle(noise, nu=3, nv=2, m=0):
    o = O.Oracle([_patch(nu, nv, m)], nu * nv, 1, 1, ENVS, noise=dict(dict(noise_enable=1, seed=SEED, hyst_mode="off"), **noise))
    E = len(ENVS)
    o.set_geometry(np.ones((E, 1), np.int32), np.full((E, 1, 4), 0.030, np.float32))
    return o


def _inputs(z):
    E = len(ENVS)
    return dict(link_pos=np.tile(np.array([0, 0, z], np.float32), (E, 1, 1)),
                link_quat=np.tile(np.array([1, 0, 0, 0], np.float32), (E, 1, 1)),
                link_linvel=np.zeros((E, 1, 3), np.float32), link_angvel=np.zeros((E, 1, 3), np.float32),
                obj_pos=np.zeros((E, 1, 3), np.float32), obj_quat=np.tile(np.array([1, 0, 0, 0], np.float32), (E, 1, 1)),
                obj_linvel=np.zeros((E, 1, 3), np.float32), obj_angvel=np.zeros((E, 1, 3), np.float32))


def _u(w):
    return (2.0 * (int(w) >> 9) + 1.0) / 16777216.0


def _bm(wa, wb):
    r = math.sqrt(-2.0 * math.log(_u(wa)))
    return r * math.cos(2.0 * math.pi * _u(wb)), r * math.sin(2.0 * math.pi * _u(wb))


WANT = ("depth", "prox", "marker", "depth_noisy", "prox_noisy", "marker_noisy", "dead")


def test_depth_and_prox_draws_known_answers():
    sw_d, sr_d, sw_p, sr_p = (float(np.float32(v)) for v in (2e-4, 1e-5, 1e-2, 1e-3))
    o = _oracle(dict(sigma_white_depth=2e-4, sigma_rw_depth=1e-5, sigma_white_prox=1e-2, sigma_rw_prox=1e-3))
    x = _inputs(-0.0315)                               # centre taxels 0.5 mm inside the sphere: depth and prox are non-zero
    for ep in (0, 1):
        Dd = np.zeros((2, 6)); Dp = np.zeros((2, 6))
        for n in range(3):
            r = o.step(x, want=WANT)
            assert (r["depth"] > 0).any() and (r["prox"] > 0).all()
            for e, env in enumerate(ENVS):
                for j in range(6):
                    w = O.philox((int(env), j, n, (ep << 4) | 10), KEY)
                    zd, zp = _bm(w[0], w[1]), _bm(w[2], w[3])
                    Dd[e, j] += sr_d * zd[0]; Dp[e, j] += sr_p * zp[0]
                    np.testing.assert_allclose(r["depth_noisy"][e, j], r["depth"][e, j] + sw_d * zd[1] + Dd[e, j], rtol=1e-12, atol=1e-18)
                    np.testing.assert_allclose(r["prox_noisy"][e, j], r["prox"][e, j] + sw_p * zp[1] + Dp[e, j], rtol=1e-12, atol=1e-18)
        o.reset()


def test_marker_draws_dead_gain_stuck_known_answers():
    p_dead = 0.6
    sw, sr = float(np.float32(1e-4)), float(np.float32(1e-5))
    gmin, gmax, lo, hi = (float(np.float32(v)) for v in (0.85, 1.15, -0.3, 0.2))
    o = _oracle(dict(sigma_white_marker=1e-4, sigma_rw_marker=1e-5, p_dead=p_dead, gain_min=0.85, gain_max=1.15,
                     stuck_min_marker=-0.3, stuck_max_marker=0.2), nu=4, nv=4, m=3)
    x = _inputs(-0.0295)                               # 0.5 mm inside the sphere: the markers move
    thr = int(math.floor(float(np.float32(p_dead)) * 4294967296.0))
    for ep in (0, 1):
        D = np.zeros((2, 9, 3))
        n_dead = 0
        for n in range(3):
            r = o.step(x, want=WANT)
            assert np.abs(r["marker"]).max() > 1e-3
            for e, env in enumerate(ENVS):
                for m in range(9):
                    probe = 0x80000000 + m
                    w0 = O.philox((int(env), probe, n, (ep << 4) | 0), KEY)
                    w1 = O.philox((int(env), probe, n, (ep << 4) | 1), KEY)
                    zr01, zr2w0, zw12 = _bm(w0[0], w0[1]), _bm(w0[2], w0[3]), _bm(w1[0], w1[1])
                    z_rw = (zr01[0], zr01[1], zr2w0[0]); z_w = (zr2w0[1], zw12[0], zw12[1])
                    dead = int(O.philox((int(env), probe, 0, (ep << 4) | 2), KEY)[0]) < thr
                    g = gmin + (gmax - gmin) * _u(O.philox((int(env), probe, 0, (ep << 4) | 3), KEY)[0])
                    ws = O.philox((int(env), probe, 0, (ep << 4) | 4), KEY)
                    for c in range(3):
                        D[e, m, c] += sr * z_rw[c]
                        want = lo + (hi - lo) * _u(ws[c]) if dead else g * r["marker"][e, m, c] + sw * z_w[c] + D[e, m, c]
                        np.testing.assert_allclose(r["marker_noisy"][e, m, c], want, rtol=1e-12, atol=1e-18)
                    n_dead += dead
        assert 6 < n_dead < 3 * 18 - 6                  # both outcomes occur
        o.reset()


def test_stuck_values_and_shared_probe_draws_of_depth_and_prox():
    # a dead taxel's depth / prox read their own stuck values (stream 11 words 0 / 1); gain and dead are the taxel's
    gmin, gmax = float(np.float32(0.8)), float(np.float32(1.2))
    o = _oracle(dict(p_dead=0.5, gain_min=0.8, gain_max=1.2, stuck_min_depth=1e-3, stuck_max_depth=2e-3, stuck_min_prox=0.5,
                     stuck_max_prox=0.6), nu=4, nv=4)
    x = _inputs(-0.0315)
    for ep in (0, 1):
        r = o.step(x, want=WANT)
        for e, env in enumerate(ENVS):
            for j in range(16):
                ws = O.philox((int(env), j, 0, (ep << 4) | 11), KEY)
                g = gmin + (gmax - gmin) * _u(O.philox((int(env), j, 0, (ep << 4) | 3), KEY)[0])
                if r["dead"][e, j]:
                    np.testing.assert_allclose(r["depth_noisy"][e, j], float(np.float32(1e-3)) + (float(np.float32(2e-3)) - float(np.float32(1e-3))) * _u(ws[0]), rtol=1e-12)
                    np.testing.assert_allclose(r["prox_noisy"][e, j], float(np.float32(0.5)) + (float(np.float32(0.6)) - float(np.float32(0.5))) * _u(ws[1]), rtol=1e-12)
                else:
                    np.testing.assert_allclose(r["depth_noisy"][e, j], g * r["depth"][e, j], rtol=1e-12, atol=1e-18)
                    np.testing.assert_allclose(r["prox_noisy"][e, j], g * r["prox"][e, j], rtol=1e-12, atol=1e-18)
        assert 4 < r["dead"].sum() < 28
        o.reset()


def test_bias_quantisation_and_maxwell_on_scalar_channels():
    # bias: exact shift; quantize: multiples of q within q/2; Maxwell step response X (1 + beta e^{-k dt / tau}) (P13)
    o = _oracle(dict(bias_depth=3e-4, bias_prox=-2e-3, bias_marker=0.01), nu=4, nv=4, m=3)
    x = _inputs(-0.0295)
    r = o.step(x, want=WANT)
    np.testing.assert_allclose(r["depth_noisy"] - r["depth"], float(np.float32(3e-4)), rtol=0, atol=1e-15)
    np.testing.assert_allclose(r["prox_noisy"] - r["prox"], float(np.float32(-2e-3)), rtol=0, atol=1e-15)
    np.testing.assert_allclose(r["marker_noisy"] - r["marker"], float(np.float32(0.01)), rtol=0, atol=1e-15)
    q = float(np.float32(1e-4))
    oq = _oracle(dict(quant_depth=1e-4, quant_prox=1e-2, quant_marker=1e-4), nu=4, nv=4, m=3)
    rq = oq.step(x, want=WANT)
    k = rq["depth_noisy"] / q
    assert np.abs(k - np.rint(k)).max() < 1e-4 and np.abs(rq["depth_noisy"] - rq["depth"]).max() <= 0.5 * q * (1 + 1e-5)
    assert len(np.unique(np.rint(k))) > 2
    km = rq["marker_noisy"] / q
    assert np.abs(km - np.rint(km)).max() < 1e-4 and np.abs(rq["marker_noisy"] - rq["marker"]).max() <= 0.5 * q * (1 + 1e-5)
    kp = rq["prox_noisy"] / float(np.float32(1e-2))
    assert np.abs(kp - np.rint(kp)).max() < 1e-4
    assert np.isfinite(rq["aux_sq_depth"]).all() and (rq["aux_sq_depth"] >= 0).all() and rq["aux_sq_depth"].max() <= 0.5 * q * (1 + 1e-5)
    beta, tau, dt = float(np.float32(0.5)), float(np.float32(0.05)), float(np.float32(0.005))
    om = _oracle(dict(hyst_mode="maxwell", beta=0.5, tau=0.05), nu=4, nv=4, m=3)
    for kstep in range(4):
        rm = om.step(x, want=WANT)
        f = 1.0 + beta * math.exp(-kstep * dt / tau)
        np.testing.assert_allclose(rm["depth_noisy"], f * rm["depth"], rtol=1e-12, atol=1e-18)
        np.testing.assert_allclose(rm["prox_noisy"], f * rm["prox"], rtol=1e-12, atol=1e-18)
        np.testing.assert_allclose(rm["marker_noisy"], f * rm["marker"], rtol=1e-12, atol=1e-16)
    # ASYM loading from rest: y_1 = alpha_load x
    oa = _oracle(dict(hyst_mode="asym", alpha_load=0.8, alpha_unload=0.5), nu=4, nv=4, m=3)
    ra = oa.step(x, want=WANT)
    np.testing.assert_allclose(ra["depth_noisy"], float(np.float32(0.8)) * ra["depth"], rtol=1e-12, atol=1e-18)


def test_depth_noisy_senses_with_the_perturbed_radius_eq26():
    # Eq. 26: depth_noisy = [max(0, R_j + eps_j) - phi]_+, eps_j from stream 8 (the same draw the noisy force uses)
    rho = float(np.float32(5e-4))
    o = _oracle(dict(radius_noise=5e-4), nu=4, nv=4)
    x = _inputs(-0.0318)
    r = o.step(x, want=WANT)
    for e, env in enumerate(ENVS):
        for j in range(16):
            eps = -rho + 2 * rho * _u(O.philox((int(env), j, 0, 8), KEY)[0])
            want = max(0.0, max(0.0, float(np.float32(R_TAX)) + eps) - r["aux_phi"][e, j])
            np.testing.assert_allclose(r["depth_noisy"][e, j], want, rtol=0, atol=1e-15)
    assert (r["depth_noisy"] != r["depth"]).any()


def test_read_delay_of_the_scalar_readouts():
    """Eq. 25 / Table 3: every sensor honours the read delay.  Only the signal is delayed (y_{t - Delta_n}); the bias is
    that of step t; steps before the episode began read 0 (Q12); Delta_n = max(0, Delta + k_n) with k_n from stream 9,
    taxel word 0xffffffff -- the same draw as the force / torque readout of that env and step (one sensor read)."""
    zs = [-0.0316, -0.0312, -0.0319, -0.0314, -0.0317, -0.0311, -0.0318, -0.0313]      # a different indentation every step
    bias = float(np.float32(3e-4))
    # fixed delay of 2 steps, no jitter
    o = _oracle(dict(read_delay=2, bias_depth=3e-4, bias_prox=3e-4, bias_marker=3e-4), nu=4, nv=4, m=3)
    hist = []
    for n, z in enumerate(zs):
        r = o.step(_inputs(z), want=WANT)
        hist.append({k: r[k].copy() for k in ("depth", "prox", "marker")})
        for k in ("depth", "prox", "marker"):
            want = (hist[n - 2][k] if n >= 2 else 0.0 * hist[n][k]) + bias
            np.testing.assert_allclose(r[k + "_noisy"], want, rtol=1e-12, atol=1e-18)
        if n >= 2:
            assert np.abs(hist[n]["depth"] - hist[n - 2]["depth"]).max() > 5e-5          # the delay is visible
    # a reset starts a new episode: the history is gone
    o.reset()
    r = o.step(_inputs(zs[0]), want=WANT)
    np.testing.assert_allclose(r["depth_noisy"], 0.0 * r["depth"] + bias, rtol=0, atol=1e-18)
    # jitter: Delta_n = max(0, 1 + k_n), k_n in {-1, 0, 1}, per (env, step); shared with ft_noisy
    J = 1
    o = _oracle(dict(read_delay=1, read_jitter=J), nu=4, nv=4, m=3)
    hist, seen = [], set()
    for n, z in enumerate(zs):
        r = o.step(_inputs(z), want=WANT + ("ft", "ft_noisy"))
        hist.append({k: r[k].copy() for k in ("depth", "prox", "marker", "ft")})
        for e, env in enumerate(ENVS):
            w0 = O.philox((int(env), 0xFFFFFFFF, n, 9), KEY)[0]
            delta = max(0, 1 + ((int(w0) >> 9) * (2 * J + 1) >> 23) - J)
            seen.add(delta)
            for k, kn in (("depth", "depth_noisy"), ("prox", "prox_noisy"), ("marker", "marker_noisy"), ("ft", "ft_noisy")):
                want = hist[n - delta][k][e] if n - delta >= 0 else 0.0 * hist[n][k][e]
                np.testing.assert_allclose(r[kn][e], want, rtol=1e-12, atol=1e-18)
    assert seen == {0, 1, 2}
