"""Known-answer pins for the Philox counter layout and the word -> channel assignment of the oracle's draws.

SURVEY 8(c) O8 / DESIGN.md section 2 fix: key = (seed_lo, seed_hi); counter = (env, taxel, n, episode << 4 | stream);
  stream 0 words (0,1),(2,3) -> Box-Muller -> drift normals of channels (0,1),(2,3); stream 1 words (0,1) -> channels (4,5);
  stream 2, n = 0, word 0    -> dead iff word < floor(p_dead 2^32)                                   (Eq. 28)
  stream 3, n = 0, word 0    -> gain gamma = g_min + (g_max - g_min) u                                (Eq. 27)
  streams 4 / 5, n = 0       -> stuck readout z_bj, words like streams 0 / 1                          (Eq. 28)
  streams 6 / 7, step n      -> white noise n_t, words like streams 0 / 1                             (Eq. 25)
The statistical pins of test_oracle_pins.py (moments, ranges, independence) cannot tell two counter words or two
output words apart.  Here every draw is REBUILT in the test from `O.philox` (itself pinned by the Random123
known-answer vectors) with the uniform / Box-Muller rule written out with `math`, on a scene with a non-zero global
env id, a non-zero taxel, step n >= 1, a 64-bit seed with distinct halves, and again after a reset (episode 1).
Swapping env and taxel in the counter, n and the episode word, the key halves, or feeding channels 4-5 from words
2-3 fails these tests (checked against deliberately mutated copies of oracle.cpp).
"""
import math

import numpy as np

from oracle import oracle as O

SEED = 0x1234567899ABCDEF
KEY = (SEED & 0xFFFFFFFF, SEED >> 32)
ENVS = np.array([7, 300001])
R_TAX = 2.0e-3


def _patch(nu=3, nv=2):
    return dict(link=0, origin=(0, 0, 0), u_axis=(1, 0, 0), v_axis=(0, 1, 0), size_u=0.006, size_v=0.004, nu=nu, nv=nv,
                radius=R_TAX, marker_nu=0, marker_nv=0)


def _oracle(noise, nu=3, nv=2):
    o = O.Oracle([_patch(nu, nv)], nu * nv, 1, 1, ENVS, noise=dict(dict(noise_enable=1, seed=SEED, hyst_mode="off"), **noise))
    E = len(ENVS)
    o.set_geometry(np.ones((E, 1), np.int32), np.full((E, 1, 4), 0.030, np.float32))
    return o


def _inputs(z):
    E = len(ENVS)
    d = dict(link_pos=np.tile(np.array([0, 0, z], np.float32), (E, 1, 1)),
             link_quat=np.tile(np.array([1, 0, 0, 0], np.float32), (E, 1, 1)),
             link_linvel=np.zeros((E, 1, 3), np.float32), link_angvel=np.zeros((E, 1, 3), np.float32),
             obj_pos=np.zeros((E, 1, 3), np.float32), obj_quat=np.tile(np.array([1, 0, 0, 0], np.float32), (E, 1, 1)),
             obj_linvel=np.zeros((E, 1, 3), np.float32), obj_angvel=np.zeros((E, 1, 3), np.float32))
    return d


def _u(w):
    return (2.0 * (int(w) >> 9) + 1.0) / 16777216.0          # O8: u = (2 (w >> 9) + 1) 2^-24


def _bm(wa, wb):
    r = math.sqrt(-2.0 * math.log(_u(wa)))                  # O8: Box-Muller on a word pair
    return r * math.cos(2.0 * math.pi * _u(wb)), r * math.sin(2.0 * math.pi * _u(wb))


def _six_normals(env, j, n, ep, s_lo, s_hi):
    """Six N(0,1) of one (env, taxel, step): stream s_lo words (0,1),(2,3) -> channels 0-3, stream s_hi words (0,1) -> 4-5."""
    w0 = O.philox((env, j, n, (ep << 4) | s_lo), KEY)
    w1 = O.philox((env, j, n, (ep << 4) | s_hi), KEY)
    return np.array(_bm(w0[0], w0[1]) + _bm(w0[2], w0[3]) + _bm(w1[0], w1[1]))


def _six_uniforms(env, j, ep, s_lo, s_hi):
    w0 = O.philox((env, j, 0, (ep << 4) | s_lo), KEY)
    w1 = O.philox((env, j, 0, (ep << 4) | s_hi), KEY)
    return np.array([_u(w) for w in (w0[0], w0[1], w0[2], w0[3], w1[0], w1[1])])


def _dead(env, j, ep, p):
    return int(O.philox((env, j, 0, (ep << 4) | 2), KEY)[0]) < int(math.floor(float(np.float32(p)) * 4294967296.0))


def test_drift_draws_known_answers():
    # Eq. 25 drift, no contact: ft_noisy[e, j, c] after step n = sum_{m <= n} sigma_c z_c(env, j, m, episode)
    sf, st = float(np.float32(1e-3)), float(np.float32(2e-5))
    o = _oracle(dict(sigma_rw_force=1e-3, sigma_rw_torque=2e-5))
    far = _inputs(-0.5)
    sig = np.array([sf] * 3 + [st] * 3)
    for ep in (0, 1):
        acc = np.zeros((len(ENVS), 6, 6))
        for n in range(3):
            out = o.step(far)["ft_noisy"]
            for e, env in enumerate(ENVS):
                for j in range(6):
                    acc[e, j] += sig * _six_normals(int(env), j, n, ep, 0, 1)
            np.testing.assert_allclose(out, acc, rtol=1e-12, atol=1e-18)
        o.reset()
    # the six channels of one (env, taxel, step) are six DIFFERENT words (a repeated pair would show here)
    z = _six_normals(7, 5, 2, 0, 0, 1)
    assert len(np.unique(np.round(z, 12))) == 6


def test_dead_mask_known_answers():
    # Eq. 28: dead iff word 0 of stream 2 at n = 0 is below floor(p 2^32); constant over the episode, re-drawn at reset
    p = 0.3
    o = _oracle(dict(p_dead=p, sigma_rw_force=1e-3, sigma_rw_torque=1e-5), nu=8, nv=8)
    far = _inputs(-0.5)
    for ep in (0, 1, 2):
        want = np.array([[_dead(int(env), j, ep, p) for j in range(64)] for env in ENVS])
        assert 5 < want.sum() < 60                              # both outcomes occur
        for n in range(2):
            got = o.step(far)["dead"].astype(bool)
            np.testing.assert_array_equal(got, want)
        o.reset()


def test_gain_known_answers():
    # Eq. 27: gamma = g_min + (g_max - g_min) u(word 0 of stream 3, n = 0), one value for the six channels
    gmin, gmax = float(np.float32(0.8)), float(np.float32(1.2))
    o = _oracle(dict(gain_min=0.8, gain_max=1.2))
    touch = _inputs(-0.0315)                                    # the patch centre sits 0.5 mm inside the r = 30 mm sphere
    for ep in (0, 1):
        for n in range(2):
            r = o.step(touch)
            assert (np.abs(r["ft"][..., 2]) > 1e-3).all()
            for e, env in enumerate(ENVS):
                for j in range(6):
                    g = gmin + (gmax - gmin) * _u(O.philox((int(env), j, 0, (ep << 4) | 3), KEY)[0])
                    np.testing.assert_allclose(r["ft_noisy"][e, j], g * r["ft"][e, j], rtol=1e-12, atol=1e-18)
        o.reset()


def test_white_noise_known_answers():
    # Eq. 25 n_t: streams 6 / 7 of the step counter, Box-Muller laid out like the drift draws; nothing accumulates
    sf, st = float(np.float32(2e-3)), float(np.float32(3e-5))
    o = _oracle(dict(sigma_white_force=2e-3, sigma_white_torque=3e-5))
    far = _inputs(-0.5)
    sig = np.array([sf] * 3 + [st] * 3)
    for ep in (0, 1):
        for n in range(3):
            out = o.step(far)["ft_noisy"]
            for e, env in enumerate(ENVS):
                for j in range(6):
                    np.testing.assert_allclose(out[e, j], sig * _six_normals(int(env), j, n, ep, 6, 7), rtol=1e-12, atol=1e-18)
        o.reset()


def test_stuck_value_known_answers():
    # Eq. 28 z_bj ~ U[l, u]: streams 4 (channels 0-3) / 5 (channels 4-5) at n = 0, one value per channel and episode
    lf, hf, lt, ht = (float(np.float32(v)) for v in (0.5, 1.5, -0.02, -0.01))
    p = 0.5
    o = _oracle(dict(p_dead=p, stuck_min_force=0.5, stuck_max_force=1.5, stuck_min_torque=-0.02, stuck_max_torque=-0.01),
                nu=4, nv=4)
    far = _inputs(-0.5)
    lo, hi = np.array([lf] * 3 + [lt] * 3), np.array([hf] * 3 + [ht] * 3)
    for ep in (0, 1):
        for n in range(2):
            out = o.step(far)
            n_dead = 0
            for e, env in enumerate(ENVS):
                for j in range(16):
                    if _dead(int(env), j, ep, p):
                        n_dead += 1
                        assert out["dead"][e, j] == 1
                        np.testing.assert_allclose(out["ft_noisy"][e, j], lo + (hi - lo) * _six_uniforms(int(env), j, ep, 4, 5),
                                                   rtol=1e-12, atol=1e-18)
                    else:
                        assert out["dead"][e, j] == 0 and not out["ft_noisy"][e, j].any()
            assert 4 < n_dead < 28
        o.reset()
