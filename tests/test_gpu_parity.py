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


def _assert_ok(rep, max_band_frac=1e-3):
    print(json.dumps({k: v for k, v in rep.items()}, default=str))
    assert not rep["failures"], rep["failures"]
    n = max(rep["checked"], 1)
    assert rep["ft_exempt"] + rep["contact_tainted"] <= max(20, max_band_frac * n), rep


def _parity(w, ids=None, steps=None, **kw):
    from parity import run_parity
    return run_parity(w, lambda ww: _sim(ww, **kw), lambda ww, i, t: _orc(ww, i, t, **kw), ids, steps,
                      kw.get("outputs"), threads=os.cpu_count() or 1)


def test_config1_tiny():
    _assert_ok(_parity(W.config(1)))


def test_config2_primitives_small():
    _assert_ok(_parity(W.config(2, n_envs=192)))          # every primitive class, ragged last block


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
