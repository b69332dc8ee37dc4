"""Pins of oracle.evaluate_blended (blended multi-head inference, Fig. 5): it is defined as a
linear combination of single-head evaluations, each pinned in test_oracle_model.py; what is checked here is the
combination itself: one-hot weights reproduce the single-head result, the energy of an isolated atom is the weighted sum
of the closed-form head outputs, forces stay exact gradients of the blended energy (central differences), and branch
skipping is the same as zeroing the skipped weights."""
import dataclasses

import numpy as np

import gen
import oracle


def _setup(n=3, H=4):
    mc = dataclasses.replace(gen.model_cfg(1), H=H)
    b = gen.make_batch(1, 0, n)
    w = gen.make_weights(mc, 5)
    return mc, b, w


def test_one_hot_weights_equal_single_head():
    mc, b, w = _setup()
    heads = np.array([2, 0, 3], np.int32)
    hw = np.zeros((3, mc.H))
    hw[np.arange(3), heads] = 1.0
    ref = oracle.evaluate(mc, w, dataclasses.replace(b, head=heads))
    out = oracle.evaluate_blended(mc, w, b, hw)
    assert np.allclose(out["energy"], ref["energy"], rtol=0, atol=1e-13 * np.abs(ref["energy"]).max())
    assert np.allclose(out["forces"], ref["forces"], rtol=0, atol=1e-12 * np.abs(ref["forces"]).max())


def test_isolated_atom_weighted_sum_of_heads():
    from helpers import single
    mc, _, w = _setup()
    atom = single([6], [[0.0, 0.0, 0.0]], 0)
    hw = np.array([[0.1, 0.2, 0.3, 0.4]])
    singles = [oracle.evaluate(mc, w, dataclasses.replace(atom, head=np.array([h], np.int32)))["energy"][0]
               for h in range(mc.H)]
    out = oracle.evaluate_blended(mc, w, atom, hw)
    assert abs(out["energy"][0] - float(np.dot(hw[0], singles))) < 1e-13 * max(1.0, max(abs(x) for x in singles))
    assert np.abs(out["forces"]).max() == 0.0


def test_forces_are_gradients_of_the_blended_energy():
    mc, b, w = _setup(n=1)
    rng = np.random.default_rng(1)
    hw = rng.dirichlet(np.ones(mc.H), size=1)
    out = oracle.evaluate_blended(mc, w, b, hw)
    h = 1e-4
    for (i, a) in [(0, 0), (5, 2), (11, 1)]:
        ep = []
        for sgn in (+1, -1):
            pos = b.pos.copy()
            pos[i, a] += sgn * h
            ep.append(oracle.evaluate_blended(mc, w, dataclasses.replace(b, pos=pos), hw, forces=False)["energy"][0])
        fd = -(ep[0] - ep[1]) / (2 * h)
        assert abs(fd - out["forces"][i, a]) < 1e-6 * max(1.0, np.abs(out["forces"]).max())


def test_branch_skipping_is_zeroing():
    mc, b, w = _setup()
    hw = np.array([[0.90, 0.05, 0.04, 0.01], [0.25, 0.25, 0.25, 0.25], [0.0, 0.02, 0.97, 0.01]])
    skipped = oracle.evaluate_blended(mc, w, b, hw, skip_below=0.03)
    zeroed = oracle.evaluate_blended(mc, w, b, np.where(hw < 0.03, 0.0, hw))
    assert np.array_equal(skipped["energy"], zeroed["energy"]) and np.array_equal(skipped["forces"], zeroed["forces"])
    full = oracle.evaluate_blended(mc, w, b, hw)
    assert not np.allclose(full["energy"], skipped["energy"], rtol=1e-12, atol=0)
