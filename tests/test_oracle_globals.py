"""Pins of the oracle's global attributes ("global attributes such as charge and spin used as additional input
features"; reading Q30: s0_i = emb[Z_i] + glob_W . (charge, spin) of the atom's structure)."""
import dataclasses

import numpy as np

import gen
import oracle


def _setup():
    mc = dataclasses.replace(gen.model_cfg(1), n_global=2)
    w = gen.make_weights(mc, 1)
    assert w.size == gen.weights_count(gen.model_cfg(1)) + 2 * mc.F == oracle.weights_count(mc)
    return mc, w, gen.make_batch(1, 0, 4)


def test_zero_attributes_reduce_to_the_plain_model():
    mc, w, b = _setup()
    base = oracle.evaluate(gen.model_cfg(1), w[:gen.weights_count(gen.model_cfg(1))], b)
    z = oracle.evaluate(mc, w, b, globals_=np.zeros((b.n_structs, 2)))
    assert np.array_equal(z["energy"], base["energy"]) and np.array_equal(z["forces"], base["forces"])
    n = oracle.evaluate(mc, w, b)                       # no attributes given = zeros
    assert np.array_equal(n["energy"], base["energy"])


def test_attributes_shift_the_embedding_linearly_and_locally():
    mc, w, b = _setup()
    gl = np.array([[1.0, 3.0], [0.0, 1.0], [-2.0, 2.0], [0.0, 0.0]])
    out = oracle.evaluate(mc, w, b, globals_=gl, features=True)
    # equivalent model: the attribute term folded into a per-structure embedding table (closed form of Q30)
    F = mc.F
    wl = {n: (sh, off) for n, sh, _, off in gen.weights_layout(mc)}
    gw = w[wl["glob_W"][1]:wl["glob_W"][1] + 2 * F].reshape(F, 2)
    base_mc = gen.model_cfg(1)
    for g in range(b.n_structs):
        w2 = w[:gen.weights_count(base_mc)].copy()
        emb = w2[:(mc.Zmax + 1) * F].reshape(mc.Zmax + 1, F)
        emb += gw @ gl[g]
        ref = oracle.evaluate(base_mc, w2, b.select([g]))
        assert np.allclose(ref["energy"][0], out["energy"][g], rtol=1e-13, atol=0)
        assert np.allclose(ref["forces"], out["forces"][b.struct_ptr[g]:b.struct_ptr[g + 1]], rtol=1e-11, atol=1e-11)
    # a structure's attributes change only that structure
    gl2 = gl.copy(); gl2[1] = [5.0, -1.0]
    o2 = oracle.evaluate(mc, w, b, globals_=gl2)
    same = [0, 2, 3]
    assert np.array_equal(o2["energy"][same], out["energy"][same]) and o2["energy"][1] != out["energy"][1]
    # forces stay the gradient of the energy (dual numbers do not see the attributes: check by central differences)
    h = 1e-5
    for (i, c) in ((1, 0), (40, 2)):
        p = b.pos.copy(); p[i, c] += h
        ep = oracle.evaluate(mc, w, dataclasses.replace(b, pos=p), forces=False, globals_=gl)["energy"].sum()
        p[i, c] -= 2 * h
        em = oracle.evaluate(mc, w, dataclasses.replace(b, pos=p), forces=False, globals_=gl)["energy"].sum()
        assert abs(-(ep - em) / (2 * h) - out["forces"][i, c]) < 1e-6 * np.abs(out["forces"]).max()
