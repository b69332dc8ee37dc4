"""Pins of the Bessel radial basis of the oracle (the paper's lead model: "Radial basis 4 (Bessel)"):
b_n(d) = sqrt(2/r_c) sin(n pi d / r_c) / d, n = 1..K.  Textbook facts used as pins: b_n(r_c) = 0; b_n(d) -> n pi
sqrt(2/r_c) / r_c as d -> 0; orthonormality  int_0^rc b_m b_n d^2 dd = delta_mn  (quadrature); and, for the whole model
with this basis, forces = dual-number forces = central differences of the energy, net force zero."""
import dataclasses

import numpy as np

import gen
import oracle

RC, K = 5.0, 4


def test_bessel_closed_forms_and_orthonormality():
    g, c = oracle.rbf_cutoff_typed(RC, K, RC, "bessel")
    assert np.abs(g).max() < 1e-15 and abs(c) < 1e-16
    g0, _ = oracle.rbf_cutoff_typed(1e-9, K, RC, "bessel")
    assert np.allclose(g0, np.arange(1, K + 1) * np.pi * np.sqrt(2.0 / RC) / RC, rtol=1e-12)
    # a value typed by hand: n = 2, d = 1.25 = rc/4 -> sin(pi/2) = 1 -> sqrt(2/5) / 1.25
    g1, _ = oracle.rbf_cutoff_typed(1.25, K, RC, "bessel")
    assert abs(g1[1] - np.sqrt(0.4) / 1.25) < 1e-15
    # orthonormality with weight d^2 (composite Simpson, 4001 nodes)
    d = np.linspace(1e-12, RC, 4001)
    G = np.array([oracle.rbf_cutoff_typed(float(x), K, RC, "bessel")[0] for x in d])
    wq = np.ones_like(d); wq[1:-1:2] = 4.0; wq[2:-1:2] = 2.0; wq *= (d[1] - d[0]) / 3.0
    gram = (G * (wq * d * d)[:, None]).T @ G
    assert np.abs(gram - np.eye(K)).max() < 1e-9
    # the Gaussian basis is untouched by the new entry point
    ga, _ = oracle.rbf_cutoff(2.0, 20, RC)
    gb, _ = oracle.rbf_cutoff_typed(2.0, 20, RC, "gaussian")
    assert np.array_equal(ga, gb)


def test_bessel_model_forces():
    mc = dataclasses.replace(gen.model_cfg(1), K=K, rbf="bessel")
    b = gen.make_batch(1, 0, 2)
    w = gen.make_weights(mc, 3)
    out = oracle.evaluate(mc, w, b)
    fd = oracle.forces_dual(mc, w, b)
    scale = np.abs(out["forces"]).max()
    assert np.abs(out["forces"] - fd).max() < 1e-11 * scale
    h = 1e-4
    for (i, a) in [(0, 1), (9, 0), (20, 2)]:
        e = []
        for sgn in (+1, -1):
            pos = b.pos.copy(); pos[i, a] += sgn * h
            e.append(oracle.evaluate(mc, w, dataclasses.replace(b, pos=pos), forces=False)["energy"].sum())
        assert abs(-(e[0] - e[1]) / (2 * h) - out["forces"][i, a]) < 1e-6 * scale
    for g in range(b.n_structs):
        a0, a1 = b.struct_ptr[g], b.struct_ptr[g + 1]
        assert np.abs(out["forces"][a0:a1].sum(0)).max() < 1e-11 * scale
    # and the basis matters: the Gaussian model with the same weights gives another energy
    e_gauss = oracle.evaluate(dataclasses.replace(mc, rbf="gaussian"), w, b, forces=False)["energy"]
    assert not np.allclose(e_gauss, out["energy"], rtol=1e-6, atol=0)
