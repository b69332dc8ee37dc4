"""Pins of the all-images periodic radius graph of the oracle (PAPER.md:269 periodic boundary
conditions with cells narrower than twice the cutoff): independent image enumeration in numpy, textbook shell counts of a
ONE-atom simple-cubic cell (every neighbour is an image of the atom itself), equality with the minimum-image graph when
every cell width is at least 2 r_c, symmetry of the edge set, and — what minimum image cannot give in a narrow cell —
an energy that is smooth where a pair crosses half the cell (forces = central differences there)."""
import dataclasses

import numpy as np

import gen
import oracle
from helpers import edge_set, edges_by_image_enumeration, single


def narrow_cell(n=10, L=7.0, seed=2):
    rng = np.random.default_rng(seed)
    pos = rng.uniform(0, L, (n, 3))
    return single(rng.integers(1, 9, n), pos, 0, np.eye(3) * L, [1, 1, 1])


def test_matches_independent_enumeration_and_is_symmetric():
    for b, rc in ((narrow_cell(), 5.0), (narrow_cell(6, 4.0, 5), 6.0), (gen.make_batch(3, 2, 1), 6.0)):
        nb = oracle.neighbours(b, rc, all_images=True)
        es = edge_set(nb)
        assert len(es) == len(nb["send"])                                  # no duplicates
        assert es == edges_by_image_enumeration(b, rc, nimg=3)
        assert all((j, i, -a, -bb, -c) in es for (i, j, a, bb, c) in es)   # i<-j with s  <=>  j<-i with -s
    # slab: one axis not periodic -> no shift on it
    b = narrow_cell()
    b = dataclasses.replace(b, pbc=np.array([[1, 1, 0]], np.uint8))
    nb = oracle.neighbours(b, 5.0, all_images=True)
    assert np.all(nb["shift"][:, 2] == 0) and edge_set(nb) == edges_by_image_enumeration(b, 5.0, nimg=3)


def test_one_atom_simple_cubic_shell_counts():
    a = 2.0
    b = single([6], [[0.3, 0.1, 0.2]], 0, np.eye(3) * a, [1, 1, 1])
    # shells of the simple cubic lattice at d/a = 1, sqrt2, sqrt3, 2, sqrt5, sqrt6, sqrt8, 3: 6, 12, 8, 6, 24, 24, 12, 30
    counts = np.cumsum([6, 12, 8, 6, 24, 24, 12, 30])
    radii = a * np.sqrt([1, 2, 3, 4, 5, 6, 8, 9])
    for k in range(len(radii) - 1):
        rc = 0.5 * (radii[k] + radii[k + 1])
        nb = oracle.neighbours(b, rc, all_images=True)
        assert len(nb["send"]) == counts[k] and np.all(nb["send"] == 0)
    assert len(oracle.neighbours(b, 0.9 * a, all_images=True)["send"]) == 0
    assert len(oracle.neighbours(b, 10.0, all_images=False)["send"]) == 0   # minimum image: no self edge at all


def test_equals_minimum_image_in_wide_cells():
    b = gen.make_batch(5, n_atoms=400)            # L = 17.1 A >= 2 * 5 A
    assert edge_set(oracle.neighbours(b, 5.0, all_images=True)) == edge_set(oracle.neighbours(b, 5.0))


def test_energy_is_smooth_across_half_the_cell():
    """Two atoms in a 7 A cell, r_c = 5 A: moving one atom across x = L/2 swaps the minimum image, so the minimum-image
    energy has a kink there; with all images both copies are neighbours on either side and forces are exact gradients."""
    L, rc = 7.0, 5.0
    mc = dataclasses.replace(gen.model_cfg(1), cutoff=rc, pbc_images="all")
    w = gen.make_weights(mc, 8)
    def batch(x):
        return single([6, 8], [[0.0, 0.0, 0.0], [x, 0.4, 0.2]], 0, np.eye(3) * L, [1, 1, 1])
    h = 1e-5
    x0 = L / 2 + 3e-6                              # the central difference straddles the image switch
    out = oracle.evaluate(mc, w, batch(x0))
    ep = oracle.evaluate(mc, w, batch(x0 + h), forces=False)["energy"][0]
    em = oracle.evaluate(mc, w, batch(x0 - h), forces=False)["energy"][0]
    scale = max(1.0, np.abs(out["forces"]).max())
    assert abs(-(ep - em) / (2 * h) - out["forces"][1, 0]) < 1e-7 * scale
    # the same difference quotient with the minimum-image graph is off by far more: the kink this mode removes
    mc_min = dataclasses.replace(mc, pbc_images="minimum")
    kp = oracle.evaluate(mc_min, w, batch(x0 + h), forces=False)["energy"][0]
    km = oracle.evaluate(mc_min, w, batch(x0 - h), forces=False)["energy"][0]
    assert abs(-(kp - km) / (2 * h) - oracle.evaluate(mc_min, w, batch(x0))["forces"][1, 0]) > 1e-2
    assert np.abs(out["forces"].sum(0)).max() < 1e-11 * scale
    assert np.abs(out["forces"] - oracle.forces_dual(mc, w, batch(x0))).max() < 1e-11 * scale
