"""Pins for the oracle's radius graph (SURVEY.md §8(c) B1 and "What pins each part / Neighbour sets")."""
import os
from collections import Counter
from fractions import Fraction

import numpy as np
import pytest

import gen
import oracle
from helpers import edge_set, edges_by_image_enumeration, single

GOLD = os.path.join(os.path.dirname(__file__), "golden", "lattice_shells.txt")


def _shells(kind):
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, p, q, c = line.split()
        if k == kind:
            out[Fraction(int(p), int(q))] = int(c)
    return out


def _lattice(kind, m, a):
    g = np.arange(m, dtype=np.float64)
    corner = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    sites = corner if kind == "sc" else np.concatenate([corner, corner + 0.5])
    return sites * a


@pytest.mark.parametrize("kind,m,rc_over_a", [("sc", 7, 3.05), ("bcc", 5, 2.05)])
def test_textbook_shell_counts(kind, m, rc_over_a):
    a = 1.3
    pos = _lattice(kind, m, a)
    L = m * a
    assert L >= 2 * rc_over_a * a
    b = single(np.ones(len(pos)), pos, cell=np.eye(3) * L, pbc=[1, 1, 1])
    nb = oracle.neighbours(b, rc_over_a * a)
    d2 = (nb["rvec"] ** 2).sum(1) / (a * a)
    expect = _shells(kind)
    for i in (0, len(pos) // 2, len(pos) - 1):
        mine = Counter(Fraction(int(round(x * 4)), 4) for x in d2[nb["recv"] == i])
        assert dict(mine) == expect, (kind, i)
    # every atom has the same degree
    assert len(set(np.diff(nb["rowptr"]).tolist())) == 1


def test_matches_image_enumeration_periodic_and_scipy():
    rng = np.random.default_rng(1)
    L = 11.0
    rc = 5.0
    pos = rng.uniform(-3, 14, size=(60, 3))            # atoms outside the cell are allowed (Q14)
    b = single(np.ones(60), pos, cell=np.eye(3) * L, pbc=[1, 1, 1])
    nb = oracle.neighbours(b, rc)
    assert edge_set(nb) == edges_by_image_enumeration(b, rc)
    # library cross-check: scipy periodic KD-tree pair count
    from scipy.spatial import cKDTree
    tree = cKDTree(np.mod(pos, L), boxsize=L)
    assert 2 * len(tree.query_pairs(rc)) == len(nb["recv"])


def test_mixed_pbc_and_triclinic():
    rng = np.random.default_rng(2)
    rc = 3.0
    C = np.array([[9.0, 0.0, 0.0], [1.0, 8.5, 0.0], [0.5, -0.7, 9.5]])
    pos = rng.uniform(0, 1, size=(40, 3)) @ C
    for pbc in ([1, 1, 1], [1, 0, 1], [0, 0, 1]):
        b = single(np.ones(40), pos, cell=C, pbc=pbc)
        nb = oracle.neighbours(b, rc)
        assert edge_set(nb) == edges_by_image_enumeration(b, rc), pbc
        # r = x_j - x_i + shift.C
        r = pos[nb["send"]] - pos[nb["recv"]] + nb["shift"].astype(float) @ C
        assert np.allclose(r, nb["rvec"], atol=1e-13)


def test_symmetry_and_sorted_csr():
    b = gen.make_batch(3, 0, 2)
    nb = oracle.neighbours(b, 6.0)
    es = edge_set(nb)
    assert all((j, i, -a, -bb, -c) in es for (i, j, a, bb, c) in es)
    assert len(es) == len(nb["recv"])                   # at most one edge per ordered pair (Q12)
    assert len({(i, j) for (i, j, *_s) in es}) == len(es)
    # receiver-sorted, ascending sender inside a row
    assert np.all(np.diff(nb["recv"]) >= 0)
    for i in range(0, b.n_atoms, 17):
        row = nb["send"][nb["rowptr"][i]:nb["rowptr"][i + 1]]
        assert np.all(np.diff(row) > 0)
    assert nb["rowptr"][-1] == len(nb["recv"])


def test_lattice_translation_invariance():
    b = gen.make_batch(3, 0, 1)
    L = b.cell[0, 0, 0]
    nb = oracle.neighbours(b, 6.0)
    rng = np.random.default_rng(3)
    moved = b.pos + rng.integers(-2, 3, size=b.pos.shape) * L
    nb2 = oracle.neighbours(gen.Batch(b.Z, moved, b.struct_ptr, b.head, b.cell, b.pbc), 6.0)
    assert np.array_equal(nb["recv"], nb2["recv"]) and np.array_equal(nb["send"], nb2["send"])
    assert np.allclose(nb["rvec"], nb2["rvec"], atol=1e-9)


def test_nonperiodic_equals_huge_cell_and_no_cross_structure_edges():
    b = gen.make_batch(2, 0, 6)
    nb = oracle.neighbours(b, 5.0)
    S = b.n_structs
    big = gen.Batch(b.Z, b.pos, b.struct_ptr, b.head, np.tile(np.eye(3) * 1e4, (S, 1, 1)), np.ones((S, 3), np.uint8))
    nb2 = oracle.neighbours(big, 5.0)
    assert edge_set(nb) == edge_set(nb2)
    sof = np.repeat(np.arange(S), np.diff(b.struct_ptr))
    assert np.array_equal(sof[nb["recv"]], sof[nb["send"]])
    # plain definition on the whole batch
    assert edge_set(nb) == edges_by_image_enumeration(b, 5.0)
    d = np.linalg.norm(nb["rvec"], axis=1)
    assert d.max() < 5.0 and d.min() >= 0.9 - 1e-12


def test_small_cell_keeps_nearest_image_only():
    # Q13: cell narrower than 2 rc -> exactly one (the nearest) image per ordered pair
    b = gen.make_batch(3, 5, 1)
    L = b.cell[0, 0, 0]
    assert L < 12.0
    nb = oracle.neighbours(b, 6.0)
    allimg = edges_by_image_enumeration(b, 6.0)
    mine = edge_set(nb)
    assert mine <= allimg
    pairs = {(i, j) for (i, j, *_s) in allimg if i != j}
    assert {(i, j) for (i, j, *_s) in mine} == pairs     # every pair with some image inside rc is kept once
    # and it is the nearest image
    dmin = {}
    for (i, j, a, bb, c) in allimg:
        if i == j:
            continue
        r = b.pos[j] - b.pos[i] + np.array([a, bb, c]) * L
        dmin[(i, j)] = min(dmin.get((i, j), 1e9), np.linalg.norm(r))
    d = np.linalg.norm(nb["rvec"], axis=1)
    for e in range(0, len(d), 101):
        assert abs(d[e] - dmin[(int(nb["recv"][e]), int(nb["send"][e]))]) < 1e-12


def test_empty_and_single_atom():
    b = single([1], [[0.0, 0.0, 0.0]])
    nb = oracle.neighbours(b, 5.0)
    assert len(nb["recv"]) == 0 and nb["rowptr"].tolist() == [0, 0]
