"""Pins of the oracle's max-neighbour cap (Table V "Max neighbors 20"; "64" with periodic boundary
conditions; reading Q16): every receiver keeps its nearest max_neighbors senders inside the cutoff."""
import dataclasses

import numpy as np

import gen
import oracle
from helpers import edge_set, single


def _brute(batch, rc, k):
    """Independent numpy restatement: all pairs of a structure, sort by distance, keep k (non-periodic)."""
    out = set()
    sp = batch.struct_ptr
    for g in range(batch.n_structs):
        idx = np.arange(sp[g], sp[g + 1])
        for i in idx:
            d = np.linalg.norm(batch.pos[idx] - batch.pos[i], axis=1)
            cand = [(d[q], int(j)) for q, j in enumerate(idx) if j != i and d[q] < rc]
            for _, j in sorted(cand)[:k]:
                out.add((int(i), j, 0, 0, 0))
    return out


def test_cap_against_numpy_sort_and_limits():
    b = gen.make_batch(2, 0, 6)
    full = oracle.neighbours(b, 5.0)
    deg = np.diff(full["rowptr"])
    for k in (1, 4, 12, int(deg.max()), 500):
        nb = oracle.neighbours(b, 5.0, max_neighbors=k)
        assert edge_set(nb) == _brute(b, 5.0, k)
        assert np.array_equal(np.diff(nb["rowptr"]), np.minimum(deg, k))
    assert edge_set(oracle.neighbours(b, 5.0, max_neighbors=int(deg.max()))) == edge_set(full)
    nb = oracle.neighbours(b, 5.0, max_neighbors=4)              # the set is NOT symmetric any more
    es = edge_set(nb)
    assert any((j, i, 0, 0, 0) not in es for (i, j, _, _, _) in es)


def test_cap_on_a_simple_cubic_lattice_keeps_the_first_shells():
    """Textbook: simple cubic, spacing a: 6 nearest neighbours at a, then 12 at a sqrt(2).  Cap 6 = exactly the first shell,
    cap 18 = the first two shells (periodic, minimum image, cell of 6 spacings >= 2 r_c)."""
    a, n = 1.5, 6
    g = np.stack(np.meshgrid(*[np.arange(n)] * 3, indexing="ij"), -1).reshape(-1, 3) * a
    b = single(np.full(len(g), 6), g, cell=np.eye(3) * a * n, pbc=[1, 1, 1])
    for k, dmax in ((6, a), (18, a * np.sqrt(2))):
        nb = oracle.neighbours(b, 4.4, max_neighbors=k)
        assert np.all(np.diff(nb["rowptr"]) == k)
        d = np.linalg.norm(nb["rvec"], axis=1)
        assert d.max() < dmax + 1e-12 and np.isclose(np.sort(d)[-1], dmax)


def test_capped_model_forces_are_the_gradient_of_its_energy():
    """The reverse sweep on an ASYMMETRIC edge set: dual numbers (independent of the hand-written sweep), central
    differences with the edge list re-derived (positions well away from any rank swap), sum F = 0, head locality."""
    mc = dataclasses.replace(gen.model_cfg(1), max_neighbors=5)
    w = gen.make_weights(mc, 1)
    b = gen.make_batch(1, 0, 3)
    out = oracle.evaluate(mc, w, b)
    assert out["n_edges"] == 5 * b.n_atoms
    fd = oracle.forces_dual(mc, w, b)
    assert np.abs(out["forces"] - fd).max() < 1e-11 * np.abs(fd).max()
    for g in range(b.n_structs):
        f = out["forces"][b.struct_ptr[g]:b.struct_ptr[g + 1]]
        assert np.abs(f.sum(0)).max() < 1e-10 * np.abs(f).max()
    # central differences of the capped energy (the cap makes E only piecewise smooth: the step is far smaller than the
    # smallest gap between the 5th and 6th neighbour distances of this seeded input)
    nbf = oracle.neighbours(b, mc.cutoff)
    gaps = []
    for i in range(b.n_atoms):
        d = np.sort(np.linalg.norm(nbf["rvec"][nbf["rowptr"][i]:nbf["rowptr"][i + 1]], axis=1))
        if len(d) > 5:
            gaps.append(d[5] - d[4])
    assert min(gaps) > 1e-3
    h = 1e-5
    for (i, c) in ((0, 0), (7, 1), (20, 2)):
        p = b.pos.copy(); p[i, c] += h
        ep = oracle.evaluate(mc, w, dataclasses.replace(b, pos=p), forces=False)["energy"].sum()
        p[i, c] -= 2 * h
        em = oracle.evaluate(mc, w, dataclasses.replace(b, pos=p), forces=False)["energy"].sum()
        assert abs(-(ep - em) / (2 * h) - out["forces"][i, c]) < 1e-6 * np.abs(out["forces"]).max()
    # a cap at least as large as the largest degree changes nothing
    big = dataclasses.replace(mc, max_neighbors=64)
    ref = oracle.evaluate(gen.model_cfg(1), w, b)
    o2 = oracle.evaluate(big, w, b)
    assert np.array_equal(o2["energy"], ref["energy"]) and np.array_equal(o2["forces"], ref["forces"])
