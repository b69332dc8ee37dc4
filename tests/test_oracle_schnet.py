"""Pins of the SchNet oracle (oracle/schnet_oracle.py, reading Q31) against things it does
not compute itself: a restatement with explicit Python loops over atoms and edges, closed forms, invariances, central
differences of its own energy (pins the reverse-mode forces), and the cutoff's continuity."""
import dataclasses
import math

import numpy as np
import pytest

import gen
from helpers import random_rotation, single, with_pos
from oracle.schnet_oracle import evaluate_schnet


def _mc(**kw):
    base = dict(F=32, T=2, K=8, H=2, cutoff=5.0, backbone="schnet")
    base.update(kw)
    return gen.ModelCfg(**base)


def _silu(x):
    return x / (1.0 + np.exp(-x))


def _loops(mc, w, b):
    """Independent restatement: plain loops, edges by brute force over all pairs (non-periodic inputs only)."""
    L = {n: w[off:off + int(np.prod(sh))].reshape(sh) for n, sh, _, off in gen.weights_layout(mc)}
    N = b.n_atoms
    a2s = np.repeat(np.arange(b.n_structs), np.diff(b.struct_ptr))
    x = L["emb"][b.Z].copy()
    dmu = mc.cutoff / (mc.K - 1)
    for t in range(mc.T):
        p = f"b{t}."
        x1 = np.array([L[p + "in_W"] @ x[i] for i in range(N)])
        m = np.zeros_like(x)
        for i in range(N):
            for j in range(N):
                if i == j or a2s[i] != a2s[j]:
                    continue
                d = math.sqrt(((b.pos[j] - b.pos[i]) ** 2).sum())
                if d >= mc.cutoff:
                    continue
                g = np.array([math.exp(-(d - k * dmu) ** 2 / (2 * dmu * dmu)) for k in range(mc.K)])
                Wf = (L[p + "flt_W2"] @ _silu(L[p + "flt_W1"] @ g + L[p + "flt_b1"]) + L[p + "flt_b2"]) * 0.5 * (math.cos(math.pi * d / mc.cutoff) + 1)
                m[i] += x1[j] * Wf
        x = np.array([x[i] + L[p + "out_W2"] @ _silu(L[p + "out_W1"] @ m[i] + L[p + "out_b1"]) + L[p + "out_b2"] for i in range(N)])
    E = np.zeros(b.n_structs)
    for i in range(N):
        h = b.head[a2s[i]]
        E[a2s[i]] += L[f"h{h}.out_w2"] @ _silu(L[f"h{h}.out_W1"] @ x[i] + L[f"h{h}.out_b1"]) + L[f"h{h}.out_b2"][0]
    return E


@pytest.fixture(scope="module")
def tiny():
    mc = _mc()
    b = dataclasses.replace(gen.make_batch(1, 0, 3), head=np.array([0, 1, 1], np.int32))
    return mc, gen.make_weights(mc, 7), b


def test_energy_against_explicit_loops(tiny):
    mc, w, b = tiny
    out = evaluate_schnet(mc, w, b, forces=False)
    assert out["n_edges"] > 100
    assert np.allclose(out["energy"], _loops(mc, w, b), rtol=1e-12, atol=1e-12)


def test_isolated_atoms_closed_form():
    mc = _mc()
    w = gen.make_weights(mc, 7)
    L = {n: w[off:off + int(np.prod(sh))].reshape(sh) for n, sh, _, off in gen.weights_layout(mc)}
    b = single([1, 8, 6], [[0, 0, 0], [20, 0, 0], [0, 30, 0]], head=1)
    x = L["emb"][b.Z].copy()
    for t in range(mc.T):   # no edges: m = 0, x += B2 silu(b1) + b2
        x = x + L[f"b{t}.out_W2"] @ _silu(L[f"b{t}.out_b1"]) + L[f"b{t}.out_b2"]
    e = sum(L["h1.out_w2"] @ _silu(L["h1.out_W1"] @ xi + L["h1.out_b1"]) + L["h1.out_b2"][0] for xi in x)
    out = evaluate_schnet(mc, w, b)
    assert out["n_edges"] == 0
    assert abs(out["energy"][0] - e) < 1e-12 * max(1.0, abs(e))
    assert np.abs(out["forces"]).max() == 0.0


def test_forces_are_minus_the_gradient(tiny):
    mc, w, b = tiny
    out = evaluate_schnet(mc, w, b)
    h = 3e-4
    for (i, a) in ((0, 0), (5, 1), (20, 2), (40, 0)):
        def en(delta):
            p = b.pos.copy(); p[i, a] += delta
            return evaluate_schnet(mc, w, with_pos(b, p), forces=False)["energy"].sum()
        fd = -(8.0 * (en(h) - en(-h)) - (en(2 * h) - en(-2 * h))) / (12.0 * h)
        assert abs(fd - out["forces"][i, a]) < 5e-8 * np.abs(out["forces"]).max()
    for g in range(b.n_structs):
        f = out["forces"][b.struct_ptr[g]:b.struct_ptr[g + 1]]
        p = b.pos[b.struct_ptr[g]:b.struct_ptr[g + 1]]
        assert np.abs(f.sum(0)).max() < 1e-11 * np.abs(f).max()                       # no net force
        assert np.abs(np.cross(p, f).sum(0)).max() < 1e-10 * np.abs(f).max()          # no net torque


def test_invariances(tiny):
    mc, w, b = tiny
    out = evaluate_schnet(mc, w, b)
    rng = np.random.default_rng(2)
    R = random_rotation(rng, improper=True)
    o2 = evaluate_schnet(mc, w, with_pos(b, b.pos @ R.T + np.array([3.0, -2.0, 1.0])))
    assert np.allclose(o2["energy"], out["energy"], rtol=1e-12)
    assert np.allclose(o2["forces"], out["forces"] @ R.T, rtol=1e-9, atol=1e-12)
    # permutation inside a structure; structures are independent of the rest of the batch; head locality
    n0 = b.struct_ptr[1]
    perm = np.concatenate([rng.permutation(n0), np.arange(n0, b.n_atoms)])
    o3 = evaluate_schnet(mc, w, dataclasses.replace(b, Z=b.Z[perm], pos=b.pos[perm]))
    assert np.allclose(o3["energy"], out["energy"], rtol=1e-12)
    assert np.allclose(o3["forces"], out["forces"][perm], rtol=1e-9, atol=1e-12)
    o4 = evaluate_schnet(mc, w, b.select([1]))
    assert np.allclose(o4["energy"], out["energy"][1:2], rtol=1e-12)
    o5 = evaluate_schnet(mc, w, dataclasses.replace(b, head=np.array([1, 1, 1], np.int32)))
    assert o5["energy"][0] != out["energy"][0] and np.allclose(o5["energy"][1:], out["energy"][1:], rtol=1e-13)


def test_cutoff_is_smooth_and_strict():
    mc = _mc(T=1)
    w = gen.make_weights(mc, 3)
    def en(d):
        return evaluate_schnet(mc, w, single([6, 8], [[0, 0, 0], [d, 0, 0]], 0), forces=False)
    far, near = en(mc.cutoff + 1e-6), en(mc.cutoff - 1e-6)
    assert far["n_edges"] == 0 and near["n_edges"] == 2
    assert abs(near["energy"][0] - far["energy"][0]) < 1e-9          # c(d) -> 0 quadratically at the cutoff
    assert abs(en(2.0)["energy"][0] - far["energy"][0]) > 1e-3


def test_periodic_images_and_lattice_translation():
    mc = _mc(cutoff=4.0)
    w = gen.make_weights(mc, 5)
    b = dataclasses.replace(gen.make_batch(3, 0, 1, n_atoms=54), head=np.array([1], np.int32))
    out = evaluate_schnet(mc, w, b)
    p = b.pos.copy()
    p[3] += b.cell[0][0] - 2 * b.cell[0][2]          # move one atom by a lattice vector combination
    o2 = evaluate_schnet(mc, w, with_pos(b, p))
    assert np.allclose(o2["energy"], out["energy"], rtol=1e-12)
    assert np.allclose(o2["forces"], out["forces"], rtol=1e-8, atol=1e-11)
    big = dataclasses.replace(b, cell=None, pbc=None)   # without the images the energy differs
    assert abs(evaluate_schnet(mc, w, big, forces=False)["energy"][0] - out["energy"][0]) > 1e-6
