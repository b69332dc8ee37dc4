"""Pins for the oracle's forward pass, readout and forces (SURVEY.md §8(c) "What pins each part")."""
import dataclasses
import os

import numpy as np
import pytest

import gen
import oracle
from helpers import edges_by_image_enumeration, random_rotation, single, torch_painn, with_pos

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def silu(x):
    return x / (1.0 + np.exp(-x))


@pytest.fixture(scope="module")
def tiny():
    mc = gen.model_cfg(1)
    return mc, gen.make_weights(mc, 1), gen.make_batch(1)


# ----------------------------------------------------------------------------- RBF / cutoff closed forms
def test_rbf_cutoff_closed_forms():
    rows = [l.split() for l in open(os.path.join(GOLD, "rbf_cutoff_closed_forms.txt")) if l.strip() and l[0] != "#"]
    K, rc = 20, 5.0
    for q, where, k, val in rows:
        val = float(val)
        if q == "cutoff":
            _, c = oracle.rbf_cutoff(float(where) * rc, K, rc)
            assert abs(c - val) < 1e-15
        else:
            off = {"rbf_at_centre": 0, "rbf_one_spacing": 1, "rbf_two_spacings": 2}[q]
            for kk in (0, 3, K - 3):
                g, _ = oracle.rbf_cutoff((kk + off) * rc / (K - 1), K, rc)
                assert abs(g[kk] - val) < 1e-14
    # monotone decreasing envelope, smooth at rc: c'(rc) = 0 by central difference
    h = 1e-6
    _, cm = oracle.rbf_cutoff(rc - h, K, rc)
    assert 0 <= cm < 1e-11


# ----------------------------------------------------------------------------- symmetry pins
def test_rotation_translation_inversion_invariance_and_equivariance(tiny):
    mc, w, b = tiny
    ref = oracle.evaluate(mc, w, b, features=True)
    rng = np.random.default_rng(0)
    for improper in (False, True):
        R = random_rotation(rng, improper)
        t = rng.normal(size=3) * 3
        out = oracle.evaluate(mc, w, with_pos(b, b.pos @ R.T + t), features=True)
        assert np.allclose(out["energy"], ref["energy"], rtol=0, atol=1e-11)
        assert np.allclose(out["s"], ref["s"], atol=1e-11)
        # v is a vector feature: v(Rx)[i,:,f] = R v(x)[i,:,f]
        assert np.allclose(out["v"], np.einsum("ab,ibf->iaf", R, ref["v"]), atol=1e-11)
        assert np.allclose(out["forces"], ref["forces"] @ R.T, atol=1e-10)
    inv = oracle.evaluate(mc, w, with_pos(b, -b.pos))               # E(x) = E(-x)  (Q4 sign independence)
    assert np.allclose(inv["energy"], ref["energy"], atol=1e-11)
    assert np.abs(ref["v"]).max() > 1e-3                             # the vector channel is alive


def test_permutation_within_structure(tiny):
    mc, w, b = tiny
    ref = oracle.evaluate(mc, w, b)
    rng = np.random.default_rng(1)
    perm = np.concatenate([b.struct_ptr[g] + rng.permutation(b.struct_ptr[g + 1] - b.struct_ptr[g])
                           for g in range(b.n_structs)])
    out = oracle.evaluate(mc, w, dataclasses.replace(b, Z=b.Z[perm], pos=b.pos[perm]))
    assert np.allclose(out["energy"], ref["energy"], atol=1e-11)
    assert np.allclose(out["forces"], ref["forces"][perm], atol=1e-11)


def test_batch_composition_and_head_locality():
    mc = gen.model_cfg(2)
    mc = dataclasses.replace(mc, F=16, T=2)
    w = gen.make_weights(mc, 2)
    b = gen.make_batch(2, 0, 5)
    ref = oracle.evaluate(mc, w, b)
    for g in (0, 3):
        alone = oracle.evaluate(mc, w, b.select([g]))
        a, e = b.struct_ptr[g], b.struct_ptr[g + 1]
        assert alone["energy"][0] == ref["energy"][g]
        assert np.array_equal(alone["forces"], ref["forces"][a:e])
    # changing one structure's head changes only that structure
    h2 = b.head.copy()
    h2[2] = (h2[2] + 5) % mc.H
    out = oracle.evaluate(mc, w, dataclasses.replace(b, head=h2))
    keep = np.arange(5) != 2
    assert np.array_equal(out["energy"][keep], ref["energy"][keep])
    assert out["energy"][2] != ref["energy"][2]
    a, e = b.struct_ptr[2], b.struct_ptr[3]
    assert np.array_equal(out["forces"][:a], ref["forces"][:a]) and np.array_equal(out["forces"][e:], ref["forces"][e:])
    assert not np.allclose(out["forces"][a:e], ref["forces"][a:e])


def test_single_head_equals_copied_heads():
    mc1 = gen.ModelCfg(F=16, T=1, K=8, H=1)
    w1 = gen.make_weights(mc1, 7)
    mcH = dataclasses.replace(mc1, H=4)
    lay = dict((n, (sh, off)) for n, sh, _f, off in gen.weights_layout(mc1))
    trunk_len = lay["h0.out_W1"][1]
    wH = np.concatenate([w1[:trunk_len]] + [w1[trunk_len:]] * 4)
    b = gen.make_batch(1, 0, 3)
    r1 = oracle.evaluate(mc1, w1, b)
    rH = oracle.evaluate(mcH, wH, dataclasses.replace(b, head=np.array([3, 0, 2], np.int32)))
    assert np.array_equal(r1["energy"], rH["energy"]) and np.array_equal(r1["forces"], rH["forces"])


# ----------------------------------------------------------------------------- closed forms
def _isolated_atom_energy(mc, W, z, head):
    """No neighbours: s' = s, v = 0, P = Q = 0, n = sqrt(eps), dot = 0  =>  s <- s + a_ss only."""
    F = mc.F
    s = W["emb"][z].copy()
    for t in range(mc.T):
        p = f"b{t}."
        n = np.full(F, np.sqrt(mc.norm_eps))
        k = silu(W[p + "upd_A1"] @ np.concatenate([s, n]) + W[p + "upd_c1"])
        a = W[p + "upd_A2"] @ k + W[p + "upd_c2"]
        s = s + a[2 * F:]
    hp = f"h{head}."
    return W[hp + "out_w2"] @ silu(W[hp + "out_W1"] @ s + W[hp + "out_b1"]) + W[hp + "out_b2"][0]


def test_isolated_atoms_and_zero_filter_closed_form():
    mc = gen.ModelCfg(F=8, T=3, K=6, H=3)
    w = gen.make_weights(mc, 11)
    W = gen.synth.unpack_weights(mc, w)
    # (v) atoms farther apart than the cutoff
    Z = np.array([1, 8, 26, 79], np.int32)
    pos = np.array([[0, 0, 0], [7, 0, 0], [0, 9, 0], [20, 20, 20]], np.float64)
    b = single(Z, pos, head=2)
    out = oracle.evaluate(mc, w, b, features=True)
    want = [_isolated_atom_energy(mc, W, z, 2) for z in Z]
    assert out["n_edges"] == 0
    assert np.allclose(out["eatom"], want, rtol=1e-13)
    assert abs(out["energy"][0] - sum(want)) < 1e-12
    assert np.abs(out["forces"]).max() == 0.0
    # (vi) same closed form for a dense molecule once the filter is zeroed: messages vanish
    w0 = w.copy()
    for name, shape, _f, off in gen.weights_layout(mc):
        if ".flt_" in name:
            w0[off:off + int(np.prod(shape))] = 0.0
    m = gen.make_batch(1, 0, 1)
    m = dataclasses.replace(m, head=np.array([1], np.int32))
    out0 = oracle.evaluate(mc, w0, m)
    want0 = sum(_isolated_atom_energy(mc, gen.synth.unpack_weights(mc, w0), z, 1) for z in m.Z)
    assert out0["n_edges"] > 0 and abs(out0["energy"][0] - want0) < 1e-11
    assert np.abs(out0["forces"]).max() < 1e-12


def test_two_atom_hand_expanded():
    """(vii) T=1, F=2, K=3 diatomic written out term by term for atom 0 <- atom 1 and back."""
    mc = gen.ModelCfg(F=2, T=1, K=3, H=1, cutoff=4.0)
    w = gen.make_weights(mc, 13)
    W = gen.synth.unpack_weights(mc, w)
    d = 1.7
    x = np.array([[0.3, -0.2, 0.1], [0.3, -0.2, 0.1 + d]])
    Z = [6, 8]
    out = oracle.evaluate(mc, w, single(Z, x), features=True)
    rc, K, F = mc.cutoff, mc.K, mc.F
    mu = np.array([0.0, 2.0, 4.0])
    g = np.exp(-(d - mu) ** 2 / (2 * 2.0 ** 2))
    c = 0.5 * (np.cos(np.pi * d / rc) + 1)
    filt = (W["b0.flt_W"] @ g + W["b0.flt_b"]) * c                       # same for both directions
    s = [W["emb"][6], W["emb"][8]]
    phi = [W["b0.msg_W2"] @ silu(W["b0.msg_W1"] @ si + W["b0.msg_b1"]) + W["b0.msg_b2"] for si in s]
    etot = 0.0
    for i, j, uz in ((0, 1, +1.0), (1, 0, -1.0)):                        # u = (x_j - x_i)/d along z
        xmsg = phi[j] * filt
        s1 = s[i] + xmsg[:F]
        v1 = np.zeros((3, F))
        v1[2] = xmsg[F:2 * F] * uz                                       # v_j = 0 in the first block
        P, Q = v1 @ W["b0.upd_U"].T, v1 @ W["b0.upd_V"].T
        n = np.sqrt((Q ** 2).sum(0) + mc.norm_eps)
        k = silu(W["b0.upd_A1"] @ np.concatenate([s1, n]) + W["b0.upd_c1"])
        a = W["b0.upd_A2"] @ k + W["b0.upd_c2"]
        s2 = s1 + a[F:2 * F] * (P * Q).sum(0) + a[2 * F:]
        v2 = v1 + a[:F] * P
        assert np.allclose(out["s"][i], s2, rtol=1e-13)
        assert np.allclose(out["v"][i], v2, rtol=1e-12, atol=1e-15)
        etot += W["h0.out_w2"] @ silu(W["h0.out_W1"] @ s2 + W["h0.out_b1"]) + W["h0.out_b2"][0]
    assert abs(out["energy"][0] - etot) < 1e-13
    # (v of forces) diatomic: equal, opposite, along the bond
    f = out["forces"]
    assert np.allclose(f[0], -f[1], atol=1e-13) and np.abs(f[:, :2]).max() < 1e-13 and abs(f[0, 2]) > 1e-6


# ----------------------------------------------------------------------------- third opinion (torch FP64 + autograd)
@pytest.mark.parametrize("cfg_id", [1, 3])
def test_torch_third_opinion(cfg_id):
    mc = dataclasses.replace(gen.model_cfg(cfg_id), F=16, T=2, K=10)
    w = gen.make_weights(mc, cfg_id)
    b = gen.make_batch(cfg_id, 0, 2, n_atoms=54 if cfg_id == 3 else None)
    if cfg_id == 3:   # make the cell >= 2 rc so that image enumeration == minimum image
        mc = dataclasses.replace(mc, cutoff=4.0)
    es = sorted(edges_by_image_enumeration(b, mc.cutoff))
    recv = [e[0] for e in es]
    send = [e[1] for e in es]
    shift = [e[2:] for e in es]
    ref = torch_painn(mc, w, b, (recv, send, shift))
    out = oracle.evaluate(mc, w, b, features=True)
    assert out["n_edges"] == len(es)
    assert np.allclose(out["energy"], ref["energy"], rtol=1e-12, atol=1e-12)
    assert np.allclose(out["s"], ref["s"], rtol=1e-11, atol=1e-12)
    assert np.allclose(out["v"], ref["v"], rtol=1e-11, atol=1e-12)
    assert np.allclose(out["forces"], ref["forces"], rtol=1e-9, atol=1e-11)


# ----------------------------------------------------------------------------- forces
def _fd_force(mc, w, b, i, a, g, h=3e-4):
    """-dE_g/dx_{i,a} by the five-point central difference (error O(h^4))."""
    def en(delta):
        p = b.pos.copy()
        p[i, a] += delta
        return oracle.evaluate(mc, w, with_pos(b, p), forces=False)["energy"][g]
    return -(8.0 * (en(h) - en(-h)) - (en(2 * h) - en(-2 * h))) / (12.0 * h)


def test_forces_dual_numbers_and_finite_differences(tiny):
    mc, w, b = tiny
    b = b.select([0, 5])
    out = oracle.evaluate(mc, w, b)
    fd = oracle.forces_dual(mc, w, b)
    assert np.abs(fd - out["forces"]).max() < 1e-12 * max(1.0, np.abs(fd).max())
    sof = np.repeat(np.arange(b.n_structs), np.diff(b.struct_ptr))
    rng = np.random.default_rng(5)
    for _ in range(6):
        i, a = int(rng.integers(b.n_atoms)), int(rng.integers(3))
        num = _fd_force(mc, w, b, i, a, sof[i])
        assert abs(num - out["forces"][i, a]) < 5e-9 * max(1.0, abs(num))


def test_net_force_and_torque_vanish():
    mc = dataclasses.replace(gen.model_cfg(2), F=32, T=2)
    w = gen.make_weights(mc, 2)
    b = gen.make_batch(2, 10, 4)
    out = oracle.evaluate(mc, w, b)
    scale = np.abs(out["forces"]).max()
    for g in range(b.n_structs):
        a, e = b.struct_ptr[g], b.struct_ptr[g + 1]
        assert np.abs(out["forces"][a:e].sum(0)).max() < 1e-12 * scale
        assert np.abs(np.cross(b.pos[a:e], out["forces"][a:e]).sum(0)).max() < 1e-11 * scale


def test_periodic_forces():
    mc = dataclasses.replace(gen.model_cfg(3), F=16, T=2, K=12, cutoff=4.0)
    w = gen.make_weights(mc, 3)
    b = gen.make_batch(3, 0, 1, n_atoms=54)             # L = 8.77 A >= 2 rc
    assert b.cell[0, 0, 0] >= 2 * mc.cutoff
    out = oracle.evaluate(mc, w, b)
    assert np.abs(out["forces"].sum(0)).max() < 1e-12 * np.abs(out["forces"]).max()
    fd = oracle.forces_dual(mc, w, b)
    assert np.abs(fd - out["forces"]).max() < 1e-12 * np.abs(fd).max()
    # energy and forces unchanged when one atom is moved by a lattice vector
    p = b.pos.copy()
    p[7] += b.cell[0][1] - 2 * b.cell[0][2]
    out2 = oracle.evaluate(mc, w, with_pos(b, p))
    assert abs(out2["energy"][0] - out["energy"][0]) < 1e-10
    assert np.allclose(out2["forces"], out["forces"], atol=1e-10)
    for (i, a) in ((3, 0), (20, 2)):
        num = _fd_force(mc, w, b, i, a, 0)
        assert abs(num - out["forces"][i, a]) < 5e-9 * max(1.0, abs(num))


# ----------------------------------------------------------------------------- stored expected values (regression)
def test_golden_cfg1_written_by_oracle_script(tiny):
    mc, w, b = tiny
    path = os.path.join(GOLD, "cfg1_oracle.npz")
    if not os.path.exists(path):
        pytest.skip("golden file not generated")
    gold = np.load(path)
    out = oracle.evaluate(mc, w, b)
    assert np.allclose(out["energy"], gold["energy"], rtol=1e-12)
    assert np.allclose(out["forces"], gold["forces"], rtol=1e-10, atol=1e-12)
    assert out["n_edges"] == int(gold["n_edges"])
