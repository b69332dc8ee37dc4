"""Pins of the oracle's pooled graph-level head ("Output heads 16 (graph-level)", "2 shared layers (dim 50) +
2 branch layers (dim 776)"; reading Q29): x_g = mean_i s_i -> 2 shared Linear+SiLU (d1) -> per head 2 Linear+SiLU
(d2) -> linear output."""
import dataclasses

import numpy as np

import gen
import oracle
from helpers import single


def _mc(**kw):
    return dataclasses.replace(gen.model_cfg(1), head_type="pooled", head_d1=10, head_d2=24, H=3, **kw)


def _silu(x):
    return x / (1.0 + np.exp(-x))


def _head_numpy(mc, w, s, sptr, head):
    """Independent restatement of the head alone, on the trunk features the oracle reports."""
    L = {n: (sh, off) for n, sh, _, off in gen.weights_layout(mc)}
    g = lambda n: w[L[n][1]:L[n][1] + int(np.prod(L[n][0]))].reshape(L[n][0])
    out = []
    for q in range(len(head)):
        x = s[sptr[q]:sptr[q + 1]].mean(0)
        y = _silu(g("pool.W1") @ x + g("pool.b1"))
        y = _silu(g("pool.W2") @ y + g("pool.b2"))
        h = head[q]
        z = _silu(g(f"h{h}.br_W1") @ y + g(f"h{h}.br_b1"))
        z = _silu(g(f"h{h}.br_W2") @ z + g(f"h{h}.br_b2"))
        out.append(g(f"h{h}.br_w3") @ z + g(f"h{h}.br_b3")[0])
    return np.array(out)


def test_parameter_count_of_the_papers_head():
    """16 heads x (50*776 + 776 + 776*776 + 776 + 776 + 1) + shared (337*50 + 50 + 50*50 + 50): with the lead model's trunk
    (hidden 337, 2 blocks, 4 radial functions; Table V) the total is the paper's 'about 12.1 M parameters'."""
    mc = gen.ModelCfg(F=352, T=2, K=4, H=16, head_type="pooled", head_d1=50, head_d2=776)   # F: multiple of 32 near 337
    n = gen.weights_count(mc)
    assert n == oracle.weights_count(mc)
    heads = 16 * (50 * 776 + 776 + 776 * 776 + 776 + 776 + 1) + 352 * 50 + 50 + 50 * 50 + 50
    assert n - heads == 87 * 352 + 2 * (11 * 352 * 352 + 3 * 352 * 4 + 11 * 352)
    assert 11.5e6 < n < 13.5e6


def test_energy_is_the_mlp_of_the_mean_feature():
    mc = _mc()
    w = gen.make_weights(mc, 1)
    b = dataclasses.replace(gen.make_batch(1, 0, 5), head=np.array([0, 2, 1, 2, 0], np.int32))
    out = oracle.evaluate(mc, w, b, features=True)
    ref = _head_numpy(mc, w, out["s"], b.struct_ptr, b.head)
    assert np.allclose(out["energy"], ref, rtol=1e-13, atol=1e-13)
    # head locality
    b2 = dataclasses.replace(b, head=np.array([0, 1, 1, 2, 0], np.int32))
    o2 = oracle.evaluate(mc, w, b2)
    same = [0, 2, 3, 4]
    assert np.array_equal(o2["energy"][same], out["energy"][same]) and o2["energy"][1] != out["energy"][1]
    assert np.array_equal(o2["forces"][b.struct_ptr[2]:], out["forces"][b.struct_ptr[2]:])


def test_mean_pooling_is_size_invariant():
    """Two copies of a molecule farther apart than the cutoff inside ONE structure have the features of the single molecule,
    so the mean-pooled head gives the same energy (a sum-pooled or atom-wise head would give twice the energy)."""
    mc = _mc()
    w = gen.make_weights(mc, 1)
    one = gen.make_batch(1, 0, 1)
    two = single(np.concatenate([one.Z, one.Z]), np.concatenate([one.pos, one.pos + np.array([40.0, 0, 0])]), head=0)
    e1 = oracle.evaluate(mc, w, one)
    e2 = oracle.evaluate(mc, w, two)
    assert np.allclose(e2["energy"], e1["energy"], rtol=1e-12)
    assert np.allclose(e2["forces"][:one.n_atoms], 0.5 * e1["forces"], rtol=1e-10, atol=1e-12)   # each copy carries half


def test_forces_are_the_gradient_of_the_pooled_energy():
    mc = _mc()
    w = gen.make_weights(mc, 1)
    b = dataclasses.replace(gen.make_batch(1, 0, 2), head=np.array([1, 2], np.int32))
    out = oracle.evaluate(mc, w, b)
    fd = oracle.forces_dual(mc, w, b)
    assert np.abs(out["forces"] - fd).max() < 1e-11 * np.abs(fd).max()
    h = 1e-5
    for (i, c) in ((0, 0), (17, 2)):
        p = b.pos.copy(); p[i, c] += h
        ep = oracle.evaluate(mc, w, dataclasses.replace(b, pos=p), forces=False)["energy"].sum()
        p[i, c] -= 2 * h
        em = oracle.evaluate(mc, w, dataclasses.replace(b, pos=p), forces=False)["energy"].sum()
        assert abs(-(ep - em) / (2 * h) - out["forces"][i, c]) < 1e-6 * np.abs(out["forces"]).max()
    for g in range(b.n_structs):
        f = out["forces"][b.struct_ptr[g]:b.struct_ptr[g + 1]]
        assert np.abs(f.sum(0)).max() < 1e-10 * np.abs(f).max()
