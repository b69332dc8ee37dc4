"""Pins for oracle.branch_weights — the composition -> softmax branch-weight MLP of the paper's blended inference
(reading Q28).  CPU only; none of the expected values comes from the oracle itself."""
import math

import numpy as np

import gen
import oracle


def _rand_structs(rng, S, zmax, nmax=30):
    n = rng.integers(1, nmax + 1, S)
    sp = np.concatenate([[0], np.cumsum(n)]).astype(np.int32)
    Z = rng.integers(1, zmax + 1, sp[-1]).astype(np.int32)
    return Z, sp


def test_parameter_count_matches_the_papers_24500():
    # PAPER.md:354 "comprises 24,500 parameters"; Q28's widths give 24,528.
    assert gen.branch_mlp_count(gen.BRANCH_MLP_WIDTHS) == 24528
    assert abs(gen.branch_mlp_count(gen.BRANCH_MLP_WIDTHS) - 24500) / 24500 < 2e-3
    assert gen.make_branch_mlp().shape == (24528,)


def test_rows_are_a_probability_vector_and_order_and_size_invariant():
    rng = np.random.default_rng(1)
    Z, sp = _rand_structs(rng, 12, 118)
    p = gen.make_branch_mlp()
    w = oracle.branch_weights(Z, sp, gen.BRANCH_MLP_WIDTHS, p)
    assert w.shape == (12, 16) and (w > 0).all()
    assert np.abs(w.sum(1) - 1).max() < 1e-14
    # composition does not depend on the order of the atoms ...
    Zp = Z.copy()
    for g in range(12):
        Zp[sp[g]:sp[g + 1]] = rng.permutation(Z[sp[g]:sp[g + 1]])
    assert np.abs(oracle.branch_weights(Zp, sp, gen.BRANCH_MLP_WIDTHS, p) - w).max() < 1e-14
    # ... nor on the size of the structure: a doubled structure has the same fractions
    Z2 = np.concatenate([np.tile(Z[sp[g]:sp[g + 1]], 2) for g in range(12)])
    sp2 = (2 * sp).astype(np.int32)
    assert np.abs(oracle.branch_weights(Z2, sp2, gen.BRANCH_MLP_WIDTHS, p) - w).max() < 1e-13


def test_zero_last_layer_gives_uniform_weights_and_softmax_shift_invariance():
    rng = np.random.default_rng(2)
    Z, sp = _rand_structs(rng, 5, 20)
    widths = (20, 7, 5)
    p = rng.normal(size=gen.branch_mlp_count(widths))
    last = 5 * 7 + 5
    p0 = p.copy()
    p0[-last:] = 0.0
    assert np.abs(oracle.branch_weights(Z, sp, widths, p0) - 0.2).max() < 1e-16
    p1 = p.copy()
    p1[-5:] += 3.25                                   # same constant on every logit
    assert np.abs(oracle.branch_weights(Z, sp, widths, p1) - oracle.branch_weights(Z, sp, widths, p)).max() < 1e-14


def test_two_heads_one_hidden_unit_is_a_logistic_function():
    # widths (2, 1, 2): h = silu(a1 c1 + a2 c2 + b); logits l_k = u_k h + d_k; two-class softmax = logistic of l_0 - l_1.
    a1, a2, b, u0, u1, d0, d1 = 0.7, -1.3, 0.2, 1.5, -0.4, 0.1, 0.3
    p = np.array([a1, a2, b, u0, u1, d0, d1])
    Z = np.array([1, 1, 2, 1, 2, 2, 2, 2, 1], np.int32)          # structures: {1,1,2,1}, {2,2,2,2}, {1}
    sp = np.array([0, 4, 8, 9], np.int32)
    w = oracle.branch_weights(Z, sp, (2, 1, 2), p)
    for g, (c1, c2) in enumerate([(0.75, 0.25), (0.0, 1.0), (1.0, 0.0)]):
        t = a1 * c1 + a2 * c2 + b
        h = t / (1.0 + math.exp(-t))
        w0 = 1.0 / (1.0 + math.exp(-((u0 - u1) * h + d0 - d1)))
        assert abs(w[g, 0] - w0) < 1e-15 and abs(w[g, 1] - (1 - w0)) < 1e-15


def test_against_library_routines():
    """bincount / linear / silu / softmax from numpy and torch, FP64: catches a transposed matrix, a wrong layer order, a
    missing bias or activation, an activation after the last layer, counts instead of fractions."""
    import torch
    import torch.nn.functional as Fn
    rng = np.random.default_rng(3)
    Z, sp = _rand_structs(rng, 40, 118, nmax=60)
    widths = gen.BRANCH_MLP_WIDTHS
    p = gen.make_branch_mlp()
    w = oracle.branch_weights(Z, sp, widths, p)
    comp = np.stack([np.bincount(Z[sp[g]:sp[g + 1]], minlength=119)[1:] / (sp[g + 1] - sp[g]) for g in range(40)])
    x, off = torch.tensor(comp), 0
    for l in range(3):
        n_in, n_out = widths[l], widths[l + 1]
        W = torch.tensor(p[off:off + n_in * n_out].reshape(n_out, n_in))
        off += n_in * n_out
        bb = torch.tensor(p[off:off + n_out])
        off += n_out
        x = Fn.linear(x, W, bb)
        if l < 2:
            x = Fn.silu(x)
    ref = Fn.softmax(x, dim=1).numpy()
    assert np.abs(w - ref).max() < 1e-13
    # the seeded router is as peaked as the paper's (~81 % of the branches negligible)
    b = gen.make_batch(2, 0, 256)
    wb = oracle.branch_weights(b.Z, b.struct_ptr, widths, p)
    assert 0.7 < np.mean(wb < 0.01) < 0.9


def test_empty_structure_and_pure_element():
    widths = (4, 3, 2)
    rng = np.random.default_rng(4)
    p = rng.normal(size=gen.branch_mlp_count(widths))
    W1, b1 = p[:12].reshape(3, 4), p[12:15]
    W2, b2 = p[15:21].reshape(2, 3), p[21:23]
    Z = np.array([3, 3, 3], np.int32)
    sp = np.array([0, 0, 3], np.int32)                # structure 0 empty, structure 1 pure element 3
    w = oracle.branch_weights(Z, sp, widths, p)
    for g, pre in enumerate([b1, W1[:, 2] + b1]):     # c = 0 -> biases only; c = e_3 -> third column
        h = pre / (1 + np.exp(-pre))
        l = W2 @ h + b2
        assert abs(w[g, 0] - 1 / (1 + math.exp(l[1] - l[0]))) < 1e-15
