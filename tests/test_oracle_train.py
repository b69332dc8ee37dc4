"""-m "not gpu": pins of oracle/train_oracle.py, the oracle of the training step (PAPER.md:220-240
Table V).  No CUDA kernel of this step exists yet; the oracle is pinned first.  Each pin is something other than the file
itself: the hand-written C++ oracle (energies, forces, and central differences of the loss built from ITS energies and
forces), closed forms, and the optimiser of the library the paper's code base uses."""
import numpy as np
import pytest

import gen
import oracle
from oracle import train_oracle as T


def _case(n_structs=4, seed=0, cid=1):
    mc = gen.model_cfg(cid)
    w = gen.make_weights(mc, cid)
    b = gen.make_batch(cid, 0, n_structs)
    ref = oracle.evaluate(mc, w, b)
    rng = np.random.default_rng(seed)
    # labels: the model's own outputs moved by far more than any finite-difference step moves them, so that no residual
    # changes sign inside a difference quotient
    E_ref = ref["energy"] + rng.choice([-1.0, 1.0], ref["energy"].shape) * rng.uniform(0.5, 2.0, ref["energy"].shape)
    F_ref = ref["forces"] + rng.choice([-1.0, 1.0], ref["forces"].shape) * rng.uniform(0.5, 2.0, ref["forces"].shape)
    return mc, w, b, ref, E_ref, F_ref


def _loss_from_cpp_oracle(mc, w, b, E_ref, F_ref, lam):
    out = oracle.evaluate(mc, w, b)
    return np.abs(out["energy"] - E_ref).mean() + lam * np.abs(out["forces"] - F_ref).mean()


def test_torch_restatement_matches_the_cpp_oracle():
    for cid, n in ((1, 6), (2, 2)):
        mc, w, b, ref, _, _ = _case(n, cid=cid)
        E, F = T.energy_forces(mc, w, b)
        assert np.abs(E - ref["energy"]).max() <= 1e-12 * np.abs(ref["energy"]).max()
        assert np.abs(F - ref["forces"]).max() <= 1e-11 * np.abs(ref["forces"]).max()


def test_periodic_batch_matches_the_cpp_oracle():
    mc = gen.model_cfg(3)
    import dataclasses
    mc = dataclasses.replace(mc, F=32, T=2, H=2)
    w = gen.make_weights(mc, 3)
    b = gen.make_batch(3, 0, 1)
    b.head[:] = 1
    ref = oracle.evaluate(mc, w, b)
    E, F = T.energy_forces(mc, w, b)
    assert np.abs(E - ref["energy"]).max() <= 1e-12 * np.abs(ref["energy"]).max()
    assert np.abs(F - ref["forces"]).max() <= 1e-10 * np.abs(ref["forces"]).max()


@pytest.mark.parametrize("lam", [0.0, 94.8])
def test_loss_gradient_against_central_differences_of_the_cpp_oracle(lam):
    """dL/dtheta (reverse mode, second order through the forces) against (L(theta + h e_k) - L(theta - h e_k)) / 2h with L
    assembled from the C++ oracle's energies and forces: three entries of EVERY parameter array."""
    mc, w, b, ref, E_ref, F_ref = _case(4)
    L, g, mae_e, mae_f = T.loss_and_gradient(mc, w, b, E_ref, F_ref, force_weight=lam)
    assert abs(L - _loss_from_cpp_oracle(mc, w, b, E_ref, F_ref, lam)) <= 1e-12 * abs(L)
    rng = np.random.default_rng(1)
    worst = 0.0
    for name, shape, _, off in gen.weights_layout(mc):
        size = int(np.prod(shape))
        for k in off + rng.choice(size, min(3, size), replace=False):
            if name == "emb" and (k - off) // mc.F not in set(b.Z.tolist()):
                assert g[k] == 0.0                      # an element that does not occur in the batch
                continue
            h = 1e-5 * max(1.0, abs(w[k]))
            wp, wm = w.copy(), w.copy()
            wp[k] += h
            wm[k] -= h
            fd = (_loss_from_cpp_oracle(mc, wp, b, E_ref, F_ref, lam) - _loss_from_cpp_oracle(mc, wm, b, E_ref, F_ref, lam)) / (2 * h)
            err = abs(fd - g[k]) / max(abs(fd), abs(g[k]), 1e-6 * np.abs(g).max())
            worst = max(worst, err)
            assert err < 2e-6, (name, int(k - off), fd, g[k])
    assert worst > 0.0


def test_output_bias_gradient_closed_form():
    """dE_s/d(b2 of head h) = number of atoms of s if s uses head h, and the forces do not depend on it:
    dL/db2_h = (1/S) sum_s sign(E_s - E*_s) n_s [head_s = h], whatever the force weight."""
    mc = gen.model_cfg(2)
    import dataclasses
    mc = dataclasses.replace(mc, F=32, T=2, H=3)
    w = gen.make_weights(mc, 2)
    b = gen.make_batch(2, 0, 5)
    b.head[:] = np.array([0, 2, 2, 1, 0], np.int32)
    ref = oracle.evaluate(mc, w, b)
    E_ref = ref["energy"] + np.array([1.0, -2.0, 0.5, 3.0, -0.25])
    F_ref = ref["forces"] + 0.3
    _, g, _, _ = T.loss_and_gradient(mc, w, b, E_ref, F_ref, force_weight=94.8)
    lay = {name: off for name, _, _, off in gen.weights_layout(mc)}
    n_s = np.diff(b.struct_ptr)
    sign = np.sign(ref["energy"] - E_ref)
    for h in range(mc.H):
        want = (sign * n_s * (b.head == h)).sum() / b.n_structs
        assert abs(g[lay[f"h{h}.out_b2"]] - want) < 1e-12


def test_rotating_the_batch_and_its_force_labels_leaves_energy_loss_and_gradient_alone():
    mc, w, b, ref, E_ref, F_ref = _case(3)
    L0, g0, _, _ = T.loss_and_gradient(mc, w, b, E_ref, ref["forces"], force_weight=0.0)   # MAE(E) alone is invariant
    q, _ = np.linalg.qr(np.random.default_rng(5).normal(size=(3, 3)))
    b2 = gen.Batch(Z=b.Z, pos=b.pos @ q.T, struct_ptr=b.struct_ptr, head=b.head, cell=None, pbc=None)
    L1, g1, _, _ = T.loss_and_gradient(mc, w, b2, E_ref, ref["forces"] @ q.T, force_weight=0.0)
    assert abs(L0 - L1) < 1e-10 * abs(L0)
    assert np.abs(g0 - g1).max() < 1e-9 * np.abs(g0).max()


def test_adamw_first_step_closed_form_and_decay_only():
    rng = np.random.default_rng(2)
    th, g = rng.normal(size=50), rng.normal(size=50)
    lr, wd, eps = 6.34e-4, 0.01, 1e-8
    new, st = T.adamw_update(th, g, T.AdamWState())
    # t = 1: m_hat = g, v_hat = g^2  ->  theta (1 - lr wd) - lr g / (|g| + eps)
    assert np.allclose(new, th * (1 - lr * wd) - lr * g / (np.abs(g) + eps), rtol=0, atol=1e-15)
    assert st.t == 1 and np.allclose(st.m, 0.1 * g) and np.allclose(st.v, 0.001 * g * g)
    new0, _ = T.adamw_update(th, np.zeros(50), T.AdamWState())
    assert np.allclose(new0, th * (1 - lr * wd), rtol=0, atol=1e-18)      # zero gradient: decoupled decay alone


def test_adamw_written_out_equals_the_library_optimiser_over_ten_steps():
    import torch
    rng = np.random.default_rng(3)
    th0 = rng.normal(size=40)
    p = torch.tensor(th0.copy(), requires_grad=True)
    opt = torch.optim.AdamW([p], lr=T.LR, betas=T.BETAS, eps=T.EPS, weight_decay=T.WEIGHT_DECAY)
    th, st = th0.copy(), T.AdamWState()
    for step in range(10):
        g = rng.normal(size=40) * (1.0 + step)
        p.grad = torch.tensor(g.copy())
        opt.step()
        th, st = T.adamw_update(th, g, st)
        assert np.abs(p.detach().numpy() - th).max() < 1e-14


def test_steps_on_one_batch_lower_its_loss():
    mc, w, b, ref, E_ref, F_ref = _case(2)
    st, losses = None, []
    for _ in range(12):
        out = T.train_step(mc, w, b, E_ref, F_ref, st)
        w, st = out["weights"], out["state"]
        losses.append(out["loss"])
    assert st.t == 12 and losses[-1] < 0.9 * losses[0]
