"""-m gpu: the composition -> softmax router (pnn_branch_weights, reading Q28)
against oracle.branch_weights, and the whole Fig. 5 pipeline (router -> branch skipping -> blended energy -> one reverse
sweep) against the oracle's router feeding oracle.evaluate_blended.  Weights lie in [0,1]: absolute tolerances 1e-12 (FP64
router) and 2e-5 (FP32 router: logits of size ~30 carry 1e-6 of FP32 rounding)."""
import numpy as np
import pytest

import gen
import oracle
from gpu_common import make_model, to_device
from helpers import energy_rel_err, force_rel_err

pytestmark = pytest.mark.gpu
WIDTHS = gen.BRANCH_MLP_WIDTHS


def gpu_weights(net, Z, sp):
    import torch
    hw = net.branch_weights(torch.from_numpy(np.ascontiguousarray(Z, np.int32)).cuda(),
                            torch.from_numpy(np.ascontiguousarray(sp, np.int32)).cuda())
    torch.cuda.synchronize()
    return hw.double().cpu().numpy()


def ragged_composition_batch():
    """cfg2 molecules plus the degenerate cases: an empty structure, pure elements, element 118, one big structure; 261
    structures = 65 full CTAs of 4 and a tail of 1."""
    b = gen.make_batch(2, 0, 256)
    rng = np.random.default_rng(11)
    extra = [np.zeros(0, np.int32), np.full(7, 26, np.int32), np.array([118], np.int32),
             rng.integers(1, 119, 5000).astype(np.int32), np.array([1, 118, 1, 8], np.int32)]
    Z = np.concatenate([b.Z] + extra).astype(np.int32)
    sp = np.concatenate([b.struct_ptr, b.struct_ptr[-1] + np.cumsum([len(x) for x in extra])]).astype(np.int32)
    return Z, sp


@pytest.mark.parametrize("precision,tol", [("fp64", 1e-12), ("fp32", 2e-5), ("bf16", 2e-5)])
def test_router_matches_oracle(precision, tol):
    mc = gen.model_cfg(2)
    Z, sp = ragged_composition_batch()
    p = gen.make_branch_mlp()
    net = make_model(mc, gen.make_weights(mc, 2), precision, 16, 64, 8, False)
    try:
        net.set_branch_mlp(WIDTHS, p)
        w = gpu_weights(net, Z, sp)
        net.check()
    finally:
        net.close()
    ref = oracle.branch_weights(Z, sp, WIDTHS, p)
    assert w.shape == ref.shape == (261, 16)
    assert np.abs(w - ref).max() < tol
    assert np.abs(w.sum(1) - 1).max() < (1e-12 if precision == "fp64" else 1e-5)


def test_other_widths_and_single_layer():
    mc = gen.model_cfg(1)                                         # H = 1 ... use a router with its own head count
    rng = np.random.default_rng(5)
    Z = rng.integers(1, 11, 333).astype(np.int32)
    sp = np.array([0, 1, 1, 50, 333], np.int32)
    from paper_2604_15380_b200 import binding as B
    import torch
    net = make_model(mc, gen.make_weights(mc, 1), "fp64", 16, 64, 8, False)
    try:
        for widths in [(10, 3), (10, 256, 5), (10, 33, 17, 9, 2)]:
            p = rng.normal(size=gen.branch_mlp_count(widths))
            h = B.pnn_branch_mlp_create(widths, p, B.PNN_FP64)
            out = torch.empty((4, widths[-1]), dtype=torch.float64, device="cuda")
            B.pnn_branch_weights(h, net.ws, 333, 4, torch.from_numpy(Z).cuda(), torch.from_numpy(sp).cuda(), out)
            torch.cuda.synchronize()
            B.pnn_branch_mlp_destroy(h)
            assert np.abs(out.cpu().numpy() - oracle.branch_weights(Z, sp, widths, p)).max() < 1e-12
        net.check()
    finally:
        net.close()


def test_errors():
    from paper_2604_15380_b200 import binding as B
    import torch
    p = gen.make_branch_mlp()
    with pytest.raises(B.PnnError):
        B.pnn_branch_mlp_create(WIDTHS, p[:-1], B.PNN_FP32)       # parameter count does not match the widths
    with pytest.raises(B.PnnError):
        B.pnn_branch_mlp_create((118, 300, 16), np.zeros(118 * 300 + 300 + 300 * 16 + 16), B.PNN_FP32)
    mc = gen.model_cfg(2)
    net = make_model(mc, gen.make_weights(mc, 2), "fp32", 16, 64, 8, False)
    try:
        net.set_branch_mlp(WIDTHS, p)
        gpu_weights(net, np.array([1, 119, 6], np.int32), np.array([0, 3], np.int32))
        with pytest.raises(B.PnnError) as ei:
            net.check()
        assert ei.value.status == -6                              # PNN_ERR_BAD_INPUT
        with pytest.raises(ValueError):
            net.set_branch_mlp((118, 8, 4), np.zeros(gen.branch_mlp_count((118, 8, 4))))     # 4 heads != H
    finally:
        net.close()


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_fig5_pipeline_router_skipping_blend_one_reverse_sweep(precision):
    import torch
    mc, b = gen.model_cfg(2), gen.make_batch(2, 40, 10)
    w, p = gen.make_weights(mc, 2), gen.make_branch_mlp()
    skip = 0.01
    hw_ref = oracle.branch_weights(b.Z, b.struct_ptr, WIDTHS, p)
    # the skipping decision w < 0.01 must not hinge on FP32 rounding of the router for this seeded batch
    assert np.abs(hw_ref - skip).min() > 1e-4
    assert np.mean(hw_ref < skip) > 0.5
    ref = oracle.evaluate_blended(mc, w, b, hw_ref, skip_below=skip)
    net = make_model(mc, w, precision, b.n_atoms, b.n_atoms * 96, b.n_structs, True)
    try:
        net.set_branch_mlp(WIDTHS, p)
        t = to_device(b)
        hw = net.branch_weights(t["Z"], t["struct_ptr"])
        e, f = net.eval_blended(t["Z"], t["pos"], t["struct_ptr"], hw, t["cell"], t["pbc"], skip_below=skip)
        torch.cuda.synchronize()
        net.check()
        e, f = e.double().cpu().numpy(), f.double().cpu().numpy()
    finally:
        net.close()
    # FP32: the router's 1e-6 weight error enters E linearly on top of the model's own 1e-5 / 1e-4
    te, tf = (1e-10, 1e-10) if precision == "fp64" else (2e-5, 1e-4)
    assert energy_rel_err(e, ref["energy"]).max() < te
    assert force_rel_err(f, ref["forces"], b.struct_ptr).max() < tf
