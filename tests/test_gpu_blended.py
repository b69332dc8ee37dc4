"""-m gpu: blended multi-head evaluation (pnn_eval_blended; Fig. 5) against
oracle.evaluate_blended on the same seeded inputs: FP64 1e-10, FP32 1e-5 / 1e-4, BF16 relative L2 2e-2."""
import dataclasses

import numpy as np
import pytest

import gen
import oracle
from gpu_common import make_model, to_device
from helpers import energy_rel_err, force_rel_err

pytestmark = pytest.mark.gpu


def run_blended(mc, w, b, hw, precision, skip_below=0.0, forces=True):
    import torch
    net = make_model(mc, w, precision, b.n_atoms, b.n_atoms * 96, b.n_structs, forces)
    try:
        t = to_device(b)
        dt = torch.float64 if precision == "fp64" else torch.float32
        hwt = torch.from_numpy(np.ascontiguousarray(hw)).to(dt).cuda()
        e, f = net.eval_blended(t["Z"], t["pos"], t["struct_ptr"], hwt, t["cell"], t["pbc"], forces=forces,
                                skip_below=skip_below)
        torch.cuda.synchronize()
        net.check()
        return e.double().cpu().numpy(), None if f is None else f.double().cpu().numpy()
    finally:
        net.close()


def weights_for(S, H, seed=3):
    rng = np.random.default_rng(seed)
    hw = rng.dirichlet(0.3 * np.ones(H), size=S)          # peaked softmax-like weights, rows sum to 1
    return np.round(hw, 6)                                  # exactly representable decisions around the threshold


def l2_rel(a, b):
    return float(np.sqrt(((a - b) ** 2).sum() / (b ** 2).sum()))


@pytest.mark.parametrize("precision", ["fp64", "fp32", "bf16"])
@pytest.mark.parametrize("cfg_id,count", [(2, 12), (3, 1)])
def test_blended_matches_oracle(precision, cfg_id, count):
    mc, b = gen.model_cfg(cfg_id), gen.make_batch(cfg_id, 4, count)
    w = gen.make_weights(mc, cfg_id)
    hw = weights_for(b.n_structs, mc.H)
    skip = 0.02
    e, f = run_blended(mc, w, b, hw, precision, skip_below=skip)
    ref = oracle.evaluate_blended(mc, w, b, hw, skip_below=skip)
    if precision == "bf16":
        assert l2_rel(e, ref["energy"]) < 2e-2 and l2_rel(f, ref["forces"]) < (2e-2 if cfg_id == 2 else 8e-2)
    else:
        te, tf = (1e-10, 1e-10) if precision == "fp64" else (1e-5, 1e-4)
        assert energy_rel_err(e, ref["energy"]).max(initial=0.0) < te
        assert force_rel_err(f, ref["forces"], b.struct_ptr).max() < tf


def test_one_hot_equals_single_head_path():
    from gpu_common import run_gpu
    mc, b = gen.model_cfg(2), gen.make_batch(2, 0, 10)
    w = gen.make_weights(mc, 2)
    hw = np.zeros((b.n_structs, mc.H))
    hw[np.arange(b.n_structs), b.head] = 1.0
    e, f = run_blended(mc, w, b, hw, "fp64")
    single = run_gpu(mc, w, b, "fp64")
    assert np.abs(e - single["energy"]).max() < 1e-11 * np.abs(single["energy"]).max()
    assert np.abs(f - single["forces"]).max() < 1e-10 * np.abs(single["forces"]).max()


def test_blended_energy_only_workspace():
    mc, b = gen.model_cfg(2), gen.make_batch(2, 30, 6)
    w = gen.make_weights(mc, 2)
    hw = weights_for(b.n_structs, mc.H, seed=9)
    e, _ = run_blended(mc, w, b, hw, "fp32", forces=False)
    ref = oracle.evaluate_blended(mc, w, b, hw, forces=False)
    assert energy_rel_err(e, ref["energy"]).max() < 1e-5
