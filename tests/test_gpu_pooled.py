"""-m gpu parity of the pooled graph-level heads (reading Q29) against the oracle."""
import dataclasses

import numpy as np
import pytest

import gen
import oracle
from gpu_common import make_model, run_gpu
from helpers import energy_rel_err, force_rel_err

pytestmark = pytest.mark.gpu


def _l2(a, b):
    return np.sqrt(((a - b) ** 2).sum() / (b ** 2).sum())


@pytest.mark.parametrize("precision", ["fp64", "fp32", "bf16"])
@pytest.mark.parametrize("cfg_id,d1,d2,n_structs", [(1, 10, 24, 7), (2, 50, 776, 21)])
def test_pooled_head_against_oracle(precision, cfg_id, d1, d2, n_structs):
    """cfg2 with the paper's head widths (50, 776) and 16 heads; 21 structures over 16 heads: tiles of one to three
    structures, heads without any structure, and (FP64, groups of 4 / FP32, groups of 8) ragged tiles."""
    mc = dataclasses.replace(gen.model_cfg(cfg_id), head_type="pooled", head_d1=d1, head_d2=d2)
    w = gen.make_weights(mc, cfg_id)
    b = gen.make_batch(cfg_id, 1, n_structs)
    if cfg_id == 2:   # pile several structures on one head so that one head spans more than one tile
        hd = b.head.copy(); hd[:11] = 3
        b = dataclasses.replace(b, head=hd)
    ref = oracle.evaluate(mc, w, b)
    out = run_gpu(mc, w, b, precision)
    eonly = run_gpu(mc, w, b, precision, forces=False)
    assert np.array_equal(eonly["energy"], out["energy"])
    if precision == "bf16":
        assert _l2(out["energy"], ref["energy"]) < 2e-2
        assert _l2(out["forces"], ref["forces"]) < 2e-2
    else:
        te, tf = (1e-10, 1e-10) if precision == "fp64" else (1e-5, 1e-4)
        assert energy_rel_err(out["energy"], ref["energy"]).max() < te
        assert force_rel_err(out["forces"], ref["forces"], b.struct_ptr).max() < tf


def test_pooled_head_periodic_and_capped():
    """cfg3 (periodic cells) with the max-neighbour cap: pooled adjoint into the scatter-form reverse sweep."""
    mc = dataclasses.replace(gen.model_cfg(3), head_type="pooled", head_d1=16, head_d2=40, max_neighbors=20)
    w = gen.make_weights(mc, 3)
    b = gen.make_batch(3, 0, 2, n_atoms=54)
    ref = oracle.evaluate(mc, w, b)
    out = run_gpu(mc, w, b, "fp64")
    assert energy_rel_err(out["energy"], ref["energy"]).max() < 1e-10
    assert force_rel_err(out["forces"], ref["forces"], b.struct_ptr).max() < 1e-10


def test_bad_head_index_and_blended_call():
    import paper_2604_15380_b200 as pnn
    import torch
    mc = dataclasses.replace(gen.model_cfg(1), head_type="pooled", head_d1=10, head_d2=24)
    w = gen.make_weights(mc, 1)
    b = gen.make_batch(1, 0, 4)
    bad = dataclasses.replace(b, head=np.array([0, mc.H, 1, 0], np.int32))
    with pytest.raises(pnn.PnnError) as ei:
        run_gpu(mc, w, bad, "fp32")
    assert ei.value.status == -6
    net = make_model(mc, w, "fp32", b.n_atoms, b.n_atoms * 64, b.n_structs)
    try:
        t = dict(Z=torch.from_numpy(b.Z.astype(np.int32)).cuda(), pos=torch.from_numpy(b.pos).cuda(),
                 sptr=torch.from_numpy(b.struct_ptr.astype(np.int32)).cuda())
        hw = torch.full((b.n_structs, mc.H), 1.0 / mc.H, dtype=torch.float32, device="cuda")
        with pytest.raises(pnn.PnnError) as ei:
            net.eval_blended(t["Z"], t["pos"], t["sptr"], hw)
        assert ei.value.status == -4
    finally:
        net.close()
