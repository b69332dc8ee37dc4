"""-m gpu parity of the global attributes (charge, spin; reading Q30) against the oracle."""
import dataclasses

import numpy as np
import pytest

import gen
import oracle
from gpu_common import run_gpu
from helpers import energy_rel_err, force_rel_err

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision", ["fp64", "fp32", "bf16"])
def test_global_attributes_against_oracle(precision):
    mc = dataclasses.replace(gen.model_cfg(2), n_global=2)
    w = gen.make_weights(mc, 2)
    b = gen.make_batch(2, 3, 9)
    rng = np.random.default_rng(5)
    # (charge, spin multiplicity) scaled by 0.2: with random N(0, 1) attribute columns, raw integers blow the activations of
    # this untrained network up to 1e9, where BF16 rounding alone exceeds 2e-2
    gl = 0.2 * np.stack([rng.integers(-2, 3, b.n_structs), rng.integers(1, 4, b.n_structs)], 1).astype(np.float64)
    ref = oracle.evaluate(mc, w, b, globals_=gl)
    plain = oracle.evaluate(mc, w, b)
    assert np.abs(ref["energy"] - plain["energy"]).max() > 1e-3 * np.abs(plain["energy"]).max()   # they matter
    out = run_gpu(mc, w, b, precision, globals_=gl)
    zero = run_gpu(mc, w, b, precision)                       # no attributes given = zeros
    if precision == "bf16":
        assert np.sqrt(((out["energy"] - ref["energy"]) ** 2).sum() / (ref["energy"] ** 2).sum()) < 2e-2
        assert np.sqrt(((out["forces"] - ref["forces"]) ** 2).sum() / (ref["forces"] ** 2).sum()) < 2e-2
        assert np.sqrt(((zero["energy"] - plain["energy"]) ** 2).sum() / (plain["energy"] ** 2).sum()) < 2e-2
    else:
        te, tf = (1e-10, 1e-10) if precision == "fp64" else (1e-5, 1e-4)
        assert energy_rel_err(out["energy"], ref["energy"]).max() < te
        assert force_rel_err(out["forces"], ref["forces"], b.struct_ptr).max() < tf
        assert energy_rel_err(zero["energy"], plain["energy"]).max() < te


def test_globals_need_a_model_with_global_columns():
    import paper_2604_15380_b200 as pnn
    import torch
    from gpu_common import make_model
    mc = gen.model_cfg(1)
    b = gen.make_batch(1)
    net = make_model(mc, gen.make_weights(mc, 1), "fp32", b.n_atoms, b.n_atoms * 64, b.n_structs)
    with pytest.raises(pnn.PnnError) as ei:
        pnn.pnn_set_globals(net.ws, b.n_structs, torch.zeros((b.n_structs, 2), dtype=torch.float64, device="cuda"))
    assert ei.value.status == -1
    net.close()
