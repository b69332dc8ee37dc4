"""-m gpu parity of the second backbone (SchNet continuous-filter convolutions, schnet.cu, DESIGN.md
reading Q31) against its oracle (oracle/schnet_oracle.py), through the same C ABI as the PaiNN path."""
import dataclasses

import numpy as np
import pytest

import gen
from gpu_common import make_model, run_gpu
from helpers import energy_rel_err, force_rel_err, single
from oracle.schnet_oracle import evaluate_schnet

pytestmark = pytest.mark.gpu

TOL = {"fp64": (1e-10, 1e-10), "fp32": (1e-5, 1e-4)}


def _mol_batch(H):
    b = gen.concat_batches([gen.make_batch(2, 40, 4), single([8], [[0.0, 0.0, 0.0]], 0),
                            single([1, 6, 7], [[0, 0, 0], [0, 0, 9.5], [0.9, 0, 0]], 0), gen.make_batch(2, 90, 2)])
    return dataclasses.replace(b, head=(np.arange(b.n_structs) % H).astype(np.int32))


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("F,K,H,T,rbf", [(32, 8, 1, 2, "gaussian"), (64, 20, 3, 3, "gaussian"), (128, 20, 16, 2, "gaussian"),
                                         (96, 4, 2, 2, "bessel"), (256, 32, 2, 1, "gaussian")])
def test_schnet_molecules(precision, F, K, H, T, rbf):
    mc = gen.ModelCfg(F=F, T=T, K=K, H=H, cutoff=5.0, rbf=rbf, backbone="schnet")
    w = gen.make_weights(mc, 500 + F + K)
    b = _mol_batch(H)
    ref = evaluate_schnet(mc, w, b)
    out = run_gpu(mc, w, b, precision)
    te, tf = TOL[precision]
    assert energy_rel_err(out["energy"], ref["energy"]).max() < te
    assert force_rel_err(out["forces"], ref["forces"], b.struct_ptr).max() < tf
    eo = run_gpu(mc, w, b, precision, forces=False)
    assert energy_rel_err(eo["energy"], ref["energy"]).max() < te


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_schnet_crystals(precision):
    mc = gen.ModelCfg(F=64, T=2, K=20, H=2, cutoff=6.0, backbone="schnet")
    w = gen.make_weights(mc, 61)
    b = dataclasses.replace(gen.make_batch(3, 4, 2), head=np.array([1, 0], np.int32))
    ref = evaluate_schnet(mc, w, b)
    out = run_gpu(mc, w, b, precision)
    te, tf = TOL[precision]
    assert energy_rel_err(out["energy"], ref["energy"]).max() < te
    assert force_rel_err(out["forces"], ref["forces"], b.struct_ptr).max() < (tf if precision == "fp64" else 1e-3)


def test_schnet_all_images_and_unsupported_options():
    import paper_2604_15380_b200 as pnn
    rng = np.random.default_rng(3)
    L = 4.2
    b = single(rng.integers(1, 9, 16), rng.uniform(0, L, (16, 3)), 0, np.eye(3) * L, [1, 1, 1])
    mc = gen.ModelCfg(F=64, T=2, K=12, H=1, cutoff=5.0, pbc_images="all", backbone="schnet")
    w = gen.make_weights(mc, 9)
    ref = evaluate_schnet(mc, w, b)
    out = run_gpu(mc, w, b, "fp64", max_edges=16 * 400)
    assert energy_rel_err(out["energy"], ref["energy"]).max() < 1e-10
    assert force_rel_err(out["forces"], ref["forces"], b.struct_ptr).max() < 1e-10
    for kw in (dict(precision="bf16"), dict(max_neighbors=20), dict(head_type="pooled")):
        with pytest.raises(pnn.PnnError):
            mcx = dataclasses.replace(mc, **{k: v for k, v in kw.items() if k != "precision"})
            make_model(mcx, gen.make_weights(mcx, 9) if kw.get("head_type") is None else np.zeros(1), kw.get("precision", "fp32"),
                       16, 6400, 1)
