"""-m gpu: parity on model shapes other than the five configs, chosen to reach every tiling branch of the kernels:
feature widths that give 1, 2, 3, 4, 5 and 8 slabs of 32 (F = 32 ... 256, including widths that are not a multiple of 64
or 128), radial-basis counts on both sides of the 16-column MMA padding (K = 5, 15, 16, 20, 31, 32), one and several
heads, molecules (degree ~12), crystals (degree > 48: several staging rounds per receiver) and a mixed batch with
isolated atoms."""
import dataclasses

import numpy as np
import pytest

import gen
import oracle
from gpu_common import run_gpu
from helpers import energy_rel_err, force_rel_err, single

pytestmark = pytest.mark.gpu

SHAPES = [(32, 5, 1), (64, 15, 2), (96, 16, 3), (128, 31, 1), (160, 20, 4), (192, 32, 2), (224, 8, 1), (256, 12, 16)]


def l2_rel(a, b):
    return float(np.sqrt(((a - b) ** 2).sum() / max((b ** 2).sum(), 1e-300)))


def batch_for(kind: str, H: int) -> gen.Batch:
    if kind == "mol":
        b = gen.concat_batches([gen.make_batch(2, 40, 5), single([8], [[0.0, 0.0, 0.0]], 0),
                                single([1, 6], [[0, 0, 0], [0, 0, 9.5]], 0), gen.make_batch(2, 90, 3)])
    else:
        b = gen.make_batch(3, 11, 1)
    return dataclasses.replace(b, head=(np.arange(b.n_structs) % H).astype(np.int32))


@pytest.mark.parametrize("F,K,H", SHAPES)
@pytest.mark.parametrize("kind", ["mol", "xtal"])
@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_shapes(F, K, H, kind, precision):
    rc = 5.0 if kind == "mol" else 6.0
    mc = gen.ModelCfg(F=F, T=2, K=K, H=H, cutoff=rc)
    w = gen.make_weights(mc, 100 + F + K)
    b = batch_for(kind, H)
    out = run_gpu(mc, w, b, precision)
    ref = oracle.evaluate(mc, w, b)
    if precision == "fp32":
        assert energy_rel_err(out["energy"], ref["energy"]).max() < 1e-5
        assert force_rel_err(out["forces"], ref["forces"], b.struct_ptr).max() < 1e-4
    else:
        assert l2_rel(out["energy"], ref["energy"]) < 2e-2
        assert l2_rel(out["forces"], ref["forces"]) < (2e-2 if kind == "mol" else 8e-2)


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_energy_only_shapes(precision):
    mc = gen.ModelCfg(F=96, T=3, K=20, H=2, cutoff=5.0)
    w = gen.make_weights(mc, 77)
    b = batch_for("mol", 2)
    out = run_gpu(mc, w, b, precision, forces=False)
    ref = oracle.evaluate(mc, w, b, forces=False)
    tol = 1e-5 if precision == "fp32" else 2e-2
    assert (energy_rel_err(out["energy"], ref["energy"]).max() if precision == "fp32" else l2_rel(out["energy"], ref["energy"])) < tol


@pytest.mark.parametrize("precision", ["fp64", "fp32", "bf16"])
@pytest.mark.parametrize("F,K,kind", [(64, 4, "mol"), (256, 4, "xtal"), (128, 8, "mol"), (32, 1, "mol")])
def test_bessel_basis(F, K, kind, precision):
    """The paper's lead model uses 4 Bessel radial functions; pnn_config.rbf = PNN_RBF_BESSEL."""
    rc = 5.0 if kind == "mol" else 6.0
    mc = gen.ModelCfg(F=F, T=2, K=K, H=2, cutoff=rc, rbf="bessel")
    w = gen.make_weights(mc, 300 + F + K)
    b = batch_for(kind, 2)
    out = run_gpu(mc, w, b, precision)
    ref = oracle.evaluate(mc, w, b)
    if precision == "bf16":
        assert l2_rel(out["energy"], ref["energy"]) < 2e-2
        assert l2_rel(out["forces"], ref["forces"]) < (2e-2 if kind == "mol" else 8e-2)
    else:
        te, tf = (1e-10, 1e-10) if precision == "fp64" else (1e-5, 1e-4)
        assert energy_rel_err(out["energy"], ref["energy"]).max() < te
        assert force_rel_err(out["forces"], ref["forces"], b.struct_ptr).max() < tf
