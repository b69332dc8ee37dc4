"""-m gpu: the all-images periodic radius graph (pnn_config.pbc_images = PNN_IMAGES_ALL) against the oracle: edge sets
bit-exact after canonical sort (several edges per ordered pair and self-image edges included), then energies and forces
in FP64 / FP32 / BF16 on cells narrower than twice the cutoff."""
import dataclasses

import numpy as np
import pytest

import gen
import oracle
from gpu_common import gpu_edge_set, run_gpu
from helpers import edge_set, energy_rel_err, force_rel_err, single

pytestmark = pytest.mark.gpu


def narrow_cell(n, L, seed, tric=False):
    rng = np.random.default_rng(seed)
    C = np.eye(3) * L
    if tric:
        C = np.array([[L, 0.0, 0.0], [0.3 * L, 0.9 * L, 0.0], [0.1 * L, -0.2 * L, 1.1 * L]])
    pos = rng.uniform(-0.2, 1.2, (n, 3)) @ C                      # some atoms outside the cell (Q14)
    return single(rng.integers(1, 9, n), pos, 0, C, [1, 1, 1])


def cases():
    one = single([6], [[0.3, 0.1, 0.2]], 0, np.eye(3) * 2.4, [1, 1, 1])          # every neighbour is a self image
    slab = dataclasses.replace(narrow_cell(14, 6.5, 4), pbc=np.array([[1, 1, 0]], np.uint8))
    mixed = gen.concat_batches([gen.make_batch(2, 0, 3), narrow_cell(9, 7.0, 1), one, gen.make_batch(3, 5, 1),
                                gen.make_batch(5, n_atoms=600), narrow_cell(12, 8.0, 2, tric=True), slab])
    return {"narrow": narrow_cell(10, 7.0, 2), "one_atom": one, "triclinic": narrow_cell(12, 8.0, 3, tric=True),
            "slab": slab, "cfg3": gen.make_batch(3, 2, 2), "mixed": mixed}


@pytest.mark.parametrize("name", ["narrow", "one_atom", "triclinic", "slab", "cfg3", "mixed"])
def test_graph_all_images_bit_exact(name):
    b = cases()[name]
    rc = 6.0 if name == "cfg3" else 5.0
    mc = dataclasses.replace(gen.model_cfg(1), cutoff=rc, H=16, pbc_images="all")
    out = run_gpu(mc, gen.make_weights(mc, 1), b, "fp32", forces=False, want_graph=True, max_edges=b.n_atoms * 160 + 256)
    nb = oracle.neighbours(b, rc, all_images=True)
    assert np.array_equal(out["rowptr"], nb["rowptr"])
    assert gpu_edge_set(out["rowptr"], out["col"], out["shift"]) == edge_set(nb)
    assert len(out["col"]) == len(nb["send"]) > 0


@pytest.mark.parametrize("precision", ["fp64", "fp32", "bf16"])
@pytest.mark.parametrize("name", ["narrow", "one_atom", "cfg3"])
def test_values_all_images(name, precision):
    b = cases()[name]
    if name == "cfg3":
        mc = dataclasses.replace(gen.model_cfg(3), T=2, pbc_images="all")
    else:
        mc = dataclasses.replace(gen.model_cfg(2), T=2, pbc_images="all")
    w = gen.make_weights(mc, 21)
    out = run_gpu(mc, w, b, precision, max_edges=b.n_atoms * 160 + 256)
    ref = oracle.evaluate(mc, w, b)
    if precision == "bf16":
        l2 = lambda a, r: float(np.sqrt(((a - r) ** 2).sum() / max((r ** 2).sum(), 1e-300)))
        assert l2(out["energy"], ref["energy"]) < 2e-2
        if name != "one_atom":                                     # one atom: the force is zero by symmetry
            assert l2(out["forces"], ref["forces"]) < 8e-2
    else:
        te, tf = (1e-10, 1e-10) if precision == "fp64" else (1e-5, 1e-4)
        assert energy_rel_err(out["energy"], ref["energy"]).max() < te
        if name == "one_atom":
            assert np.abs(out["forces"]).max() <= tf * max(1.0, np.abs(ref["energy"]).max())
        else:
            assert force_rel_err(out["forces"], ref["forces"], b.struct_ptr).max() < tf
