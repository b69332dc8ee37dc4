"""-m gpu: parity of the FP64 tensor-core kernels (edge_dmma.cu, gemm_dmma.cu: used by the FP64 model whenever F is a
multiple of 64) against the oracle at 1e-10, on shapes chosen to reach their branches: 1..8 k-steps of 4 radial functions
(K = 4 Bessel, 7, 20, 32: zero-padded fragments), 1..4 feature slabs, molecules (one or two 8-row tiles per receiver, rows
past the end, isolated atoms = receivers without a pass), crystals (7-8 tiles), a dense cell (more than 64 neighbours:
several passes per receiver), one block (no vector input anywhere) and several, the all-images graph (self-image edges),
row counts that are not a multiple of the 128-row GEMM tile; and the plain-ALU FP64 kernels that remain for other widths."""
import dataclasses

import numpy as np
import pytest

import gen
import oracle
from gpu_common import run_gpu
from helpers import energy_rel_err, force_rel_err, single

pytestmark = pytest.mark.gpu


def _check(mc, w, b, max_edges=None, te=1e-10, tf=1e-10):
    ref = oracle.evaluate(mc, w, b)
    out = run_gpu(mc, w, b, "fp64", max_edges=max_edges)
    assert energy_rel_err(out["energy"], ref["energy"]).max() < te
    assert force_rel_err(out["forces"], ref["forces"], b.struct_ptr).max() < tf
    eo = run_gpu(mc, w, b, "fp64", forces=False, max_edges=max_edges)      # energy-only launch sequence (no tape)
    assert energy_rel_err(eo["energy"], ref["energy"]).max() < te
    return ref


def _mol_batch(H):
    b = gen.concat_batches([gen.make_batch(2, 40, 4), single([8], [[0.0, 0.0, 0.0]], 0),
                            single([1, 6, 7], [[0, 0, 0], [0, 0, 9.5], [0.9, 0, 0]], 0), gen.make_batch(2, 90, 2)])
    return dataclasses.replace(b, head=(np.arange(b.n_structs) % H).astype(np.int32))


@pytest.mark.parametrize("F,K,H,rbf", [(64, 7, 1, "gaussian"), (128, 20, 3, "gaussian"), (192, 32, 2, "gaussian"),
                                       (256, 4, 16, "bessel"), (64, 13, 2, "bessel")])
@pytest.mark.parametrize("kind", ["mol", "xtal"])
def test_fp64_tensor_shapes(F, K, H, rbf, kind):
    mc = gen.ModelCfg(F=F, T=2, K=K, H=H, cutoff=5.0 if kind == "mol" else 6.0, rbf=rbf)
    w = gen.make_weights(mc, 300 + F + K)
    b = _mol_batch(H) if kind == "mol" else dataclasses.replace(gen.make_batch(3, 5, 1), head=np.array([H - 1], np.int32))
    _check(mc, w, b)


def test_dense_cell_several_passes_per_receiver():
    """r_c = 7.5 A in the cfg3 cell (minimum image): about 105 neighbours per atom, two passes of 64 edges per receiver."""
    mc = gen.ModelCfg(F=64, T=2, K=20, H=1, cutoff=7.5)
    w = gen.make_weights(mc, 41)
    b = dataclasses.replace(gen.make_batch(3, 2, 1), head=np.array([0], np.int32))
    ref = _check(mc, w, b, max_edges=b.n_atoms * 160)
    assert ref["n_edges"] > 64 * b.n_atoms


@pytest.mark.parametrize("T", [1, 3])
def test_one_block_and_three(T):
    mc = gen.ModelCfg(F=128, T=T, K=20, H=2, cutoff=5.0)
    w = gen.make_weights(mc, 50 + T)
    _check(mc, w, _mol_batch(2))


def test_all_images_narrow_cell():
    """A 16-atom cell narrower than the cutoff with every periodic image (self-image edges, several edges per pair)."""
    rng = np.random.default_rng(3)
    L = 4.2
    pos = rng.uniform(0, L, (16, 3))
    b = single(rng.integers(1, 9, 16), pos, 0, np.eye(3) * L, [1, 1, 1])
    mc = gen.ModelCfg(F=64, T=2, K=20, H=1, cutoff=5.0, pbc_images="all")
    w = gen.make_weights(mc, 9)
    _check(mc, w, b, max_edges=16 * 400)


def test_plain_alu_fp64_kernels_for_other_widths():
    mc = gen.ModelCfg(F=96, T=2, K=20, H=2, cutoff=5.0)
    w = gen.make_weights(mc, 5)
    _check(mc, w, _mol_batch(2))
