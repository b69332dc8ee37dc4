"""-m gpu: the model variants of the widened scope (pooled heads, max-neighbour cap, second backbone) through the HOST entry
points — pnn_eval_host and the streaming driver — not only through pnn_eval: same values as the device-pointer path bit for
bit (same kernels, same launch order), and the oracle on top."""
import dataclasses

import numpy as np
import pytest

import gen
import oracle
from gpu_common import make_model, run_gpu
from helpers import energy_rel_err, force_rel_err
from oracle.schnet_oracle import evaluate_schnet

pytestmark = pytest.mark.gpu

VARIANTS = {
    "pooled": dict(head_type="pooled", head_d1=50, head_d2=72),
    "cap": dict(max_neighbors=12),
    "schnet": dict(backbone="schnet"),
}


@pytest.mark.parametrize("variant", sorted(VARIANTS))
def test_variants_through_eval_host_and_stream(variant):
    import paper_2604_15380_b200 as pnn
    import torch
    mc = dataclasses.replace(gen.ModelCfg(F=64, T=2, K=20, H=3, cutoff=5.0), **VARIANTS[variant])
    w = gen.make_weights(mc, 11)
    batches = [dataclasses.replace(b, head=(np.arange(b.n_structs) % mc.H).astype(np.int32))
               for b in (gen.make_batch(2, 0, 9), gen.make_batch(2, 9, 5), gen.make_batch(2, 14, 9))]
    maxN = max(b.n_atoms for b in batches)
    net = make_model(mc, w, "fp32", maxN, maxN * 40, 9, True)
    st = pnn.pnn_stream_create(net.model, maxN, maxN * 40, 9, pnn.PNN_ENERGY | pnn.PNN_FORCES, 2)
    try:
        eo = [np.zeros(b.n_structs, np.float32) for b in batches]
        fo = [np.zeros((b.n_atoms, 3), np.float32) for b in batches]
        for k, b in enumerate(batches):
            pnn.pnn_stream_submit(st, b.n_atoms, b.n_structs, b.Z, b.pos, b.struct_ptr, b.head, None, None, eo[k], fo[k])
        pnn.pnn_stream_drain(st)
        for k, b in enumerate(batches):
            e, f = net.eval_host(b.Z, b.pos, b.struct_ptr, b.head, forces=True)
            dev = run_gpu(mc, w, b, "fp32")
            if variant != "cap":   # the scatter-form reverse sweep of capped graphs adds forces with atomics: order varies
                assert np.array_equal(e, eo[k]) and np.array_equal(f, fo[k])
                assert np.array_equal(e, dev["energy"].astype(np.float32)) and np.array_equal(f, dev["forces"].astype(np.float32))
            else:
                assert np.array_equal(e, eo[k]) and np.allclose(f, fo[k], rtol=0, atol=1e-5 * np.abs(f).max())
            ref = evaluate_schnet(mc, w, b) if variant == "schnet" else oracle.evaluate(mc, w, b)
            assert energy_rel_err(eo[k], ref["energy"]).max() < 1e-5
            assert force_rel_err(fo[k], ref["forces"], b.struct_ptr).max() < 1e-4
    finally:
        pnn.pnn_stream_destroy(st)
        net.close()
