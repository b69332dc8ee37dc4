"""-m gpu: pnn_eval_replay (graph build + evaluation recorded once into a CUDA graph and replayed while the atoms move in place)
against the eager path pnn_build_graph + pnn_eval: bit for bit, over a short "trajectory" in which the edge set changes."""
import dataclasses

import numpy as np
import pytest

import gen
import oracle
from gpu_common import make_model, to_device
from helpers import energy_rel_err, force_rel_err

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision,cfg_id,n", [("fp64", 1, 8), ("fp32", 2, 12), ("bf16", 2, 12), ("fp32", 3, 2)])
def test_replay_matches_eager_along_a_trajectory(precision, cfg_id, n):
    import torch
    mc = gen.model_cfg(cfg_id)
    w = gen.make_weights(mc, cfg_id)
    b = gen.make_batch(cfg_id, 0, n)
    net = make_model(mc, w, precision, b.n_atoms, b.n_atoms * 96, b.n_structs, True)
    ref_net = make_model(mc, w, precision, b.n_atoms, b.n_atoms * 96, b.n_structs, True)
    try:
        t = to_device(b)
        pos = t["pos"].clone()
        energy = torch.empty(b.n_structs, dtype=net.out_dtype, device="cuda")
        forces = torch.empty((b.n_atoms, 3), dtype=net.out_dtype, device="cuda")
        rng = np.random.default_rng(1)
        edge_counts = set()
        for step in range(7):          # calls 0 and 1 eager, call 2 records, calls 3.. replay
            if step:
                pos += torch.from_numpy(rng.normal(0, 0.15, (b.n_atoms, 3))).cuda()    # in place: same buffer
            net.eval_replay(t["Z"], pos, t["struct_ptr"], t["head"], energy, forces, t["cell"], t["pbc"])
            e_ref, f_ref = ref_net.eval(t["Z"], pos, t["struct_ptr"], t["head"], t["cell"], t["pbc"])
            torch.cuda.synchronize()
            net.check(); ref_net.check()
            assert torch.equal(energy, e_ref), step
            assert torch.equal(forces, f_ref), step
            edge_counts.add(int(net.graph()[0][-1]))
        assert len(edge_counts) > 1                                   # the graph really changed under the replayed launch list
        # and the last frame against the oracle
        bb = dataclasses.replace(b, pos=pos.cpu().numpy())
        ref = oracle.evaluate(mc, w, bb)
        te, tf = {"fp64": (1e-10, 1e-10), "fp32": (1e-5, 1e-3 if cfg_id == 3 else 1e-4), "bf16": (6e-2, 2e-1)}[precision]
        assert energy_rel_err(energy.double().cpu().numpy(), ref["energy"]).max() < te
        assert force_rel_err(forces.double().cpu().numpy(), ref["forces"], b.struct_ptr).max() < tf
        # a new signature (energy only, other output buffer) drops the recorded graph and still works
        e2 = torch.empty_like(energy)
        for _ in range(4):
            net.eval_replay(t["Z"], pos, t["struct_ptr"], t["head"], e2, None, t["cell"], t["pbc"])
        torch.cuda.synchronize()
        assert torch.equal(e2, energy)
    finally:
        net.close()
        ref_net.close()


@pytest.mark.parametrize("precision", ["fp32", "bf16"])
def test_eval_host_replays_when_the_shape_repeats(precision):
    """pnn_eval_host records its device part on the third call with the same batch shape: every call gives the same bits, a
    batch of another shape in between runs eagerly, and moving the atoms (same shape) is picked up by the replayed graph."""
    mc = gen.model_cfg(2)
    w = gen.make_weights(mc, 2)
    b1, b2 = gen.make_batch(2, 0, 10), gen.make_batch(2, 10, 7)
    net = make_model(mc, w, precision, max(b1.n_atoms, b2.n_atoms), max(b1.n_atoms, b2.n_atoms) * 40, 10, True)
    ref_net = make_model(mc, w, precision, max(b1.n_atoms, b2.n_atoms), max(b1.n_atoms, b2.n_atoms) * 40, 10, True)
    try:
        def host(n, b):
            e, f = n.eval_host(b.Z, b.pos, b.struct_ptr, b.head, forces=True)
            return e.copy(), f.copy()
        e1, f1 = host(ref_net, b1)
        e2, f2 = host(ref_net, b2)
        for k in range(5):
            e, f = host(net, b1)
            assert np.array_equal(e, e1) and np.array_equal(f, f1), k
        e, f = host(net, b2)
        assert np.array_equal(e, e2) and np.array_equal(f, f2)
        moved = dataclasses.replace(b1, pos=b1.pos + np.random.default_rng(0).normal(0, 0.1, b1.pos.shape))
        em, fm = host(ref_net, moved)
        for k in range(4):
            e, f = host(net, moved if k != 1 else b1)     # same shape, other positions: the same recorded graph
            assert np.array_equal(e, e1 if k == 1 else em) and np.array_equal(f, f1 if k == 1 else fm), k
    finally:
        net.close()
        ref_net.close()


@pytest.mark.parametrize("cfg_id,precision,n", [(2, "fp32", 256), (3, "fp32", 64), (3, "bf16", 64), (4, "bf16", 4096),
                                                (5, "fp64", 1)])
def test_replay_matches_eager_at_the_sizes_bench_times(cfg_id, precision, n):
    """The launch configuration bench.py times (whole cfg2 / cfg3 / cfg5 batches, a quarter of a cfg4 batch): the replayed
    step -- persistent tcgen05 GEMMs with TMA stores, the split-K cluster GEMM, the FP64 tensor-core kernels, the forked
    graph build -- returns what the kernel-by-kernel path returns, bit for bit."""
    import torch
    mc = gen.model_cfg(cfg_id)
    w = gen.make_weights(mc, cfg_id)
    b = gen.make_batch(cfg_id, 0, n)
    want_f = cfg_id != 4
    net = make_model(mc, w, precision, b.n_atoms, b.n_atoms * (96 if cfg_id in (3, 5) else 40), b.n_structs, want_f)
    try:
        t = to_device(b)
        e_ref, f_ref = net.eval(t["Z"], t["pos"], t["struct_ptr"], t["head"], t["cell"], t["pbc"])
        e_ref = e_ref.clone()
        f_ref = None if f_ref is None else f_ref.clone()
        energy = torch.empty(b.n_structs, dtype=net.out_dtype, device="cuda")
        forces = torch.empty((b.n_atoms, 3), dtype=net.out_dtype, device="cuda") if want_f else None
        for _ in range(5):             # calls 0 and 1 eager, call 2 records, calls 3 and 4 replay
            energy.fill_(float("nan"))
            net.eval_replay(t["Z"], t["pos"], t["struct_ptr"], t["head"], energy, forces, t["cell"], t["pbc"])
        torch.cuda.synchronize()
        net.check()
        assert torch.equal(energy, e_ref)
        if want_f:
            assert torch.equal(forces, f_ref)
    finally:
        net.close()
