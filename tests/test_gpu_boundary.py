"""-m gpu tests of the boundary's error behaviour (include/pnn.h): stale graphs, edge overflow, host entry point errors,
pointer type checks of the binding."""
import dataclasses

import numpy as np
import pytest

import gen
import oracle
from gpu_common import make_model, to_device
from helpers import energy_rel_err, force_rel_err

pytestmark = pytest.mark.gpu


def test_moved_atoms_without_a_rebuild_are_reported():
    """pnn.h: pnn_eval uses the graph last built "for the same pos": positions that changed since pnn_build_graph are
    detected on the device (checksum) and reported as PNN_ERR_NO_GRAPH by pnn_check_async_errors."""
    import paper_2604_15380_b200 as pnn
    import torch
    mc, b = gen.model_cfg(1), gen.make_batch(1)
    w = gen.make_weights(mc, 1)
    net = make_model(mc, w, "fp64", b.n_atoms, b.n_atoms * 64, b.n_structs)
    t = to_device(b)
    e0, f0 = net.eval(t["Z"], t["pos"], t["struct_ptr"], t["head"])
    net.check()
    # same positions in another buffer: fine
    e1, _ = net.eval(t["Z"], t["pos"].clone(), t["struct_ptr"], t["head"], build=False)
    net.check()
    assert torch.equal(e0, e1)
    moved = t["pos"].clone()
    moved[3, 1] += 1e-3
    net.eval(t["Z"], moved, t["struct_ptr"], t["head"], build=False)
    with pytest.raises(pnn.PnnError) as ei:
        net.check()
    assert ei.value.status == -5
    # after a rebuild the moved positions evaluate, and match the oracle
    e2, f2 = net.eval(t["Z"], moved, t["struct_ptr"], t["head"])
    net.check()
    ref = oracle.evaluate(mc, w, dataclasses.replace(b, pos=moved.cpu().numpy()))
    assert energy_rel_err(e2.cpu().numpy(), ref["energy"]).max() < 1e-10
    assert force_rel_err(f2.cpu().numpy(), ref["forces"], b.struct_ptr).max() < 1e-10
    net.close()


@pytest.mark.parametrize("precision", ["fp64", "fp32", "bf16"])
def test_edge_overflow_is_never_evaluated_and_does_not_stick(precision):
    """An overflowing graph: pnn_eval's edge kernels do not touch memory past max_edges, the overflow is reported once as
    PNN_ERR_CAPACITY, pnn_eval then returns PNN_ERR_NO_GRAPH until the next build, and a later batch that fits is evaluated
    correctly (the flag of the old graph does not silence its kernels)."""
    import paper_2604_15380_b200 as pnn
    import torch
    mc = gen.model_cfg(2)
    big, small = gen.make_batch(2, 0, 6), gen.make_batch(2, 9, 2)
    w = gen.make_weights(mc, 2)
    ref = oracle.evaluate(mc, w, small)
    cap = ref["n_edges"] + 8
    assert oracle.neighbours(big, mc.cutoff)["recv"].size > cap
    net = make_model(mc, w, precision, big.n_atoms, cap, big.n_structs)
    tb, ts = to_device(big), to_device(small)
    net.eval(tb["Z"], tb["pos"], tb["struct_ptr"], tb["head"])          # overflows; must not fault
    torch.cuda.synchronize()
    with pytest.raises(pnn.PnnError) as ei:
        net.check()
    assert ei.value.status == -2
    with pytest.raises(pnn.PnnError) as ei:                             # the truncated graph is gone
        net.eval(tb["Z"], tb["pos"], tb["struct_ptr"], tb["head"], build=False)
    assert ei.value.status == -5
    # overflow NOT yet checked, then a fitting batch: its kernels must run
    net.eval(tb["Z"], tb["pos"], tb["struct_ptr"], tb["head"])
    e, f = net.eval(ts["Z"], ts["pos"], ts["struct_ptr"], ts["head"])
    torch.cuda.synchronize()
    e, f = e.double().cpu().numpy(), f.double().cpu().numpy()
    if precision == "bf16":
        assert np.sqrt(((e - ref["energy"]) ** 2).sum() / (ref["energy"] ** 2).sum()) < 2e-2
        assert np.sqrt(((f - ref["forces"]) ** 2).sum() / (ref["forces"] ** 2).sum()) < 2e-2
    else:
        te, tf = (1e-10, 1e-10) if precision == "fp64" else (1e-5, 1e-4)
        assert energy_rel_err(e, ref["energy"]).max() < te
        assert force_rel_err(f, ref["forces"], small.struct_ptr).max() < tf
    with pytest.raises(pnn.PnnError) as ei:                             # the sticky flag of the first batch is still reported
        net.check()
    assert ei.value.status == -2
    net.close()


def test_host_entry_point_returns_device_errors():
    import paper_2604_15380_b200 as pnn
    mc, b = gen.model_cfg(1), gen.make_batch(1)
    w = gen.make_weights(mc, 1)
    net = make_model(mc, w, "fp32", b.n_atoms, 100, b.n_structs)        # far too few edges
    with pytest.raises(pnn.PnnError) as ei:
        net.eval_host(b.Z, b.pos, b.struct_ptr, b.head)
    assert ei.value.status == -2
    net.close()
    net = make_model(mc, w, "fp32", b.n_atoms, b.n_atoms * 64, b.n_structs)
    bad = np.where(np.arange(b.n_atoms) == 5, 99, b.Z).astype(np.int32)
    with pytest.raises(pnn.PnnError) as ei:
        net.eval_host(bad, b.pos, b.struct_ptr, b.head)
    assert ei.value.status == -6
    e, f = net.eval_host(b.Z, b.pos, b.struct_ptr, b.head)             # and the workspace is usable afterwards
    ref = oracle.evaluate(mc, w, b)
    assert energy_rel_err(e.astype(np.float64), ref["energy"]).max() < 1e-5
    net.close()


def test_binding_rejects_wrong_dtypes_and_devices():
    import torch
    mc, b = gen.model_cfg(1), gen.make_batch(1)
    w = gen.make_weights(mc, 1)
    net = make_model(mc, w, "fp32", b.n_atoms, b.n_atoms * 64, b.n_structs)
    t = to_device(b)
    with pytest.raises(TypeError):
        net.eval(t["Z"], t["pos"].float(), t["struct_ptr"], t["head"])          # float32 positions
    with pytest.raises(TypeError):
        net.eval(t["Z"], t["pos"], t["struct_ptr"].long(), t["head"])           # int64 struct_ptr
    with pytest.raises(TypeError):
        net.eval(t["Z"].long(), t["pos"], t["struct_ptr"], t["head"])
    with pytest.raises(TypeError):
        net.eval(t["Z"], t["pos"].cpu(), t["struct_ptr"], t["head"])            # host tensor where a device one is expected
    with pytest.raises(TypeError):
        net.eval_host(b.Z.astype(np.int64), b.pos, b.struct_ptr, b.head)
    net.close()


def test_workspace_flags_are_validated():
    import paper_2604_15380_b200 as pnn
    mc = gen.model_cfg(1)
    w = gen.make_weights(mc, 1)
    cfg = pnn.pnn_config(mc.F, mc.T, mc.K, mc.H, mc.Zmax, mc.cutoff, mc.norm_eps, pnn.PNN_FP32, 0, 0)
    m = pnn.pnn_model_create(cfg, w)
    with pytest.raises(pnn.PnnError) as ei:
        pnn.pnn_workspace_create(m, 16, 64, 1, 4)
    assert ei.value.status == -1
    pnn.pnn_model_destroy(m)
