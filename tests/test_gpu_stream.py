"""-m gpu tests of the streaming driver (pnn_stream_*; BASELINE.json configs[3] "streamed in batches of 16,384")."""
import numpy as np
import pytest

import gen
import oracle
from gpu_common import make_model

pytestmark = pytest.mark.gpu


def _pinned(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).pin_memory()


@pytest.mark.parametrize("precision,forces", [("bf16", False), ("fp32", True)])
def test_streamed_batches_match_single_batches_bit_for_bit(precision, forces):
    """Six ragged batches of the cfg4 stream through a double-buffered pnn_stream: every batch equals pnn_eval_host on the
    same batch bit for bit, and sampled structures match the oracle."""
    import paper_2604_15380_b200 as pnn
    import torch
    mc = gen.model_cfg(4)
    w = gen.make_weights(mc, 4)
    sizes = [700, 512, 1, 333, 700, 64]
    batches, start = [], 0
    for n in sizes:
        batches.append(gen.make_batch(4, start, n))
        start += n
    maxN = max(b.n_atoms for b in batches)
    net = make_model(mc, w, precision, maxN, maxN * 40, max(sizes), forces)
    ref_e, ref_f = [], []
    for b in batches:
        e, f = net.eval_host(b.Z, b.pos, b.struct_ptr, b.head, forces=forces)
        ref_e.append(e.copy())
        ref_f.append(None if f is None else f.copy())
    flags = pnn.PNN_ENERGY | (pnn.PNN_FORCES if forces else 0)
    st = pnn.pnn_stream_create(net.model, maxN, maxN * 40, max(sizes), flags, 2)
    try:
        assert pnn.pnn_stream_bytes(st) > 0
        hin = [(_pinned(b.Z), _pinned(b.pos), _pinned(b.struct_ptr), _pinned(b.head)) for b in batches]
        eo = [torch.empty(b.n_structs, dtype=net.out_dtype).pin_memory() for b in batches]
        fo = [torch.empty((b.n_atoms, 3), dtype=net.out_dtype).pin_memory() if forces else None for b in batches]
        for k, b in enumerate(batches):
            z, p, sp, h = hin[k]
            pnn.pnn_stream_submit(st, b.n_atoms, b.n_structs, z.numpy(), p.numpy(), sp.numpy(), h.numpy(), None, None,
                                  eo[k].numpy(), None if fo[k] is None else fo[k].numpy())
            if k == 2:
                pnn.pnn_stream_wait(st)      # interleaved waits are allowed
        pnn.pnn_stream_drain(st)
        for k, b in enumerate(batches):
            assert np.array_equal(eo[k].numpy(), ref_e[k]), k
            if forces:
                assert np.array_equal(fo[k].numpy(), ref_f[k]), k
        assert pnn.pnn_stream_launch_count(st) > 0
        # oracle on one sampled batch
        k = 3
        ref = oracle.evaluate(mc, w, batches[k], forces=forces)
        e = eo[k].numpy().astype(np.float64)
        rel = np.sqrt(((e - ref["energy"]) ** 2).sum() / (ref["energy"] ** 2).sum())
        assert rel < (2e-2 if precision == "bf16" else 1e-5)
    finally:
        pnn.pnn_stream_destroy(st)
        net.close()


def test_stream_reports_device_errors_of_the_right_batch():
    import paper_2604_15380_b200 as pnn
    mc = gen.model_cfg(4)
    w = gen.make_weights(mc, 4)
    good, bad = gen.make_batch(4, 0, 32), gen.make_batch(4, 32, 32)
    bad_Z = bad.Z.copy()
    bad_Z[3] = 120
    net = make_model(mc, w, "bf16", 4096, 4096 * 40, 64, False)
    st = pnn.pnn_stream_create(net.model, 4096, 4096 * 40, 64, pnn.PNN_ENERGY, 2)
    try:
        e0, e1, e2 = (np.zeros(32, np.float32) for _ in range(3))
        pnn.pnn_stream_submit(st, good.n_atoms, 32, good.Z, good.pos, good.struct_ptr, good.head, None, None, e0)
        pnn.pnn_stream_submit(st, bad.n_atoms, 32, bad_Z, bad.pos, bad.struct_ptr, bad.head, None, None, e1)
        pnn.pnn_stream_wait(st)                                   # batch 0: fine
        with pytest.raises(pnn.PnnError) as ei:
            pnn.pnn_stream_wait(st)                               # batch 1: bad atomic number
        assert ei.value.status == -6
        pnn.pnn_stream_submit(st, good.n_atoms, 32, good.Z, good.pos, good.struct_ptr, good.head, None, None, e2)
        pnn.pnn_stream_drain(st)                                  # the stream goes on working
        assert np.array_equal(e0, e2)
    finally:
        pnn.pnn_stream_destroy(st)
        net.close()
