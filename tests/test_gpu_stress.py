"""-m gpu: repeated evaluations of the mbarrier-pipelined BF16 kernels (edge_tc.cu, edge_tc_bwd.cu, gemm_tc.cu).  A
producer / epilogue hand-shake that can skip a barrier phase shows up as a rare hang (round 2: the reverse edge kernel's two
producers shared one tmem_empty barrier and hung about once in 25 batches), so every evaluation here is awaited by polling
the stream with a deadline rather than by a blocking synchronize."""
import time

import numpy as np
import pytest

import gen
from gpu_common import make_model

pytestmark = pytest.mark.gpu


def _await(torch, what, deadline=20.0):
    t0 = time.time()
    while not torch.cuda.current_stream().query():
        if time.time() - t0 > deadline:
            pytest.fail(f"kernel hang: {what}", pytrace=False)
        time.sleep(0.001)


@pytest.mark.parametrize("cfg_id,n_structs,iters", [(2, 21, 160), (1, 7, 80), (3, 3, 40)])
def test_bf16_evaluations_do_not_hang(cfg_id, n_structs, iters):
    import torch
    mc = gen.model_cfg(cfg_id)
    w = gen.make_weights(mc, cfg_id)
    net = None
    first = None
    for it in range(iters):
        b = gen.make_batch(cfg_id, it % 5, n_structs) if cfg_id != 3 else gen.make_batch(3, it % 3, n_structs, n_atoms=54)
        if it % 8 == 0:   # a new model + workspace now and then, as the parity tests do
            if net is not None:
                net.close()
            net = make_model(mc, w, "bf16", b.n_atoms + 64, (b.n_atoms + 64) * 96, n_structs, True)
        dev = torch.device("cuda")
        Z = torch.from_numpy(b.Z.astype(np.int32)).to(dev); pos = torch.from_numpy(b.pos).to(dev)
        sp = torch.from_numpy(b.struct_ptr.astype(np.int32)).to(dev); hd = torch.from_numpy(b.head.astype(np.int32)).to(dev)
        cell = torch.from_numpy(b.cell).to(dev) if b.cell is not None else None
        pbc = torch.from_numpy(b.pbc.astype(np.uint8)).to(dev) if b.cell is not None else None
        for forces in (True, False):
            e, f = net.eval(Z, pos, sp, hd, cell=cell, pbc=pbc, forces=forces)
            _await(torch, f"cfg{cfg_id} iteration {it} forces={forces}")
        if it % 15 == 0:   # same batch -> bit-identical energies (no race in the data path either)
            e = e.cpu().numpy()
            if first is None:
                first = e
            else:
                assert np.array_equal(e, first)
    net.close()
