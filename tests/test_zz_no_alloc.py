"""-m gpu: pnn_build_graph_static, the entry point that allocates nothing (include/pnn.h: the graph builder with its scratch in
a file-scope static device array), against the existing path pnn_build_graph + pnn_graph_copy.  Index work: the tolerance of
the graph tests is bit-exact (rowptr, col, shift element by element).  Several calls in a row on different batches share the
static array, so stale contents of an earlier (larger, periodic) call must not leak into the next one.  The file name sorts
last on purpose: the suite runs with `pytest -x`."""
import numpy as np
import pytest

import gen
from gpu_common import make_model, to_device
from helpers import single

pytestmark = pytest.mark.gpu


def _existing_path(b, rc, all_images=False):
    """rowptr, col, shift (numpy) from pnn_build_graph on a workspace + pnn_graph_copy."""
    import torch
    import paper_2604_15380_b200 as pnn
    mc = gen.ModelCfg(F=32, T=1, K=8, H=int(b.head.max()) + 1, cutoff=rc, pbc_images="all" if all_images else "minimum")
    net = make_model(mc, gen.make_weights(mc, 1), "fp32", max(b.n_atoms, 1), pnn.PNN_STATIC_MAX_EDGES,
                     max(b.n_structs, 1), forces=False)
    try:
        t = to_device(b)
        net.build_graph(t["pos"], t["struct_ptr"], t["cell"], t["pbc"])
        _, _, _, E = pnn.pnn_graph_view(net.ws)
        rowptr = np.zeros(b.n_atoms + 1, np.int32)
        col = np.zeros(E, np.int32)
        shift = np.zeros((E, 3), np.int8)
        pnn.pnn_graph_copy(net.ws, rowptr, col, shift)
        torch.cuda.synchronize()
        return rowptr, col, shift
    finally:
        net.close()


class _Out:
    """Caller-owned output buffers, allocated ONCE and reused by every call (filled with junk before each)."""

    def __init__(self, max_atoms, max_edges):
        import torch
        dev = torch.device("cuda")
        self.rowptr = torch.empty(max_atoms + 1, dtype=torch.int32, device=dev)
        self.col = torch.empty(max_edges, dtype=torch.int32, device=dev)
        self.shift = torch.empty((max_edges, 3), dtype=torch.int8, device=dev)
        self.flags = torch.empty(1, dtype=torch.int32, device=dev)
        self.max_edges = max_edges

    def run(self, b, rc, all_images=False, max_edges=None):
        import torch
        import paper_2604_15380_b200 as pnn
        t = to_device(b)
        self.rowptr.fill_(-7); self.col.fill_(-7); self.shift.fill_(-7); self.flags.fill_(-7)
        pnn.pnn_build_graph_static(b.n_atoms, b.n_structs, t["pos"], t["struct_ptr"], t["cell"], t["pbc"], rc,
                                   pnn.PNN_IMAGES_ALL if all_images else pnn.PNN_IMAGES_MINIMUM,
                                   self.max_edges if max_edges is None else max_edges, self.rowptr, self.col, self.shift,
                                   self.flags, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        rowptr = self.rowptr[:b.n_atoms + 1].cpu().numpy()
        E = int(rowptr[-1])
        return rowptr, self.col[:E].cpu().numpy(), self.shift[:E].cpu().numpy(), int(self.flags.item())


def _same(got, ref):
    rowptr, col, shift, flags = got
    assert flags == 0
    assert np.array_equal(rowptr, ref[0])
    assert np.array_equal(col, ref[1])
    assert np.array_equal(shift, ref[2])
    assert len(col) > 0


def test_static_graph_matches_the_workspace_path_on_calls_in_a_row():
    import paper_2604_15380_b200 as pnn
    out = _Out(pnn.PNN_STATIC_MAX_ATOMS, pnn.PNN_STATIC_MAX_EDGES)
    mol = gen.make_batch(2, 0, 64)                                   # 64 molecules, about 2,600 atoms, 5 A cutoff
    xtal = gen.make_batch(3, 0, 12)                                  # 12 periodic cells of 128 atoms, 6 A, ~94,000 edges
    rng = np.random.default_rng(3)
    narrow = single(rng.integers(1, 9, 16), rng.uniform(0, 4.2, (16, 3)), 0, np.eye(3) * 4.2, [1, 1, 1])
    ref_mol, ref_xtal = _existing_path(mol, 5.0), _existing_path(xtal, 6.0)
    ref_narrow = _existing_path(narrow, 5.0, all_images=True)
    # calls in a row on the SAME static scratch: large periodic, then small, then the first again, then another mode
    _same(out.run(xtal, 6.0), ref_xtal)
    _same(out.run(mol, 5.0), ref_mol)
    _same(out.run(mol, 5.0), ref_mol)
    _same(out.run(xtal, 6.0), ref_xtal)
    _same(out.run(narrow, 5.0, all_images=True), ref_narrow)
    _same(out.run(mol, 5.0), ref_mol)


def test_static_graph_overflow_flag_limits_and_empty_batch():
    import torch
    import paper_2604_15380_b200 as pnn
    out = _Out(4096, 65536)
    mol = gen.make_batch(2, 0, 8)
    ref = _existing_path(mol, 5.0)
    E = len(ref[1])
    rowptr, _, _, flags = out.run(mol, 5.0, max_edges=E - 1)          # one edge short: flagged, rowptr still complete
    assert flags == pnn.PNN_STATIC_EDGE_OVERFLOW and np.array_equal(rowptr, ref[0])
    _same(out.run(mol, 5.0, max_edges=E), ref)                        # exactly enough, and the flag of the last call is gone
    t = to_device(mol)
    args = (t["pos"], t["struct_ptr"], None, None, 5.0, pnn.PNN_IMAGES_MINIMUM)
    for n_atoms, n_structs, max_edges, word in ((pnn.PNN_STATIC_MAX_ATOMS + 1, 8, 100, "n_atoms"),
                                                (100, pnn.PNN_STATIC_MAX_STRUCTS + 1, 100, "n_structs"),
                                                (100, 8, pnn.PNN_STATIC_MAX_EDGES + 1, "max_edges")):
        with pytest.raises(pnn.PnnError) as ei:                      # rejected on the host before anything is launched
            pnn.pnn_build_graph_static(n_atoms, n_structs, *args, max_edges, out.rowptr, out.col, out.shift, out.flags)
        assert ei.value.status == -2 and word in str(ei.value) and "limit" in str(ei.value)
    # an empty batch: rowptr = [0]
    sp = torch.zeros(1, dtype=torch.int32, device="cuda")
    out.rowptr.fill_(-7)
    pnn.pnn_build_graph_static(0, 0, None, sp, None, None, 5.0, pnn.PNN_IMAGES_MINIMUM, 0, out.rowptr, None, None, out.flags)
    torch.cuda.synchronize()
    assert int(out.rowptr[0].item()) == 0 and int(out.flags.item()) == 0
    _same(out.run(mol, 5.0), ref)
