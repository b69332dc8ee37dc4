"""Helpers for the -m gpu parity tests: run a gen.Batch through the C-ABI library on cuda:0."""
from __future__ import annotations

import numpy as np

import gen


def to_device(batch: gen.Batch):
    import torch
    dev = torch.device("cuda:0")
    t = dict(Z=torch.from_numpy(np.ascontiguousarray(batch.Z, np.int32)).to(dev),
             pos=torch.from_numpy(np.ascontiguousarray(batch.pos, np.float64)).to(dev),
             struct_ptr=torch.from_numpy(np.ascontiguousarray(batch.struct_ptr, np.int32)).to(dev),
             head=torch.from_numpy(np.ascontiguousarray(batch.head, np.int32)).to(dev),
             cell=None, pbc=None)
    if batch.cell is not None:
        t["cell"] = torch.from_numpy(np.ascontiguousarray(batch.cell, np.float64)).to(dev)
        t["pbc"] = torch.from_numpy(np.ascontiguousarray(batch.pbc, np.uint8)).to(dev)
    return t


def make_model(mc: gen.ModelCfg, weights, precision: str, max_atoms: int, max_edges: int, max_structs: int,
               forces: bool = True):
    import paper_2604_15380_b200 as pnn
    return pnn.PaiNN(mc.F, mc.T, mc.K, mc.H, weights, precision=precision, cutoff=mc.cutoff, Zmax=mc.Zmax,
                     norm_eps=mc.norm_eps, max_atoms=max_atoms, max_edges=max_edges, max_structs=max_structs,
                     forces=forces, rbf=getattr(mc, "rbf", "gaussian"),
                     pbc_images=getattr(mc, "pbc_images", "minimum"), max_neighbors=getattr(mc, "max_neighbors", 0),
                     n_global=getattr(mc, "n_global", 0), head_type=getattr(mc, "head_type", "atomwise"),
                     head_d1=getattr(mc, "head_d1", 50), head_d2=getattr(mc, "head_d2", 776),
                     backbone=getattr(mc, "backbone", "painn"))


def run_gpu(mc: gen.ModelCfg, weights, batch: gen.Batch, precision: str, forces: bool = True, max_edges=None,
            want_graph: bool = False, globals_=None):
    """Returns dict(energy, forces, [rowptr, col, shift]) as numpy arrays."""
    import torch
    if max_edges is None:
        max_edges = max(64, batch.n_atoms * 96)
    net = make_model(mc, weights, precision, max(batch.n_atoms, 1), max_edges, max(batch.n_structs, 1), forces)
    try:
        t = to_device(batch)
        gl = None if globals_ is None else torch.from_numpy(np.ascontiguousarray(globals_, np.float64)).cuda()
        e, f = net.eval(t["Z"], t["pos"], t["struct_ptr"], t["head"], t["cell"], t["pbc"], forces=forces, globals_=gl)
        torch.cuda.synchronize()
        net.check()
        out = dict(energy=e.cpu().numpy().astype(np.float64),
                   forces=None if f is None else f.cpu().numpy().astype(np.float64), launches=net.launches)
        if want_graph:
            out["rowptr"], out["col"], out["shift"] = net.graph()
        return out
    finally:
        net.close()


def gpu_edge_set(rowptr, col, shift) -> set:
    recv = np.repeat(np.arange(len(rowptr) - 1), np.diff(rowptr))
    return set(zip(recv.tolist(), col.tolist(), shift[:, 0].tolist(), shift[:, 1].tolist(), shift[:, 2].tolist()))
