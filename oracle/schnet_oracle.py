"""Oracle of the second backbone: SchNet continuous-filter convolutions on the SAME radius graph and
radial basis as the PaiNN path.  TEST INFRASTRUCTURE ONLY (imported by tests/ alone); plain PyTorch CPU ops in FP64, one
statement per equation, no blocking or fusion; shares no code with the CUDA path.

PAPER.md names the backbone and cites it ([46] at PAPER.md:147, 212: "EGNN and SchNet are the lightest backbones") but prints
no equation; the definition followed here is the published SchNet interaction block, with the readings of DESIGN.md Q31:

  x_i^0 = emb[Z_i]
  per block t:   g_e   = radial basis of d_e (K Gaussians or Bessel functions, the PaiNN path's, reading Q2)
                 W_e   = (F2 silu(F1 g_e + f1) + f2) * c(d_e)          filter-generating network times the cosine cutoff (Q3)
                 m_i   = sum_{e = (i <- j)} (A x_j) o W_e              continuous-filter convolution, A without bias
                 x_i  += B2 silu(B1 m_i + b1) + b2
  e_i = w2_h . silu(W1_h x_i + b1_h) + b2_h ,  E_g = sum_{i in g} e_i   (the atom-wise multi-head readout of the PaiNN path)
  forces = -dE/dx (the definition; evaluated by reverse-mode differentiation of the statements above, a library routine).

Activation: SiLU where SchNet has the shifted softplus (reading Q31: the one activation of this build, Q6).
Edges come from oracle.neighbours (the brute-force graph, pinned in tests/test_oracle_neighbours.py)."""
import math

import numpy as np
import torch

import gen
from . import neighbours


def _unpack(mc, w):
    t = torch.from_numpy(np.ascontiguousarray(w, np.float64))
    return {name: t[off:off + int(np.prod(shape))].reshape(shape) for name, shape, _, off in gen.weights_layout(mc)}


def _rbf(mc, d):
    K, rc = mc.K, mc.cutoff
    if getattr(mc, "rbf", "gaussian") == "bessel":
        n = torch.arange(1, K + 1, dtype=torch.float64)
        return math.sqrt(2.0 / rc) * torch.sin(n[None, :] * math.pi * d[:, None] / rc) / d[:, None]
    dmu = rc / (K - 1) if K > 1 else rc
    mu = torch.arange(K, dtype=torch.float64) * dmu
    return torch.exp(-(d[:, None] - mu[None, :]) ** 2 / (2.0 * dmu * dmu))


def evaluate_schnet(mc, weights, batch, forces: bool = True, features: bool = False):
    assert getattr(mc, "backbone", "painn") == "schnet"
    W = _unpack(mc, weights)
    assert batch.head.min(initial=0) >= 0 and batch.head.max(initial=0) < mc.H
    nb = neighbours(batch, mc.cutoff, all_images=getattr(mc, "pbc_images", "minimum") == "all")
    recv = torch.from_numpy(nb["recv"].astype(np.int64))
    send = torch.from_numpy(nb["send"].astype(np.int64))
    pos = torch.from_numpy(np.ascontiguousarray(batch.pos, np.float64)).clone().requires_grad_(forces)
    N, S = batch.n_atoms, batch.n_structs
    a2s = torch.from_numpy(np.repeat(np.arange(S), np.diff(batch.struct_ptr)).astype(np.int64))
    if batch.cell is not None and len(recv):
        cell = torch.from_numpy(np.ascontiguousarray(batch.cell, np.float64))
        off = torch.einsum("ea,eab->eb", torch.from_numpy(nb["shift"].astype(np.float64)), cell[a2s[recv]])
    else:
        off = torch.zeros((len(recv), 3), dtype=torch.float64)
    r = pos[send] - pos[recv] + off                                   # Q4: sender minus receiver
    d = torch.sqrt((r * r).sum(1))
    g = _rbf(mc, d)
    c = 0.5 * (torch.cos(math.pi * d / mc.cutoff) + 1.0)
    silu = torch.nn.functional.silu
    x = W["emb"][torch.from_numpy(batch.Z.astype(np.int64))]
    for t in range(mc.T):
        p = f"b{t}."
        Wf = (silu(g @ W[p + "flt_W1"].T + W[p + "flt_b1"]) @ W[p + "flt_W2"].T + W[p + "flt_b2"]) * c[:, None]
        x1 = x @ W[p + "in_W"].T
        m = torch.zeros_like(x).index_add(0, recv, x1[send] * Wf)
        x = x + silu(m @ W[p + "out_W1"].T + W[p + "out_b1"]) @ W[p + "out_W2"].T + W[p + "out_b2"]
    head = torch.from_numpy(batch.head.astype(np.int64))[a2s]
    W1 = torch.stack([W[f"h{h}.out_W1"] for h in range(mc.H)])[head]   # [N, F/2, F]
    b1 = torch.stack([W[f"h{h}.out_b1"] for h in range(mc.H)])[head]
    w2 = torch.stack([W[f"h{h}.out_w2"] for h in range(mc.H)])[head]
    b2 = torch.stack([W[f"h{h}.out_b2"] for h in range(mc.H)])[head][:, 0]
    eatom = (w2 * silu(torch.einsum("nof,nf->no", W1, x) + b1)).sum(1) + b2
    energy = torch.zeros(S, dtype=torch.float64).index_add(0, a2s, eatom)
    out = dict(energy=energy.detach().numpy(), forces=None, n_edges=int(len(recv)))
    if forces:
        (grad,) = torch.autograd.grad(energy.sum(), pos)
        out["forces"] = -grad.numpy()
    if features:
        out["x"] = x.detach().numpy()
        out["eatom"] = eatom.detach().numpy()
    return out
