"""Oracle of the training step (Table V: "Optimizer AdamW, lr = 6.34e-4", "Loss MAE",
"Force weight ~ 94.8", "Batch size 25 per GPU", "Precision FP64"; the backward pass dominates the training step).
TEST INFRASTRUCTURE ONLY (imported by tests/ alone); plain PyTorch CPU ops in FP64, one statement per equation, no blocking
or fusion; shares no code with the CUDA path.  NO CUDA KERNEL OF THIS STEP EXISTS YET: this file and its pins
(tests/test_oracle_train.py) are the oracle-first half of that row, committed before any kernel, as the process demands.

What one step computes (readings Q32 of DESIGN.md where the paper is silent):

  E_s, F_ia            the PaiNN energies and forces of SURVEY.md 8(c) B1-B5 / R1-R4 (restated below in torch; pinned against
                       the C++ oracle, which is written from the same passages with plain loops)
  L = (1/S) sum_s |E_s - E*_s|  +  lambda (1/3N) sum_ia |F_ia - F*_ia|      MAE of both, force weight lambda (Table V);
                       means over the batch's structures and force components (Q32a), total energies (Q32b)
  g = dL/dtheta        by reverse-mode differentiation of the statements below, a library routine: the force term needs the
                       derivative of F = -dE/dx with respect to theta (second order), which the same routine provides
                       (create_graph); sign(0) = 0 where a residual vanishes (Q32c)
  AdamW (decoupled weight decay), written out:                                                  (Q32d: beta, eps, decay)
      t <- t + 1
      theta <- theta (1 - lr wd)
      m <- beta1 m + (1 - beta1) g ;   v <- beta2 v + (1 - beta2) g o g
      theta <- theta - lr (m / (1 - beta1^t)) / (sqrt(v / (1 - beta2^t)) + eps)

Edges come from oracle.neighbours (the brute-force graph, pinned in tests/test_oracle_neighbours.py); they do not depend on
theta, and the positions are fixed during a step, so the edge set is a constant of the differentiation."""
import math
from dataclasses import dataclass, field

import numpy as np
import torch

import gen
from . import neighbours

LR = 6.34e-4           # PAPER.md:234 (Table V)
FORCE_WEIGHT = 94.8    # PAPER.md:238 (Table V, "~ 94.8")
BETAS = (0.9, 0.999)   # Q32d: the paper names AdamW and a learning rate only; these are the optimiser's published defaults
EPS = 1e-8
WEIGHT_DECAY = 0.01


def _views(mc, theta):
    """Named views into the flat parameter vector (SURVEY.md 8(b) blob layout; gen.weights_layout holds no arithmetic)."""
    return {name: theta[off:off + int(np.prod(shape))].reshape(shape) for name, shape, _, off in gen.weights_layout(mc)}


def _edges(mc, batch):
    nb = neighbours(batch, mc.cutoff, all_images=getattr(mc, "pbc_images", "minimum") == "all",
                    max_neighbors=getattr(mc, "max_neighbors", 0))
    recv = torch.from_numpy(nb["recv"].astype(np.int64))
    send = torch.from_numpy(nb["send"].astype(np.int64))
    a2s = torch.from_numpy(np.repeat(np.arange(batch.n_structs), np.diff(batch.struct_ptr)).astype(np.int64))
    if batch.cell is not None and len(recv):
        cell = torch.from_numpy(np.ascontiguousarray(batch.cell, np.float64))
        off = torch.einsum("ea,eab->eb", torch.from_numpy(nb["shift"].astype(np.float64)), cell[a2s[recv]])
    else:
        off = torch.zeros((len(recv), 3), dtype=torch.float64)
    return recv, send, off, a2s


def energy(mc, theta, batch, pos, edges):
    """E_s [S] as a differentiable function of theta (flat FP64 tensor) and pos [N,3].  SURVEY.md 8(c) B1-B5."""
    assert getattr(mc, "backbone", "painn") == "painn" and getattr(mc, "head_type", "atomwise") == "atomwise"
    assert getattr(mc, "rbf", "gaussian") == "gaussian" and getattr(mc, "n_global", 0) == 0
    W = _views(mc, theta)
    recv, send, off, a2s = edges
    F, K, rc = mc.F, mc.K, mc.cutoff
    silu = torch.nn.functional.silu
    # B1/B2: geometry, Gaussian basis, cosine cutoff (Q2, Q3, Q4: sender minus receiver)
    r = pos[send] - pos[recv] + off
    d = torch.sqrt((r * r).sum(1))
    u = r / d[:, None]
    dmu = rc / (K - 1) if K > 1 else rc
    g = torch.exp(-(d[:, None] - torch.arange(K, dtype=torch.float64)[None, :] * dmu) ** 2 / (2.0 * dmu * dmu))
    c = 0.5 * (torch.cos(math.pi * d / rc) + 1.0)
    s = W["emb"][torch.from_numpy(batch.Z.astype(np.int64))]
    v = torch.zeros(batch.n_atoms, 3, F, dtype=torch.float64)
    for t in range(mc.T):
        p = f"b{t}."
        # B3: message
        phi = silu(s @ W[p + "msg_W1"].T + W[p + "msg_b1"]) @ W[p + "msg_W2"].T + W[p + "msg_b2"]
        w = (g @ W[p + "flt_W"].T + W[p + "flt_b"]) * c[:, None]
        x = phi[send] * w
        s1 = s + torch.zeros_like(s).index_add(0, recv, x[:, :F])
        v1 = v + torch.zeros_like(v).index_add(0, recv, x[:, F:2 * F, None].transpose(1, 2) * u[:, :, None]
                                               + x[:, 2 * F:, None].transpose(1, 2) * v[send])
        # B4: update
        P = v1 @ W[p + "upd_U"].T
        Q = v1 @ W[p + "upd_V"].T
        n = torch.sqrt((Q * Q).sum(1) + mc.norm_eps)
        a = silu(torch.cat([s1, n], 1) @ W[p + "upd_A1"].T + W[p + "upd_c1"]) @ W[p + "upd_A2"].T + W[p + "upd_c2"]
        s = s1 + a[:, F:2 * F] * (P * Q).sum(1) + a[:, 2 * F:]
        v = v1 + a[:, None, :F] * P
    # B5: the structure's head, atom-wise, summed per structure
    ha = torch.from_numpy(batch.head.astype(np.int64))[a2s]
    W1 = torch.stack([W[f"h{h}.out_W1"] for h in range(mc.H)])[ha]
    b1 = torch.stack([W[f"h{h}.out_b1"] for h in range(mc.H)])[ha]
    w2 = torch.stack([W[f"h{h}.out_w2"] for h in range(mc.H)])[ha]
    b2 = torch.stack([W[f"h{h}.out_b2"] for h in range(mc.H)])[ha][:, 0]
    e = (w2 * silu(torch.einsum("nof,nf->no", W1, s) + b1)).sum(1) + b2
    return torch.zeros(batch.n_structs, dtype=torch.float64).index_add(0, a2s, e)


def energy_forces(mc, weights, batch):
    """(E [S], F [N,3]) as numpy FP64: the torch restatement alone, for the pin against the C++ oracle."""
    theta = torch.from_numpy(np.ascontiguousarray(weights, np.float64))
    pos = torch.from_numpy(np.ascontiguousarray(batch.pos, np.float64)).clone().requires_grad_(True)
    E = energy(mc, theta, batch, pos, _edges(mc, batch))
    (gx,) = torch.autograd.grad(E.sum(), pos)
    return E.detach().numpy(), -gx.numpy()


def loss_and_gradient(mc, weights, batch, E_ref, F_ref, force_weight=FORCE_WEIGHT):
    """L (float), dL/dtheta [P] (numpy FP64), and the two MAE terms.  F = -dE/dx is kept differentiable in theta
    (create_graph), so that the gradient of the force term is the exact second-order expression, not an approximation."""
    theta = torch.from_numpy(np.ascontiguousarray(weights, np.float64)).clone().requires_grad_(True)
    pos = torch.from_numpy(np.ascontiguousarray(batch.pos, np.float64)).clone().requires_grad_(True)
    E = energy(mc, theta, batch, pos, _edges(mc, batch))
    (gx,) = torch.autograd.grad(E.sum(), pos, create_graph=True)
    F = -gx
    mae_e = (E - torch.from_numpy(np.asarray(E_ref, np.float64))).abs().mean()                     # Q32a, Q32b
    mae_f = (F - torch.from_numpy(np.asarray(F_ref, np.float64))).abs().mean()
    L = mae_e + force_weight * mae_f
    (g,) = torch.autograd.grad(L, theta)
    return float(L.detach()), g.numpy().copy(), float(mae_e.detach()), float(mae_f.detach())


@dataclass
class AdamWState:
    """Optimiser state carried between steps: step count and the two moment vectors (zero before the first step)."""
    t: int = 0
    m: np.ndarray = field(default=None)
    v: np.ndarray = field(default=None)


def adamw_update(theta, g, state, lr=LR, betas=BETAS, eps=EPS, weight_decay=WEIGHT_DECAY):
    """One AdamW update of the flat vector theta with gradient g, the formulas of the header in their order, element by
    element (numpy FP64).  Returns (theta', state')."""
    theta = np.asarray(theta, np.float64)
    g = np.asarray(g, np.float64)
    m = np.zeros_like(theta) if state.m is None else state.m
    v = np.zeros_like(theta) if state.v is None else state.v
    t = state.t + 1
    theta = theta * (1.0 - lr * weight_decay)
    m = betas[0] * m + (1.0 - betas[0]) * g
    v = betas[1] * v + (1.0 - betas[1]) * g * g
    m_hat = m / (1.0 - betas[0] ** t)
    v_hat = v / (1.0 - betas[1] ** t)
    theta = theta - lr * m_hat / (np.sqrt(v_hat) + eps)
    return theta, AdamWState(t=t, m=m, v=v)


def train_step(mc, weights, batch, E_ref, F_ref, state=None, lr=LR, betas=BETAS, eps=EPS, weight_decay=WEIGHT_DECAY,
               force_weight=FORCE_WEIGHT):
    """One training step on one batch: loss, gradient, AdamW.  Returns dict(weights, state, loss, mae_e, mae_f, grad)."""
    state = state or AdamWState()
    L, g, mae_e, mae_f = loss_and_gradient(mc, weights, batch, E_ref, F_ref, force_weight)
    new_w, new_state = adamw_update(weights, g, state, lr, betas, eps, weight_decay)
    return dict(weights=new_w, state=new_state, loss=L, mae_e=mae_e, mae_f=mae_f, grad=g)
