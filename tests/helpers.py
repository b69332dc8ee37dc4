"""Test-only helpers: an independent numpy neighbour enumeration, a torch FP64 third opinion of
the PaiNN equations (SURVEY.md §8(c) pin (ix)), rotations, and the error norms of reading Q20.
None of this is used by the product or by the oracle."""
from __future__ import annotations

import dataclasses
import itertools

import numpy as np

import gen


# ----------------------------------------------------------------------------- geometry helpers
def random_rotation(rng, improper=False):
    q, r = np.linalg.qr(rng.normal(size=(3, 3)))
    q = q * np.sign(np.diag(r))
    if (np.linalg.det(q) < 0) != improper:
        q[:, 0] = -q[:, 0]
    return q


def single(Z, pos, head=0, cell=None, pbc=None) -> gen.Batch:
    Z = np.asarray(Z, np.int32)
    pos = np.asarray(pos, np.float64).reshape(-1, 3)
    return gen.Batch(Z, pos, np.array([0, len(Z)], np.int32), np.array([head], np.int32),
                     None if cell is None else np.asarray(cell, np.float64).reshape(1, 3, 3),
                     None if pbc is None else np.asarray(pbc, np.uint8).reshape(1, 3))


def with_pos(b: gen.Batch, pos) -> gen.Batch:
    return dataclasses.replace(b, pos=np.ascontiguousarray(pos, np.float64))


def edges_by_image_enumeration(batch: gen.Batch, rc: float, nimg: int = 2):
    """All (i, j, shift) with i != j or shift != 0, |x_j - x_i + shift.C| < rc, enumerating
    integer shifts in [-nimg, nimg]^3 on periodic axes.  When every cell width >= 2 rc this is
    the same set as the minimum-image rule, with no self-image edges."""
    out = set()
    sp = batch.struct_ptr
    for g in range(batch.n_structs):
        idx = range(sp[g], sp[g + 1])
        if batch.cell is not None and batch.pbc[g].any():
            C = batch.cell[g]
            rng_ = [range(-nimg, nimg + 1) if batch.pbc[g][a] else range(0, 1) for a in range(3)]
        else:
            C = np.eye(3)
            rng_ = [range(0, 1)] * 3
        for sh in itertools.product(*rng_):
            sc = np.asarray(sh, np.float64) @ C
            for i in idx:
                d = batch.pos[sp[g]:sp[g + 1]] - batch.pos[i] + sc
                d2 = (d * d).sum(1)
                for jj in np.nonzero(d2 < rc * rc)[0]:
                    j = sp[g] + jj
                    if j == i and not any(sh):
                        continue
                    out.add((int(i), int(j), int(sh[0]), int(sh[1]), int(sh[2])))
    return out


def edge_set(nb) -> set:
    return set(zip(nb["recv"].tolist(), nb["send"].tolist(), nb["shift"][:, 0].tolist(), nb["shift"][:, 1].tolist(),
                   nb["shift"][:, 2].tolist()))


# ----------------------------------------------------------------------------- error norms (Q20)
def energy_rel_err(E, Eref):
    E, Eref = np.asarray(E, np.float64), np.asarray(Eref, np.float64)
    rms = np.sqrt(np.mean(Eref ** 2)) if Eref.size else 1.0
    return np.abs(E - Eref) / np.maximum(np.abs(Eref), rms)


def force_rel_err(Fc, Fref, struct_ptr):
    """Per structure: max-abs component error / max(RMS force component of the structure, RMS over config)."""
    Fc, Fref = np.asarray(Fc, np.float64), np.asarray(Fref, np.float64)
    rms_all = np.sqrt(np.mean(Fref ** 2))
    out = np.zeros(len(struct_ptr) - 1)
    for g in range(len(struct_ptr) - 1):
        a, b = struct_ptr[g], struct_ptr[g + 1]
        if b == a:
            continue
        rms_g = np.sqrt(np.mean(Fref[a:b] ** 2))
        out[g] = np.abs(Fc[a:b] - Fref[a:b]).max() / max(rms_g, rms_all)
    return out


# ----------------------------------------------------------------------------- torch third opinion
def torch_painn(mc: gen.ModelCfg, blob, batch: gen.Batch, edges, want_forces=True, dtype=None):
    """Vectorised torch restatement with autograd forces (FP64; `dtype=torch.float32` gives the plain library
    FP32 evaluation used as the FP32 rounding floor).  `edges` = (recv, send, shift[E,3]) from an enumeration
    that does not come from the oracle."""
    import torch
    torch.set_num_threads(max(1, torch.get_num_threads()))
    DT = dtype or torch.float64
    W = {k: torch.tensor(v).to(DT) for k, v in gen.synth.unpack_weights(mc, np.asarray(blob, np.float64)).items()}
    F, K, rc = mc.F, mc.K, mc.cutoff
    recv = torch.tensor(np.asarray(edges[0], np.int64))
    send = torch.tensor(np.asarray(edges[1], np.int64))
    shift = np.asarray(edges[2], np.float64).reshape(-1, 3)
    sof = np.repeat(np.arange(batch.n_structs), np.diff(batch.struct_ptr))
    if batch.cell is not None:
        sc = np.einsum("ea,eab->eb", shift, batch.cell[sof[np.asarray(edges[0], np.int64)]])
    else:
        sc = np.zeros_like(shift)
    pos = torch.tensor(batch.pos).to(DT).requires_grad_(True)
    r = pos[send] - pos[recv] + torch.tensor(sc).to(DT)
    d = r.norm(dim=1)
    u = r / d[:, None]
    mu = torch.arange(K, dtype=DT) * (rc / (K - 1) if K > 1 else rc)
    dmu = rc / (K - 1) if K > 1 else rc
    g = torch.exp(-(d[:, None] - mu[None, :]) ** 2 / (2 * dmu * dmu))
    c = 0.5 * (torch.cos(np.pi * d / rc) + 1.0)
    silu = torch.nn.functional.silu
    N = batch.n_atoms
    s = W["emb"][torch.tensor(batch.Z.astype(np.int64))]
    v = torch.zeros(N, 3, F, dtype=DT)
    for t in range(mc.T):
        p = f"b{t}."
        phi = silu(s @ W[p + "msg_W1"].T + W[p + "msg_b1"]) @ W[p + "msg_W2"].T + W[p + "msg_b2"]
        w = (g @ W[p + "flt_W"].T + W[p + "flt_b"]) * c[:, None]
        x = phi[send] * w
        xss, xvs, xvv = x[:, :F], x[:, F:2 * F], x[:, 2 * F:]
        s1 = s + torch.zeros_like(s).index_add(0, recv, xss)
        dv = xvs[:, None, :] * u[:, :, None] + xvv[:, None, :] * v[send]
        v1 = v + torch.zeros_like(v).index_add(0, recv, dv)
        P = v1 @ W[p + "upd_U"].T
        Q = v1 @ W[p + "upd_V"].T
        n = torch.sqrt((Q * Q).sum(1) + mc.norm_eps)
        k = silu(torch.cat([s1, n], 1) @ W[p + "upd_A1"].T + W[p + "upd_c1"])
        a = k @ W[p + "upd_A2"].T + W[p + "upd_c2"]
        avv, asv, ass = a[:, :F], a[:, F:2 * F], a[:, 2 * F:]
        s = s1 + asv * (P * Q).sum(1) + ass
        v = v1 + avv[:, None, :] * P
    ha = torch.tensor(batch.head.astype(np.int64))[torch.tensor(sof)]
    W1 = torch.stack([W[f"h{h}.out_W1"] for h in range(mc.H)])[ha]
    b1 = torch.stack([W[f"h{h}.out_b1"] for h in range(mc.H)])[ha]
    w2 = torch.stack([W[f"h{h}.out_w2"] for h in range(mc.H)])[ha]
    b2 = torch.stack([W[f"h{h}.out_b2"] for h in range(mc.H)])[ha][:, 0]
    e = (w2 * silu(torch.einsum("nof,nf->no", W1, s) + b1)).sum(1) + b2
    E = torch.zeros(batch.n_structs, dtype=DT).index_add(0, torch.tensor(sof), e)
    out = dict(energy=E.detach().double().numpy(), s=s.detach().double().numpy(), v=v.detach().double().numpy())
    if want_forces:
        (gx,) = torch.autograd.grad(E.sum(), pos)
        out["forces"] = -gx.double().numpy()
    return out
