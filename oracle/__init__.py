"""ctypes loader for the CPU oracle (oracle/painn_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product (paper_2604_15380_b200/) never imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "painn_oracle.cpp")
_LIB = os.path.join(_HERE, "_build", "libpainn_oracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """g++ -O2 -fopenmp, no BLAS (BASELINE.md "CPU-baseline plan")."""
    os.makedirs(os.path.dirname(_LIB), exist_ok=True)
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build())
            lib.oracle_weights_count.restype = ctypes.c_int64
            lib.oracle_neighbours.restype = ctypes.c_int64
            lib.oracle_eval.restype = ctypes.c_int64
            lib.oracle_forces_dual.restype = None
            lib.oracle_rbf_cutoff.restype = None
            _lib = lib
    return _lib


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ct))


def _cfg_arrays(mc):
    rbf = {"gaussian": 0, "bessel": 1}[getattr(mc, "rbf", "gaussian")]
    images = {"minimum": 0, "all": 1}[getattr(mc, "pbc_images", "minimum")]
    ic = np.array([mc.F, mc.T, mc.K, mc.H, mc.Zmax, rbf, images, int(getattr(mc, "max_neighbors", 0)),
                   int(getattr(mc, "n_global", 0)), {"atomwise": 0, "pooled": 1}[getattr(mc, "head_type", "atomwise")],
                   int(getattr(mc, "head_d1", 50)), int(getattr(mc, "head_d2", 776))], np.int32)
    dc = np.array([mc.cutoff, mc.norm_eps], np.float64)
    return ic, dc


def num_threads() -> int:
    """Threads the oracle's OpenMP loops use (OMP_NUM_THREADS or all cores in the affinity mask)."""
    v = os.environ.get("OMP_NUM_THREADS")
    if v:
        return int(v.split(",")[0])
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def rbf_cutoff(d: float, K: int, rc: float):
    """(g_k(d) [K], c(d)) exactly as the forward pass evaluates them."""
    lib = _load()
    g = np.zeros(K, np.float64)
    c = np.zeros(1, np.float64)
    lib.oracle_rbf_cutoff(ctypes.c_double(d), ctypes.c_int32(K), ctypes.c_double(rc), _p(g, ctypes.c_double),
                          _p(c, ctypes.c_double))
    return g, float(c[0])


def rbf_cutoff_typed(d: float, K: int, rc: float, rbf: str):
    """(g_k(d) [K], c(d)) for the named radial basis ("gaussian" or "bessel")."""
    lib = _load()
    g = np.zeros(K, np.float64)
    c = np.zeros(1, np.float64)
    lib.oracle_rbf_cutoff_typed(ctypes.c_double(d), ctypes.c_int32(K), ctypes.c_double(rc),
                                ctypes.c_int32({"gaussian": 0, "bessel": 1}[rbf]), _p(g, ctypes.c_double),
                                _p(c, ctypes.c_double))
    return g, float(c[0])


def weights_count(mc) -> int:
    ic, _ = _cfg_arrays(mc)
    return int(_load().oracle_weights_count(_p(ic, ctypes.c_int32)))


def _prep(batch):
    Z = np.ascontiguousarray(batch.Z, np.int32)
    pos = np.ascontiguousarray(batch.pos, np.float64)
    sp = np.ascontiguousarray(batch.struct_ptr, np.int32)
    head = np.ascontiguousarray(batch.head, np.int32)
    cell = None if batch.cell is None else np.ascontiguousarray(batch.cell, np.float64)
    pbc = None if batch.pbc is None else np.ascontiguousarray(batch.pbc, np.uint8)
    return Z, pos, sp, head, cell, pbc


def neighbours(batch, cutoff: float, all_images: bool = False, max_neighbors: int = 0):
    """Brute-force radius graph. Returns dict(rowptr, recv, send, shift, rvec).
    all_images: every periodic image inside the cutoff (self images included) instead of the minimum image only.
    max_neighbors > 0: every receiver keeps its nearest max_neighbors senders only."""
    lib = _load()
    Z, pos, sp, head, cell, pbc = _prep(batch)
    N, S = Z.shape[0], head.shape[0]
    rowptr = np.zeros(N + 1, np.int32)
    lib.oracle_neighbours_capped.restype = ctypes.c_int64
    ai = ctypes.c_int32(1 if all_images else 0)
    mn = ctypes.c_int32(int(max_neighbors))
    E = lib.oracle_neighbours_capped(ctypes.c_int32(N), ctypes.c_int32(S), _p(pos, ctypes.c_double),
                                     _p(sp, ctypes.c_int32), _p(cell, ctypes.c_double), _p(pbc, ctypes.c_uint8),
                                     ctypes.c_double(cutoff), ai, mn, _p(rowptr, ctypes.c_int32), None, None, None, None)
    recv = np.zeros(E, np.int32)
    send = np.zeros(E, np.int32)
    shift = np.zeros((E, 3), np.int8)
    rvec = np.zeros((E, 3), np.float64)
    lib.oracle_neighbours_capped(ctypes.c_int32(N), ctypes.c_int32(S), _p(pos, ctypes.c_double), _p(sp, ctypes.c_int32),
                                 _p(cell, ctypes.c_double), _p(pbc, ctypes.c_uint8), ctypes.c_double(cutoff), ai, mn,
                                 _p(rowptr, ctypes.c_int32), _p(recv, ctypes.c_int32), _p(send, ctypes.c_int32),
                                 _p(shift, ctypes.c_int8), _p(rvec, ctypes.c_double))
    return dict(rowptr=rowptr, recv=recv, send=send, shift=shift, rvec=rvec)


def evaluate(mc, weights, batch, forces: bool = True, features: bool = False, globals_=None):
    """Energy [S], forces [N,3] (or None); with features=True also s [N,F], v [N,3,F], eatom [N].
    globals_ [S, mc.n_global]: the structures' global attributes (charge, spin), or None."""
    lib = _load()
    ic, dc = _cfg_arrays(mc)
    w = np.ascontiguousarray(weights, np.float64)
    assert w.size == weights_count(mc), "weight blob size mismatch"
    Z, pos, sp, head, cell, pbc = _prep(batch)
    N, S = Z.shape[0], head.shape[0]
    assert Z.min(initial=1) >= 1 and Z.max(initial=1) <= mc.Zmax
    assert head.min(initial=0) >= 0 and head.max(initial=0) < mc.H
    energy = np.zeros(S, np.float64)
    frc = np.zeros((N, 3), np.float64) if forces else None
    s_out = np.zeros((N, mc.F), np.float64) if features else None
    v_out = np.zeros((N, 3, mc.F), np.float64) if features else None
    eatom = np.zeros(N, np.float64) if features else None
    gl = None
    if globals_ is not None:
        gl = np.ascontiguousarray(globals_, np.float64)
        assert gl.shape == (S, getattr(mc, "n_global", 0))
    lib.oracle_eval_glob.restype = ctypes.c_int64
    E = lib.oracle_eval_glob(_p(ic, ctypes.c_int32), _p(dc, ctypes.c_double), _p(w, ctypes.c_double), ctypes.c_int32(N),
                             ctypes.c_int32(S), _p(Z, ctypes.c_int32), _p(pos, ctypes.c_double), _p(sp, ctypes.c_int32),
                             _p(cell, ctypes.c_double), _p(pbc, ctypes.c_uint8), _p(head, ctypes.c_int32),
                             _p(gl, ctypes.c_double), _p(energy, ctypes.c_double), _p(frc, ctypes.c_double),
                             _p(s_out, ctypes.c_double), _p(v_out, ctypes.c_double), _p(eatom, ctypes.c_double))
    out = dict(energy=energy, forces=frc, n_edges=int(E))
    if features:
        out.update(s=s_out, v=v_out, eatom=eatom)
    return out


def forces_dual(mc, weights, batch):
    """Forces by forward-mode dual numbers (3N forward evaluations; tiny inputs only)."""
    lib = _load()
    ic, dc = _cfg_arrays(mc)
    w = np.ascontiguousarray(weights, np.float64)
    Z, pos, sp, head, cell, pbc = _prep(batch)
    N, S = Z.shape[0], head.shape[0]
    frc = np.zeros((N, 3), np.float64)
    lib.oracle_forces_dual(_p(ic, ctypes.c_int32), _p(dc, ctypes.c_double), _p(w, ctypes.c_double), ctypes.c_int32(N),
                           ctypes.c_int32(S), _p(Z, ctypes.c_int32), _p(pos, ctypes.c_double), _p(sp, ctypes.c_int32),
                           _p(cell, ctypes.c_double), _p(pbc, ctypes.c_uint8), _p(head, ctypes.c_int32),
                           _p(frc, ctypes.c_double))
    return frc


def evaluate_blended(mc, weights, batch, head_weights, forces: bool = True, skip_below: float = 0.0):
    """Blended multi-head evaluation of the paper's inference pipeline (Fig. 5 at :420): every
    structure g gets E_g = sum_h w[g,h] E_g^(h), F = -dE/dx, where E^(h) is the energy with head h applied to the shared
    trunk and w [S,H] are the per-structure branch weights (in the paper a softmax over a composition MLP; here an input).
    Heads with w[g,h] < skip_below are dropped for that structure ("branch skipping").

    Written as its definition: H single-head evaluations of the oracle above, combined linearly.  Slow on purpose."""
    import dataclasses
    hw = np.asarray(head_weights, np.float64)
    S = batch.head.shape[0]
    assert hw.shape == (S, mc.H)
    hw = np.where(hw < skip_below, 0.0, hw)
    energy = np.zeros(S, np.float64)
    frc = np.zeros((batch.Z.shape[0], 3), np.float64) if forces else None
    sof = np.repeat(np.arange(S), np.diff(batch.struct_ptr))
    n_edges = 0
    for h in range(mc.H):
        if not np.any(hw[:, h] != 0.0):
            continue
        bh = dataclasses.replace(batch, head=np.full(S, h, np.int32))
        out = evaluate(mc, weights, bh, forces=forces)
        n_edges = out["n_edges"]
        energy += hw[:, h] * out["energy"]
        if forces:
            frc += hw[sof, h][:, None] * out["forces"]
    return dict(energy=energy, forces=frc, n_edges=n_edges)


def branch_weights(Z, struct_ptr, widths, params):
    """Composition-conditioned branch weights ("the MLP maps the structure's chemical-composition vector
    to softmax weights that blend these branch outputs"; "24,500 parameters ... maps per-element
    chemical-composition vectors to per-branch blending weights ... softmax-normalized").

    The paper gives neither the layer widths nor the activation nor the normalisation of the composition vector; DESIGN.md
    reading Q28 fixes them: c_z = (number of atoms of the structure with atomic number z) / (number of atoms), z = 1 ...
    widths[0] (an empty structure has c = 0); hidden layers x <- SiLU(W x + b) (the backbone's activation);
    last layer linear; w = softmax over the widths[-1] heads.  `params` = per layer W [out, in] row-major then b [out],
    FP64.  Returns [S, H] FP64.  Plain loops over structures and layers; written from the definition."""
    Z = np.asarray(Z, np.int64)
    sp = np.asarray(struct_ptr, np.int64)
    widths = [int(x) for x in widths]
    params = np.asarray(params, np.float64)
    S = sp.shape[0] - 1
    layers, off = [], 0
    for l in range(len(widths) - 1):
        n_in, n_out = widths[l], widths[l + 1]
        W = params[off:off + n_out * n_in].reshape(n_out, n_in)
        off += n_out * n_in
        b = params[off:off + n_out]
        off += n_out
        layers.append((W, b))
    assert off == params.shape[0]
    out = np.zeros((S, widths[-1]), np.float64)
    for g in range(S):
        zs = Z[sp[g]:sp[g + 1]]
        assert zs.size == 0 or (zs.min() >= 1 and zs.max() <= widths[0])
        c = np.zeros(widths[0], np.float64)
        for z in zs:
            c[z - 1] += 1.0
        if zs.size:
            c /= zs.size
        x = c
        for l, (W, b) in enumerate(layers):
            x = W @ x + b
            if l + 1 < len(layers):
                x = x / (1.0 + np.exp(-x))
        e = np.exp(x - x.max())
        out[g] = e / e.sum()
    return out
