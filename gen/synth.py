"""Counter-based seeded generators for the five BASELINE.json configs.

Every random number is a pure function of (seed, config id, structure id, purpose tag,
index...), obtained by chaining the splitmix64 finaliser over the identifiers.  Any
subset of any config can therefore be regenerated on its own (needed for the sampled
oracle parity on the 1,048,576-structure screening config).

Nothing here belongs to the method (PaiNN): only shapes, sizes, densities and value
distributions taken from BASELINE.json `configs` / SURVEY.md §8(d).  The one geometric
computation is the *rejection margin*: a structure is re-drawn if any pair distance lies
within 1e-9 Å of the cutoff (or, under PBC, within 1e-9 of the half-cell tie), so that the
edge set is unique and both implementations must agree on it bit-for-bit
(BASELINE.json `north_star`: "generators reject pairs within 1e-9 Å of the cutoff").
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Sequence

import numpy as np

BASE_SEED = 2604015380

_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_GOLD = np.uint64(0x9E3779B97F4A7C15)

# purpose tags (arbitrary distinct constants)
_T_NATOMS, _T_HEAD, _T_POS, _T_Z, _T_SHUF, _T_JIT, _T_W, _T_HW, _T_BW = 11, 12, 13, 14, 15, 16, 17, 18, 19

MARGIN = 1e-9


def _mix(x: np.ndarray) -> np.ndarray:
    x = np.asarray(x, dtype=np.uint64).copy()
    with np.errstate(over="ignore"):
        x ^= x >> np.uint64(30)
        x *= _M1
        x ^= x >> np.uint64(27)
        x *= _M2
        x ^= x >> np.uint64(31)
    return x


def _hash(*ids) -> np.ndarray:
    """uint64 hash of a tuple of (broadcastable) non-negative integer identifiers."""
    h = np.uint64(0x243F6A8885A308D3)
    with np.errstate(over="ignore"):
        for i in ids:
            h = _mix((h + _GOLD) ^ _mix(np.asarray(i, dtype=np.uint64) + _GOLD))
    return h


def _uniform(*ids) -> np.ndarray:
    """float64 in [0, 1)."""
    return (_hash(*ids) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def _normal(*ids) -> np.ndarray:
    """Standard normal by Box-Muller on two counter-based uniforms."""
    u1 = _uniform(*ids, 0)
    u2 = _uniform(*ids, 1)
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)


# ----------------------------------------------------------------------------------------------
# model configuration + weight blob
# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass(frozen=True)
class ModelCfg:
    F: int
    T: int
    K: int
    H: int
    Zmax: int = 86
    cutoff: float = 5.0
    norm_eps: float = 1e-8
    pbc_images: str = "minimum"  # or "all": every periodic image inside the cutoff (cells narrower than 2 r_c)
    rbf: str = "gaussian"   # or "bessel" (the paper's lead model uses 4 Bessel functions)
    max_neighbors: int = 0  # > 0: every receiver keeps its nearest max_neighbors senders ("Max neighbors 20")
    n_global: int = 0       # global attributes per structure (charge, spin: PAPER.md:58) entering the embedding
    head_type: str = "atomwise"  # or "pooled": the paper's graph-level head, mean pool -> 2 shared
    head_d1: int = 50            # layers of width head_d1 -> per head 2 layers of width head_d2 -> 1
    head_d2: int = 776
    backbone: str = "painn"      # or "schnet": the second backbone on the same graph


@dataclasses.dataclass
class Batch:
    Z: np.ndarray            # [N] int32
    pos: np.ndarray          # [N,3] float64
    struct_ptr: np.ndarray   # [S+1] int32
    head: np.ndarray         # [S] int32
    cell: Optional[np.ndarray] = None   # [S,3,3] float64, rows = lattice vectors
    pbc: Optional[np.ndarray] = None    # [S,3] uint8

    @property
    def n_atoms(self) -> int:
        return int(self.Z.shape[0])

    @property
    def n_structs(self) -> int:
        return int(self.head.shape[0])

    def select(self, structs: Sequence[int]) -> "Batch":
        """Sub-batch made of the listed structures (in the given order)."""
        parts = []
        for g in structs:
            a, b = int(self.struct_ptr[g]), int(self.struct_ptr[g + 1])
            parts.append(Batch(self.Z[a:b], self.pos[a:b], np.array([0, b - a], np.int32),
                               self.head[g:g + 1],
                               None if self.cell is None else self.cell[g:g + 1],
                               None if self.pbc is None else self.pbc[g:g + 1]))
        return concat_batches(parts)


def concat_batches(parts: Sequence[Batch]) -> Batch:
    Z = np.concatenate([p.Z for p in parts]).astype(np.int32)
    pos = np.concatenate([p.pos for p in parts]).astype(np.float64)
    sizes = np.concatenate([np.diff(p.struct_ptr) for p in parts])
    sp = np.zeros(sizes.size + 1, np.int32)
    sp[1:] = np.cumsum(sizes)
    head = np.concatenate([p.head for p in parts]).astype(np.int32)
    if any(p.cell is not None for p in parts):
        cells, pbcs = [], []
        for p in parts:
            if p.cell is None:
                cells.append(np.tile(np.eye(3), (p.n_structs, 1, 1)))
                pbcs.append(np.zeros((p.n_structs, 3), np.uint8))
            else:
                cells.append(p.cell)
                pbcs.append(p.pbc)
        return Batch(Z, pos, sp, head, np.concatenate(cells), np.concatenate(pbcs).astype(np.uint8))
    return Batch(Z, pos, sp, head)


def weights_layout(mc: ModelCfg):
    """[(name, shape, fan_in, offset)] in the blob order of SURVEY.md §8(b)."""
    F, T, K, H = mc.F, mc.T, mc.K, mc.H
    out, off = [], 0

    def add(name, shape, fan_in):
        nonlocal off
        out.append((name, tuple(shape), fan_in, off))
        off += int(np.prod(shape))

    add("emb", (mc.Zmax + 1, F), 1)
    if getattr(mc, "backbone", "painn") == "schnet":   # continuous-filter convolution blocks (reading Q31)
        for t in range(T):
            add(f"b{t}.flt_W1", (F, K), K); add(f"b{t}.flt_b1", (F,), K)
            add(f"b{t}.flt_W2", (F, F), F); add(f"b{t}.flt_b2", (F,), F)
            add(f"b{t}.in_W", (F, F), F)
            add(f"b{t}.out_W1", (F, F), F); add(f"b{t}.out_b1", (F,), F)
            add(f"b{t}.out_W2", (F, F), F); add(f"b{t}.out_b2", (F,), F)
        for h in range(H):
            add(f"h{h}.out_W1", (F // 2, F), F)
            add(f"h{h}.out_b1", (F // 2,), F)
            add(f"h{h}.out_w2", (F // 2,), F // 2)
            add(f"h{h}.out_b2", (1,), F // 2)
        return out
    for t in range(T):
        add(f"b{t}.msg_W1", (F, F), F)
        add(f"b{t}.msg_b1", (F,), F)
        add(f"b{t}.msg_W2", (3 * F, F), F)
        add(f"b{t}.msg_b2", (3 * F,), F)
        add(f"b{t}.flt_W", (3 * F, K), K)
        add(f"b{t}.flt_b", (3 * F,), K)
        add(f"b{t}.upd_U", (F, F), F)
        add(f"b{t}.upd_V", (F, F), F)
        add(f"b{t}.upd_A1", (F, 2 * F), 2 * F)
        add(f"b{t}.upd_c1", (F,), 2 * F)
        add(f"b{t}.upd_A2", (3 * F, F), F)
        add(f"b{t}.upd_c2", (3 * F,), F)
    if getattr(mc, "head_type", "atomwise") == "pooled":
        d1, d2 = mc.head_d1, mc.head_d2
        add("pool.W1", (d1, F), F); add("pool.b1", (d1,), F)
        add("pool.W2", (d1, d1), d1); add("pool.b2", (d1,), d1)
        for h in range(H):
            add(f"h{h}.br_W1", (d2, d1), d1); add(f"h{h}.br_b1", (d2,), d1)
            add(f"h{h}.br_W2", (d2, d2), d2); add(f"h{h}.br_b2", (d2,), d2)
            add(f"h{h}.br_w3", (d2,), d2); add(f"h{h}.br_b3", (1,), d2)
    for h in range(H if getattr(mc, "head_type", "atomwise") != "pooled" else 0):
        add(f"h{h}.out_W1", (F // 2, F), F)
        add(f"h{h}.out_b1", (F // 2,), F)
        add(f"h{h}.out_w2", (F // 2,), F // 2)
        add(f"h{h}.out_b2", (1,), F // 2)
    if getattr(mc, "n_global", 0) > 0:   # global attributes (charge, spin): glob_W [F][n_global], appended
        add("glob_W", (F, mc.n_global), 1)
    return out


def weights_count(mc: ModelCfg) -> int:
    name, shape, _, off = weights_layout(mc)[-1]
    return off + int(np.prod(shape))


def make_weights(mc: ModelCfg, cfg_id: int = 0, seed: int = BASE_SEED) -> np.ndarray:
    """Flat FP64 blob; every matrix and bias i.i.d. N(0, 1/fan_in), embedding N(0,1)."""
    blob = np.empty(weights_count(mc), np.float64)
    for tid, (name, shape, fan_in, off) in enumerate(weights_layout(mc)):
        n = int(np.prod(shape))
        z = _normal(seed, cfg_id, _T_W, tid, np.arange(n, dtype=np.uint64))
        blob[off:off + n] = z / math.sqrt(fan_in)
    return blob


def make_head_weights(cfg_id: int, struct_ids, H: int, sharpness: float = 6.0, seed: int = BASE_SEED) -> np.ndarray:
    """Per-structure branch weights [S,H] for blended multi-head inference: a softmax of seeded normal logits scaled by
    `sharpness`, rounded to 6 decimals.  Stands in for the paper's composition-MLP softmax, which on
    real inputs leaves ~81 % of the branches negligible; the default sharpness gives a similar share."""
    ids = np.asarray(struct_ids, np.uint64)
    z = np.stack([_normal(seed, cfg_id, _T_HW, ids, np.full(ids.shape, h, np.uint64)) for h in range(H)], axis=1)
    z = sharpness * z
    e = np.exp(z - z.max(axis=1, keepdims=True))
    return np.round(e / e.sum(axis=1, keepdims=True), 6)


BRANCH_MLP_WIDTHS = (118, 128, 64, 16)      # 118*128+128 + 128*64+64 + 64*16+16 = 24,528 parameters ("24,500")


def branch_mlp_count(widths: Sequence[int]) -> int:
    return sum(widths[l + 1] * widths[l] + widths[l + 1] for l in range(len(widths) - 1))


def make_branch_mlp(widths: Sequence[int] = BRANCH_MLP_WIDTHS, sharpness: float = 70.0, seed: int = BASE_SEED) -> np.ndarray:
    """Flat FP64 parameter blob of the composition -> branch-weight MLP: per layer W [out, in] row-major, then b [out].
    Seeded normals: first layer N(0,1) (its input is a composition vector whose entries sum to 1), later layers
    N(0, 1/fan_in), biases N(0, 0.01); the last layer is scaled by `sharpness` so that the softmax is as peaked as the
    paper's trained router (~81 % of the branches negligible).  No arithmetic of the method here."""
    blob = np.empty(branch_mlp_count(widths), np.float64)
    off = 0
    L = len(widths) - 1
    for l in range(L):
        n_in, n_out = widths[l], widths[l + 1]
        zw = _normal(seed, 0, _T_BW, 2 * l, np.arange(n_out * n_in, dtype=np.uint64))
        zb = _normal(seed, 0, _T_BW, 2 * l + 1, np.arange(n_out, dtype=np.uint64))
        gain = (1.0 if l == 0 else 1.0 / math.sqrt(n_in)) * (sharpness if l == L - 1 else 1.0)
        blob[off:off + n_out * n_in] = zw * gain
        off += n_out * n_in
        blob[off:off + n_out] = zb * 0.1
        off += n_out
    return blob


def unpack_weights(mc: ModelCfg, blob: np.ndarray) -> dict:
    return {name: blob[off:off + int(np.prod(shape))].reshape(shape)
            for name, shape, _, off in weights_layout(mc)}


# ----------------------------------------------------------------------------------------------
# molecules (configs 1, 2, 4): sequential insertion with rejection at min distance
# ----------------------------------------------------------------------------------------------
def make_molecules(cfg_id: int, struct_ids, n_lo: int, n_hi: int, *, density: Optional[float],
                   box: Optional[float], z_choices: np.ndarray, H: int, cutoff: float,
                   min_dist: float = 0.9, seed: int = BASE_SEED) -> Batch:
    sid = np.asarray(struct_ids, dtype=np.uint64).ravel()
    S = sid.size
    n = (n_lo + np.floor(_uniform(seed, cfg_id, sid, _T_NATOMS) * (n_hi - n_lo + 1))).astype(np.int64)
    n = np.minimum(n, n_hi)
    side = np.full(S, box, np.float64) if box is not None else np.cbrt(n / density)
    head = np.minimum((_uniform(seed, cfg_id, sid, _T_HEAD) * H).astype(np.int32), H - 1)
    nmax = int(n.max()) if S else 0
    pos = np.zeros((S, nmax, 3), np.float64)
    redraw = np.zeros(S, np.uint64)            # structure-level attempt counter (margin rejection)
    todo = np.arange(S)
    coord = np.arange(3, dtype=np.uint64)
    while todo.size:
        for k in range(nmax):
            pend = todo[n[todo] > k]
            attempt = np.zeros(S, np.uint64)
            while pend.size:
                u = _uniform(seed, cfg_id, sid[pend, None], redraw[pend, None], _T_POS, k,
                             attempt[pend, None], coord[None, :])
                cand = u * side[pend, None]
                if k > 0:
                    d2 = ((pos[pend, :k, :] - cand[:, None, :]) ** 2).sum(-1).min(-1)
                    ok = d2 >= min_dist * min_dist
                else:
                    ok = np.ones(pend.size, bool)
                pos[pend[ok], k, :] = cand[ok]
                attempt[pend[~ok]] += np.uint64(1)
                pend = pend[~ok]
        # margin check: no pair distance within MARGIN of the cutoff
        sub = pos[todo]
        d = np.sqrt(((sub[:, :, None, :] - sub[:, None, :, :]) ** 2).sum(-1))
        valid = (np.arange(nmax)[None, :] < n[todo, None])
        pairm = valid[:, :, None] & valid[:, None, :]
        bad = (np.abs(d - cutoff) < MARGIN) & pairm
        badm = bad.any(axis=(1, 2))
        redraw[todo[badm]] += np.uint64(1)
        todo = todo[badm]
    k_idx = np.arange(nmax, dtype=np.uint64)
    zi = np.minimum((_uniform(seed, cfg_id, sid[:, None], _T_Z, k_idx[None, :]) * len(z_choices)).astype(np.int64),
                    len(z_choices) - 1)
    Zall = np.asarray(z_choices, np.int32)[zi]
    mask = np.arange(nmax)[None, :] < n[:, None]
    sp = np.zeros(S + 1, np.int32)
    sp[1:] = np.cumsum(n)
    return Batch(Zall[mask].astype(np.int32), pos[mask].reshape(-1, 3).copy(), sp, head.astype(np.int32))


# ----------------------------------------------------------------------------------------------
# crystals (configs 3, 5): jittered BCC lattice in a cubic periodic cell
# ----------------------------------------------------------------------------------------------
def _crystal_margin_ok(pos: np.ndarray, L: float, cutoff: float) -> bool:
    n = pos.shape[0]
    if n <= 4096:
        d = pos[None, :, :] - pos[:, None, :]
        f = d / L
        off = ~np.eye(n, dtype=bool)
        if (np.abs(np.abs(f) - 0.5) < MARGIN)[off].any():
            return False
        r = d - np.round(f) * L
        dist = np.sqrt((r ** 2).sum(-1))
        return not (np.abs(dist - cutoff) < MARGIN)[off].any()
    from scipy.spatial import cKDTree
    assert L > 2.0 * cutoff + 1e-6, "large periodic structures need L > 2*cutoff"
    tree = cKDTree(pos, boxsize=L)
    return int(tree.count_neighbors(tree, cutoff + MARGIN)) == int(tree.count_neighbors(tree, cutoff - MARGIN))


def make_crystals(cfg_id: int, struct_ids, n_atoms: int, *, density: float, sigma: float, H: int,
                  cutoff: float, zmax: int = 86, seed: int = BASE_SEED) -> Batch:
    sid = np.asarray(struct_ids, dtype=np.uint64).ravel()
    S = sid.size
    L = float(np.cbrt(n_atoms / density))
    m = int(math.ceil((n_atoms / 2.0) ** (1.0 / 3.0) - 1e-12))
    a = L / m
    g = np.arange(m, dtype=np.float64)
    corner = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    sites = np.stack([corner, corner + 0.5], 1).reshape(-1, 3) * a        # order: (i,j,k,basis)
    nsites = sites.shape[0]
    site_idx = np.arange(nsites, dtype=np.uint64)
    coord = np.arange(3, dtype=np.uint64)
    Zs, Ps = [], []
    for s in sid:
        attempt = 0
        while True:
            keep = np.ones(nsites, bool)
            if nsites > n_atoms:
                keys = _hash(seed, cfg_id, s, attempt, _T_SHUF, site_idx)
                keep[np.argsort(keys, kind="stable")[: nsites - n_atoms]] = False
            base = sites[keep]
            at = np.arange(n_atoms, dtype=np.uint64)
            jit = _normal(seed, cfg_id, s, attempt, _T_JIT, at[:, None], coord[None, :]) * sigma
            pos = np.mod(base + jit, L)
            if _crystal_margin_ok(pos, L, cutoff):
                break
            attempt += 1
        zi = np.minimum((_uniform(seed, cfg_id, s, _T_Z, at) * zmax).astype(np.int32), zmax - 1) + 1
        Zs.append(zi.astype(np.int32))
        Ps.append(pos)
    head = np.minimum((_uniform(seed, cfg_id, sid, _T_HEAD) * H).astype(np.int32), H - 1)
    sp = np.arange(S + 1, dtype=np.int32) * n_atoms
    cell = np.tile(np.eye(3) * L, (S, 1, 1))
    pbc = np.ones((S, 3), np.uint8)
    return Batch(np.concatenate(Zs), np.concatenate(Ps), sp, head.astype(np.int32), cell, pbc)


# ----------------------------------------------------------------------------------------------
# the five BASELINE.json configs
# ----------------------------------------------------------------------------------------------
CONFIGS = {
    1: dict(name="cfg1_tiny_fp64", kind="mol", S=8, n_lo=16, n_hi=16, box=6.0, density=None,
            z_choices=(1, 6, 7, 8), model=ModelCfg(F=32, T=2, K=20, H=1, cutoff=5.0),
            precision="fp64", forces=True),
    2: dict(name="cfg2_molecular_fp32", kind="mol", S=256, n_lo=20, n_hi=60, box=None, density=0.05,
            z_choices=tuple(range(1, 87)), model=ModelCfg(F=128, T=3, K=20, H=16, cutoff=5.0),
            precision="fp32", forces=True),
    3: dict(name="cfg3_crystals", kind="xtal", S=64, n_atoms=128, density=0.08, sigma=0.1,
            model=ModelCfg(F=256, T=4, K=32, H=16, cutoff=6.0), precision="fp32", forces=True),
    4: dict(name="cfg4_screening_bf16", kind="mol", S=1048576, n_lo=8, n_hi=40, box=None, density=0.05,
            z_choices=tuple(range(1, 87)), model=ModelCfg(F=256, T=4, K=20, H=16, cutoff=5.0),
            precision="bf16", forces=False, stream_batch=16384),
    5: dict(name="cfg5_large_fp64", kind="xtal", S=1, n_atoms=100000, density=0.08, sigma=0.1,
            model=ModelCfg(F=256, T=4, K=32, H=1, cutoff=5.0), precision="fp64", forces=True),
}


def model_cfg(cfg_id: int) -> ModelCfg:
    return CONFIGS[cfg_id]["model"]


def make_batch(cfg_id: int, first: int = 0, count: Optional[int] = None, *, struct_ids=None,
               n_atoms: Optional[int] = None, seed: int = BASE_SEED) -> Batch:
    """Structures [first, first+count) (or the explicit `struct_ids`) of config `cfg_id`.

    `n_atoms` overrides the per-structure atom count of the crystal configs (scaled-down
    parity cases of config 5)."""
    c = CONFIGS[cfg_id]
    if struct_ids is None:
        if count is None:
            count = c["S"] - first
        struct_ids = np.arange(first, first + count)
    mc: ModelCfg = c["model"]
    if c["kind"] == "mol":
        return make_molecules(cfg_id, struct_ids, c["n_lo"], c["n_hi"], density=c["density"], box=c["box"],
                              z_choices=np.array(c["z_choices"]), H=mc.H, cutoff=mc.cutoff, seed=seed)
    return make_crystals(cfg_id, struct_ids, n_atoms or c["n_atoms"], density=c["density"], sigma=c["sigma"],
                         H=mc.H, cutoff=mc.cutoff, zmax=mc.Zmax, seed=seed)
