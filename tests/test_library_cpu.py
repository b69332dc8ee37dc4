"""-m "not gpu": the C-ABI library builds for sm_100a, loads, exports every symbol include/pnn.h declares, and its
host-only entry points behave; the product never routes through the oracle; host-side sharding logic incl. a
world_size-2 gloo run.  No compute calls (no GPU here)."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

import gen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pnn():
    from paper_2604_15380_b200 import build
    build.build()
    import paper_2604_15380_b200 as p
    p.lib()
    return p


def test_exports_every_declared_symbol(pnn):
    hdr = open(os.path.join(ROOT, "include", "pnn.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(pnn_[a-z_0-9]+)\s*\(", hdr))
    assert {"pnn_eval", "pnn_build_graph", "pnn_model_create", "pnn_workspace_create", "pnn_graph_view"} <= names
    lib = ctypes.CDLL(pnn.lib_path())
    for n in sorted(names):
        assert hasattr(lib, n), f"libpnn.so does not export {n}"
    for n in names:                      # the Python binding offers the same names
        assert hasattr(pnn, n), f"binding lacks {n}"


def test_weight_blob_size_matches_generators(pnn):
    for cid in gen.CONFIGS:
        mc = gen.model_cfg(cid)
        for prec in (pnn.PNN_BF16, pnn.PNN_FP32, pnn.PNN_FP64):
            cfg = pnn.pnn_config(mc.F, mc.T, mc.K, mc.H, mc.Zmax, mc.cutoff, mc.norm_eps, prec)
            assert pnn.pnn_weights_count(cfg) == gen.weights_count(mc)
    # F=256, T=4, K=32, H=16, Zmax=86 -> 3,543,824 scalars
    assert pnn.pnn_weights_count(pnn.pnn_config(256, 4, 32, 16, 86, 6.0, 1e-8, pnn.PNN_FP32)) == 3543824
    # pooled graph-level heads and global attribute columns change the blob the same way on both sides
    import dataclasses
    mc = dataclasses.replace(gen.model_cfg(2), head_type="pooled", head_d1=50, head_d2=776, n_global=2)
    cfg = pnn.pnn_config(mc.F, mc.T, mc.K, mc.H, mc.Zmax, mc.cutoff, mc.norm_eps, pnn.PNN_FP32, 0, 0, 0, 2, 1, 50, 776)
    assert pnn.pnn_weights_count(cfg) == gen.weights_count(mc)
    mcs = dataclasses.replace(gen.model_cfg(2), backbone="schnet")   # second backbone: other block arrays, same heads
    cfgs = pnn.pnn_config(mcs.F, mcs.T, mcs.K, mcs.H, mcs.Zmax, mcs.cutoff, mcs.norm_eps, pnn.PNN_FP64, 0, 0, 0, 0, 0, 50, 776, 1)
    assert pnn.pnn_weights_count(cfgs) == gen.weights_count(mcs)
    with pytest.raises(pnn.PnnError):   # the second backbone has no BF16 path
        pnn.pnn_weights_count(pnn.pnn_config(mcs.F, mcs.T, mcs.K, mcs.H, mcs.Zmax, mcs.cutoff, mcs.norm_eps, pnn.PNN_BF16, 0, 0,
                                             0, 0, 0, 50, 776, 1))
    with pytest.raises(pnn.PnnError):   # widths whose activations do not fit one CTA's shared memory
        pnn.pnn_weights_count(pnn.pnn_config(64, 2, 20, 2, 86, 5.0, 1e-8, pnn.PNN_FP64, 0, 0, 0, 0, 1, 50, 4000))


@pytest.mark.parametrize("bad", [dict(F=48), dict(F=512), dict(F=0), dict(K=1), dict(K=33), dict(T=0), dict(H=0),
                                 dict(cutoff=0.0), dict(prec=7)])
def test_invalid_configs_are_rejected(pnn, bad):
    base = dict(F=64, T=2, K=20, H=2, Zmax=86, cutoff=5.0, norm_eps=1e-8, prec=pnn.PNN_FP32)
    base.update(bad)
    with pytest.raises(pnn.PnnError) as ei:
        pnn.pnn_weights_count(pnn.pnn_config(*[base[k] for k in ("F", "T", "K", "H", "Zmax", "cutoff", "norm_eps",
                                                                  "prec")]))
    assert ei.value.status == -1


def test_status_strings(pnn):
    assert pnn.pnn_status_string(0) == "ok"
    for st in range(-6, 0):
        assert pnn.pnn_status_string(st) not in ("ok", "unknown status")


def test_fails_loudly_without_a_gpu(pnn):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    mc = gen.model_cfg(1)
    with pytest.raises(pnn.PnnError) as ei:          # no CPU fallback: model upload needs the device
        pnn.PaiNN(mc.F, mc.T, mc.K, mc.H, gen.make_weights(mc, 1), precision="fp32", max_atoms=16, max_edges=64,
                  max_structs=1)
    assert ei.value.status == -3 and "cuda" in str(ei.value).lower()


def test_product_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_2604_15380_b200")
    for dp, _, fs in os.walk(pkg):
        if os.path.basename(dp) in ("build", "__pycache__"):
            continue
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), f
                assert "painn_oracle" not in src and "oracle/" not in src, f
    ora = open(os.path.join(ROOT, "oracle", "painn_oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "libpnn" not in ora and "import paper_2604_15380_b200" not in ora and "csrc" not in ora


# ------------------------------------------------------------------------------------------------ sharding
def test_partition_properties():
    from paper_2604_15380_b200.sharding import partition
    rng = np.random.default_rng(0)
    for world in (1, 2, 3, 8):
        for n in (0, 1, 5, 257):
            cost = rng.integers(1, 100, n).astype(float)
            parts = partition(cost, world)
            assert len(parts) == world and parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            assert all(lo <= hi for lo, hi in parts)
            if n >= 8 * world:
                loads = [cost[lo:hi].sum() for lo, hi in parts]
                assert max(loads) <= cost.sum() / world + cost.max()


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r}); sys.path.insert(0, os.path.join({root!r}, "tests"))
import numpy as np, torch, torch.distributed as dist
import gen, oracle
from paper_2604_15380_b200.sharding import partition, gather_energies
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
mc = gen.model_cfg(1); w = gen.make_weights(mc, 1); b = gen.make_batch(1)
sizes = np.diff(b.struct_ptr)
parts = partition(sizes + 11.0 * sizes, 2)
lo, hi = parts[rank]
out = oracle.evaluate(mc, w, b.select(range(lo, hi)))      # stands in for the per-rank GPU evaluation (no GPU here)
e = gather_energies(torch.from_numpy(out["energy"]), [p[1] - p[0] for p in parts])
ref = oracle.evaluate(mc, w, b)["energy"]
assert np.allclose(e.numpy(), ref, rtol=0, atol=1e-12), (e, ref)
dist.barrier(); dist.destroy_process_group()
print("rank", rank, "ok")
"""


def test_two_rank_gloo_shard_and_gather(tmp_path):
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=port))
    env = dict(os.environ, OMP_NUM_THREADS="2")
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT,
                              env=env) for r in range(2)]
    outs = [p.communicate(timeout=240)[0].decode() for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    assert all("ok" in o for o in outs)
