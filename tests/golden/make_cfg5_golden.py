"""Writes tests/golden/cfg5_oracle.npz: the ORACLE's result for config 5 at FULL size (one periodic cell of 100,000 atoms,
BASELINE.json configs[4]) — calls only gen/ and oracle/, never the CUDA path.  Minutes of CPU (O(N^2) neighbour search plus
about 5.5 TFLOP of FP64 loops).  Stored: the CSR degree of every atom (uint8: the whole rowptr), the edge count, the energy,
and the forces of 2,000 seeded sample atoms.  Run: python tests/golden/make_cfg5_golden.py"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import gen      # noqa: E402
import oracle   # noqa: E402

mc = gen.model_cfg(5)
b = gen.make_batch(5)
w = gen.make_weights(mc, 5)
assert b.n_atoms == 100000
t0 = time.time()
nb = oracle.neighbours(b, mc.cutoff)
deg = np.diff(nb["rowptr"])
assert deg.max() < 256
print(f"neighbours: {nb['recv'].size} edges, {time.time() - t0:.0f} s", flush=True)
t0 = time.time()
out = oracle.evaluate(mc, w, b)
print(f"evaluate: {time.time() - t0:.0f} s, energy {out['energy']}", flush=True)
assert out["n_edges"] == nb["recv"].size
sample = np.sort(np.random.default_rng(2604015380).choice(b.n_atoms, 2000, replace=False)).astype(np.int32)
# a checksum of the sender lists (order-independent per receiver): sum and xor of senders per atom, folded
send_sum = np.zeros(b.n_atoms, np.int64)
np.add.at(send_sum, nb["recv"], nb["send"].astype(np.int64))
np.savez_compressed(os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg5_oracle.npz"),
                    degree=deg.astype(np.uint8), n_edges=np.int64(out["n_edges"]), energy=out["energy"],
                    sample=sample, forces_sample=out["forces"][sample],
                    force_rms=np.sqrt(np.mean(out["forces"] ** 2)), force_sum=out["forces"].sum(0),
                    sender_sum_sample=send_sum[sample])
print("wrote cfg5_oracle.npz")
