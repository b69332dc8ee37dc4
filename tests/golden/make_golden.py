"""Writes tests/golden/cfg1_oracle.npz: config-1 energies and forces as computed by the ORACLE
(calls only gen/ and oracle/; never the CUDA path).  Run: python tests/golden/make_golden.py"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import gen      # noqa: E402
import oracle   # noqa: E402

mc = gen.model_cfg(1)
out = oracle.evaluate(mc, gen.make_weights(mc, 1), gen.make_batch(1))
np.savez(os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_oracle.npz"),
         energy=out["energy"], forces=out["forces"], n_edges=out["n_edges"])
print("wrote cfg1_oracle.npz", out["energy"])
