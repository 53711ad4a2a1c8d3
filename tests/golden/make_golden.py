"""Writes tests/golden/tiny_path.json by calling ONLY oracle/ (never the CUDA path).
Run:  python tests/golden/make_golden.py"""
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from oracle import oracle as O            # noqa: E402
from paper_1409_2065_b200 import synth   # noqa: E402

wl = synth.make("tiny")
X = wl.X.astype(np.float64)
ei, ej, w, _ = O.knn_graph(X, None, wl.k, wl.phi)
gammas = [float(g) for g in synth.gamma_grid(1e-3, 1e3, 7)]
iters = 150
res = O.path(X, None, ei, ej, w, gammas, iters)
out = {"source": "oracle/oracle.py path(); tiny config (BASELINE.json configs[0]); no value from the CUDA path",
       "n_pairs": int(len(ei)), "gammas": gammas, "iters": iters,
       "per_gamma": [{"phi_last": float(r["phi"][-1]), "U_fro": float(np.linalg.norm(r["U"])),
                      "nclusters": int(r["nclusters"])} for r in res]}
with open(os.path.join(HERE, "tiny_path.json"), "w") as f:
    json.dump(out, f, indent=1)
print(out)
