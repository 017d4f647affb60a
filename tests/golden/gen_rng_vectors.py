"""Writes tests/golden/rng_vectors.txt: known-answer vectors of the pair hash (DESIGN.md
'RNG specification').  Calls ONLY the oracle (oracle/mdpd_ref.c); never the CUDA path.
Run from the repo root:  python tests/golden/gen_rng_vectors.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle.mdpd_ref import ref_hash  # noqa: E402

rng = np.random.default_rng(20190310134)
rows = [(0, 1, 0, 0), (0, 1, 1, 0), (0, 1, 0, 1), (1, 2, 0, 12345), (0, 2 ** 31 - 1, 2 ** 32 - 1, 2 ** 32 - 1),
        (5999, 6000, 100, 12345), (32156248, 32156249, 999, 12345)]
while len(rows) < 48:
    a, b = sorted(int(x) for x in rng.integers(0, 2 ** 25, 2))
    if a != b:
        rows.append((a, b, int(rng.integers(0, 20000)), int(rng.integers(0, 2 ** 32))))
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "rng_vectors.txt"), "w") as f:
    f.write("# Known-answer vectors of h = HASH(min tag, max tag, step, seed), DESIGN.md 'RNG specification'.\n"
            "# Written by tests/golden/gen_rng_vectors.py from the fp64 oracle (oracle/mdpd_ref.c) only.\n"
            "# The paper fixes no generator (PAPER.md L75 says only 'random variable xi_ij'); these freeze ours.\n"
            "# columns: a b step seed h(hex)\n")
    for a, b, k, s in rows:
        f.write(f"{a} {b} {k} {s} {ref_hash(a, b, k, s):08x}\n")
print("wrote", len(rows), "vectors")
