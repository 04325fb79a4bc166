"""Writes tests/golden/tiny_score.json: the ORACLE's energies, energy terms and gradients of 12 seeded genotypes of the
tiny config (BASELINE.json configs[0]).  The paper (arxiv 2007.03678) prints no worked example of the scoring function, so
this file is not a paper value: it is a regression fixture that freezes the pinned oracle (a later change of the oracle's
arithmetic must name its justification and regenerate it).  Calls only oracle/ and the seeded input generators.

    python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle                                                     # noqa: E402
from paper_2007_03678_b200 import workloads as W                  # noqa: E402  (input generators only)


def main():
    grids, lig = W.make_config("tiny")
    og, ol = oracle.Grids.from_workload(grids), oracle.Ligand.from_workload(lig)
    par = oracle.params(W.DEFAULT_PARAMS)
    G = W.make_genotypes(12, lig.R, grids, seed=0, wall_tail=0.0)
    r = oracle.score(og, ol, par, G)
    out = {"config": "tiny", "genotype_seed": 0, "n": 12,
           "genotypes_f32_hex": [g.astype(np.float32).tobytes().hex() for g in G],
           "E": [float.hex(float(v)) for v in r["E"]],
           "grad": [[float.hex(float(v)) for v in row] for row in r["grad"]],
           "npairs": int(ol.npairs), "pairs_head": ol.pairs[:8].tolist()}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_score.json"), "w") as f:
        json.dump(out, f, indent=1)
    print("wrote tiny_score.json:", out["E"][:2])


if __name__ == "__main__":
    main()
