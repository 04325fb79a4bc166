"""The oracle reproduces tests/golden/tiny_score.json (written by tests/golden/make_golden.py from the oracle alone)
bit for bit: a guard against accidental changes of the pinned oracle's arithmetic."""
import json
import os

import numpy as np


def _load():
    with open(os.path.join(os.path.dirname(__file__), "golden", "tiny_score.json")) as f:
        g = json.load(f)
    G = np.stack([np.frombuffer(bytes.fromhex(h), np.float32) for h in g["genotypes_f32_hex"]])
    E = np.array([float.fromhex(v) for v in g["E"]])
    grad = np.array([[float.fromhex(v) for v in row] for row in g["grad"]])
    return g, G, E, grad


def test_oracle_reproduces_golden_bit_for_bit(tiny, orc, par, W):
    g, G, E, grad = _load()
    assert np.array_equal(G, W.make_genotypes(12, tiny["lig"].R, tiny["grids"], seed=0, wall_tail=0.0))     # the generator is frozen too
    r = orc.score(tiny["og"], tiny["ol"], par, G)
    assert np.array_equal(r["E"], E) and np.array_equal(r["grad"], grad)
    assert tiny["ol"].npairs == g["npairs"] and tiny["ol"].pairs[:8].tolist() == g["pairs_head"]
