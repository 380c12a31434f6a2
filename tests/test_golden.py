"""The paper's printed constants (tests/golden/, each with its citation) against the oracle."""
import math
import os

import numpy as np

from oracle import solver as osv

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_filters_match_paper_text():
    rows = [l.split() for l in open(os.path.join(GOLD, "tf_filters.txt")) if l.strip() and not l.startswith("#")]
    assert [r[0] for r in rows] == ["h0", "h1", "h2"]
    for k, r in enumerate(rows):
        scale = float(r[1]) / float(r[2]) * (math.sqrt(2.0) if r[3] == "1" else 1.0)
        taps = np.array([float(x) for x in r[4:7]]) * scale
        assert np.allclose(osv.H[k], taps, rtol=0, atol=1e-16)


def test_paper_constants_are_what_the_oracle_uses():
    kv = {}
    for l in open(os.path.join(GOLD, "paper_constants.txt")):
        l = l.split("#")[0].split()
        if len(l) == 2:
            kv[l[0]] = float(l[1])
    a = osv.tf_decompose(np.zeros((2, 2, 2)))
    assert a.shape[0] - 1 == kv["n_high_bands"]
    assert osv.a2_t_next(kv["t_init"]) == (1 + math.sqrt(5)) / 2
