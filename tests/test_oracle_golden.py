"""The oracle against the hand-applied Fig. 3 formula in tests/golden/fig3_module_start.txt."""
import os

import numpy as np

import oracle
import pixgen
from helpers import P, hand_event

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "fig3_module_start.txt")


def rows():
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        cap, counts, starts = (part.split() for part in line.split("|"))
        yield int(cap[0]), [int(x) for x in counts], [int(x) for x in starts]


def test_fig3_clamp_and_scan():
    det = pixgen.detector("tiny")
    n_rows = 0
    for cap, counts, starts in rows():
        module, row, col = [], [], []
        for m, k in enumerate(counts):          # k isolated pixels in module m: k single-pixel clusters
            for j in range(k):
                module.append(m); row.append(10 + 4 * j); col.append(7 + 5 * j)
        adc = np.full(len(module), 255)          # far above the 4000 e cluster cut
        words, fed_off, _ = hand_event(det, module, row, col, adc)
        o = oracle.process(det, words, fed_off, dict(P, max_clusters_per_module=cap), max_clusters_per_event=64)
        got = o["clus_module_start"].astype(np.int64)
        assert got[:len(starts)].tolist() == starts
        assert np.all(got[len(starts):] == starts[-1])           # the other modules are empty
        assert int(o["summary"][13]) == sum(counts)               # clusters surviving the cut
        assert int(o["summary"][14]) == starts[-1]                # clusters emitted after the clamp
        n_rows += 1
    assert n_rows == 3
