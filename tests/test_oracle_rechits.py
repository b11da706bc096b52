"""Pins of the oracle's RecHits-lite (S25-S28): closed forms on hand-built clusters and an independent
vectorised recomputation (numpy group-by) on generated events."""
import numpy as np

import oracle
import pixgen
from helpers import P, hand_event


def run(det, module, row, col, adc, **kw):
    words, fed_off, perm = hand_event(det, module, row, col, adc)
    o = oracle.process(det, words, fed_off, dict(P, **kw), max_clusters_per_event=4096)
    return o, oracle.rechits(det, o), perm


def test_single_pixels_closed_form():
    det = pixgen.detector("tiny")
    pts = [(0, 0), (0, 415), (159, 0), (159, 415), (80, 208), (77, 205), (17, 52), (100, 51)]
    o, h, _ = run(det, [3] * len(pts), [p[0] for p in pts], [p[1] for p in pts], [255] * len(pts))
    assert len(h["flags"]) == len(pts)
    for g in range(len(pts)):
        r, c = int(o["row"][o["c_first_digi"][g]]), int(o["col"][o["c_first_digi"][g]])
        assert (h["min_row"][g], h["max_row"][g], h["min_col"][g], h["max_col"][g]) == (r, r, c, c)
        # S27: centre of the pixel, module centre as origin, 100 um x 150 um cells
        assert h["x_local"][g] == np.float32(np.float32(np.float32(np.float32(r) + np.float32(0.5)) - np.float32(80)) * np.float32(0.01))
        assert h["y_local"][g] == np.float32(np.float32(np.float32(np.float32(c) + np.float32(0.5)) - np.float32(208)) * np.float32(0.015))
        on_edge = r in (0, 159) or c in (0, 415)
        assert h["flags"][g] == (1 if on_edge else 0) | 4          # single pixel, never spans a read-out chip
    assert abs(float(h["x_local"][[p == (80, 208) for p in pts].index(True)]) - 0.005) < 1e-7
    assert abs(float(h["y_local"][[p == (80, 208) for p in pts].index(True)]) - 0.0075) < 1e-7


def test_spans_roc_and_edges():
    det = pixgen.detector("tiny")
    # module 0: a 2-pixel cluster across the row boundary 79|80; one across the column boundary 51|52; one inside
    rows = [79, 80, 10, 10, 120, 120, 121]
    cols = [300, 300, 51, 52, 100, 101, 101]
    o, h, _ = run(det, [0] * 7, rows, cols, [200] * 7)
    assert len(h["flags"]) == 3
    by_first = {(int(o["row"][f]), int(o["col"][f])): g for g, f in enumerate(o["c_first_digi"])}
    assert h["flags"][by_first[(79, 300)]] == 2
    assert h["flags"][by_first[(10, 51)]] == 2
    g = by_first[(120, 100)]
    assert h["flags"][g] == 0
    assert (h["min_row"][g], h["max_row"][g], h["min_col"][g], h["max_col"][g]) == (120, 121, 100, 101)


def test_full_rows_cluster_is_centred_in_x():
    """A cluster of two full rows 79 and 80: the charge does not depend on the row (gains are per column), so the
    row centroid is 79.5 and local x is 0; the box is the full width and touches both column edges."""
    det = pixgen.detector("tiny")
    cols = np.tile(np.arange(416), 2)
    rows = np.repeat([79, 80], 416)
    o, h, _ = run(det, np.full(832, 5), rows, cols, np.full(832, 120))
    assert len(h["flags"]) == 1
    assert abs(float(h["x_local"][0])) < 1e-6
    assert (h["min_row"][0], h["max_row"][0], h["min_col"][0], h["max_col"][0]) == (79, 80, 0, 415)
    assert h["flags"][0] == 1 | 2


def test_against_numpy_groupby():
    det = pixgen.detector("full")
    b = pixgen.events(det, ["pu50", "edges", "dups"], [1, 2, 3])
    for e in range(3):
        o = oracle.process(det, *b.event(e), P)
        h = oracle.rechits(det, o)
        k = len(h["flags"])
        ok = o["status"] == 0
        gid = o["clus_module_start"][o["module"][ok].astype(np.int64)].astype(np.int64) + o["clus"][ok]
        for name, arr, fn, init in (("min_row", o["row"], np.minimum, 1 << 20), ("max_row", o["row"], np.maximum, -1),
                                    ("min_col", o["col"], np.minimum, 1 << 20), ("max_col", o["col"], np.maximum, -1)):
            acc = np.full(k, init, np.int64)
            fn.at(acc, gid, arr[ok].astype(np.int64))
            assert np.array_equal(acc, h[name].astype(np.int64)), name
        np.testing.assert_allclose(h["x_local"], (o["c_y_row"].astype(np.float64) + 0.5 - 80) * 0.01, rtol=1e-5, atol=1e-6)
        np.testing.assert_allclose(h["y_local"], (o["c_x_col"].astype(np.float64) + 0.5 - 208) * 0.015, rtol=1e-5, atol=1e-6)
        assert np.all(h["max_row"] - h["min_row"] + 1 <= o["c_n_pix"]) and np.all(h["max_col"] - h["min_col"] + 1 <= o["c_n_pix"])
        assert np.array_equal((h["flags"] & 4) != 0, o["c_n_pix"] == 1)


def test_module_clamp_drops_hits_with_their_records():
    det = pixgen.detector("tiny")
    rows = [10, 20, 30, 40, 50]
    o, h, _ = run(det, [2] * 5, rows, [7] * 5, [255] * 5, max_clusters_per_module=3)
    assert len(h["flags"]) == 3 and list(h["min_row"]) == [10, 20, 30]
