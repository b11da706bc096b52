"""Pins for oracle O4-O7 (duplicates, 8-connected components, cut, renumber, records).  CPU only.

(i) scipy.ndimage.label with a 3x3 all-ones structure is an independent 8-connectivity routine;
(ii) tests/bruteforce.py restates the chain with O(n^2) adjacency and min-label relaxation;
(iii) closed forms discriminate the connectivity rule, the no-wrap rule and late merges.
"""
import numpy as np
import pytest
from scipy import ndimage

import oracle
import pixgen
from bruteforce import chain as brute_chain
from helpers import P, partition

DET = None


def det():
    global DET
    if DET is None:
        DET = pixgen.detector("tiny")
    return DET


def run_module(img_or_pixels, m=5, adc=255, params=P, order=None):
    """One module filled from a boolean image (160x416) or an (n,2) array of (row, col)."""
    if isinstance(img_or_pixels, np.ndarray) and img_or_pixels.dtype == bool:
        rc = np.argwhere(img_or_pixels)
    else:
        rc = np.asarray(img_or_pixels, np.int64).reshape(-1, 2)
    if order is not None:
        rc = rc[order]
    n = len(rc)
    a = np.full(n, adc) if np.isscalar(adc) else np.asarray(adc)
    w, fo, perm = det().stream(np.full(n, m), rc[:, 0], rc[:, 1], a)
    o = oracle.process(det(), w, fo, params)
    return o, rc[perm]


def n_clusters(o):
    return int(o["summary"][13])


@pytest.mark.parametrize("occ", [0.001, 0.01, 0.05, 0.10, 0.25, 0.40])
def test_against_scipy_label(occ):
    rng = np.random.default_rng(int(occ * 1000))
    img = rng.random((160, 416)) < occ
    lab, k = ndimage.label(img, structure=np.ones((3, 3), int))
    rc = np.argwhere(img)
    order = rng.permutation(len(rc))
    o, rc = run_module(img, order=order)
    assert np.all(o["status"] == 0)                      # adc 255 -> 33075 e, every cluster passes the cut
    assert n_clusters(o) == k
    scipy_sets = {}
    for i, (r, c) in enumerate(rc):
        scipy_sets.setdefault(lab[r, c], []).append(i)
    assert partition(o["clus"], o["module"], o["status"]) == {frozenset(v) for v in scipy_sets.values()}
    # canonical numbering: ids ordered by first digi index
    firsts = sorted(min(v) for v in scipy_sets.values())
    assert list(o["c_first_digi"]) == firsts
    for i in range(len(rc)):
        assert firsts[o["clus"][i]] <= i


def test_closed_forms():
    full = np.ones((160, 416), bool)
    assert n_clusters(run_module(full)[0]) == 1
    rr, cc = np.indices((160, 416))
    checker = (rr + cc) % 2 == 0
    o, _ = run_module(checker)
    assert n_clusters(o) == 1 and int(o["c_n_pix"][0]) == 33280   # 4-connectivity would give 33 280 singletons
    lattice = (rr % 2 == 0) & (cc % 2 == 0)
    o, _ = run_module(lattice)
    assert n_clusters(o) == 80 * 208 and np.all(o["c_n_pix"] == 1)
    stripes = rr % 2 == 0
    o, _ = run_module(stripes)
    assert n_clusters(o) == 80 and np.all(o["c_n_pix"] == 416)
    diag = [(i, i) for i in range(160)]
    assert n_clusters(run_module(diag)[0]) == 1
    anti = [(i, 200 - i) for i in range(160)]
    assert n_clusters(run_module(anti)[0]) == 1
    assert n_clusters(run_module([(7, 415), (8, 0)])[0]) == 2       # no wrap from col 415 to col 0 of the next row
    assert n_clusters(run_module([(159, 10), (0, 10)])[0]) == 2     # no wrap in rows
    assert n_clusters(run_module([(0, 0), (1, 1)])[0]) == 1
    assert n_clusters(run_module([(0, 0), (0, 2)])[0]) == 2
    assert n_clusters(run_module([(0, 0), (2, 0)])[0]) == 2


def test_late_merges():
    # U shape given arms first, bottom last; comb; spiral
    u = [(r, 10) for r in range(20)] + [(r, 14) for r in range(20)] + [(20, c) for c in range(10, 15)]
    assert n_clusters(run_module(u)[0]) == 1
    comb = [(r, c) for c in range(0, 60, 2) for r in range(30)] + [(30, c) for c in range(59)]
    assert n_clusters(run_module(comb)[0]) == 1
    img = np.zeros((160, 416), bool)
    r0, r1, c0, c1 = 10, 100, 10, 200
    while r1 - r0 > 4 and c1 - c0 > 4:                              # rectangular spiral, 1 px wide, 1 px gaps
        img[r0, c0:c1] = True; img[r0:r1, c1 - 1] = True; img[r1 - 1, c0 + 2:c1] = True; img[r0 + 2:r1, c0 + 2] = True
        img[r0 + 2, c0 + 2:c0 + 4] = True
        r0 += 4; c0 += 4; r1 -= 2; c1 -= 2
        r0 -= 2; c0 -= 2
    lab, k = ndimage.label(img, structure=np.ones((3, 3), int))
    assert n_clusters(run_module(img)[0]) == k


def test_adjacent_modules_do_not_merge():
    d = det()
    m = np.array([3, 3, 4, 4]); r = np.array([50, 51, 50, 51]); c = np.array([415, 415, 0, 0])
    w, fo, perm = d.stream(m, r, c, np.full(4, 255))
    o = oracle.process(d, w, fo, P)
    assert n_clusters(o) == 2 and sorted(o["c_n_pix"]) == [2, 2]


def test_cut_threshold_and_single_pixel_centroid():
    # charges at nominal-like gain are read back from the oracle itself; pick the cut relative to them
    o, rc = run_module([(10, 10), (10, 11), (50, 60)], adc=[60, 61, 90])
    q = o["charge"].astype(np.int64)
    pair, single = int(q[0] + q[1]), int(q[2])
    for cut, want in ((pair, {0, 1}), (pair + 1, set())):            # Q == cut keeps (S9)
        params = dict(P, cluster_charge_cut_e=cut, pixel_threshold_e=1)
        o2, _ = run_module([(10, 10), (10, 11), (50, 60)], adc=[60, 61, 90], params=params)
        kept = {i for i in range(2) if o2["status"][i] == 0}
        assert kept == want
        assert o2["status"][2] == (0 if single >= cut else 1)
    o3, _ = run_module([(50, 60)], adc=[200], params=dict(P, cluster_charge_cut_e=1))
    assert float(o3["c_x_col"][0]) == 60.0 and float(o3["c_y_row"][0]) == 50.0


def test_duplicates_first_index_wins():
    # (row,col) repeated: at distance 1, across the run, and a duplicate OF a below-threshold pixel
    rc = [(5, 5), (5, 5), (5, 6), (9, 9), (20, 20), (5, 6), (9, 9), (9, 10)]
    adc = [200, 10, 200, 10, 200, 250, 250, 200]                    # digi 3 is below threshold and owns (9,9)
    o, _ = run_module(rc, adc=adc)
    assert list(o["status"][[1, 5, 6]]) == [3, 3, 3]
    assert o["status"][3] == 2
    assert o["status"][7] in (0, 1)
    # the high-charge duplicate at (9,9) must NOT connect (9,10) to anything: (9,10) is alone
    assert o["clus"][6] == -1 and o["charge"][6] > 0
    s = dict(zip(oracle.SUMMARY, o["summary"]))
    assert s["n_duplicate"] == 3 and s["n_below_threshold"] == 1


@pytest.mark.parametrize("seed", range(12))
def test_against_bruteforce_chain(seed):
    rng = np.random.default_rng(100 + seed)
    d = det()
    n = int(rng.integers(1, 160))
    mods = np.sort(rng.integers(0, 3, n) + 7)                        # three modules, grouped
    # pixels in a small window so that touching, duplicates and merges are frequent
    r = rng.integers(40, 40 + 9, n); c = rng.integers(100, 100 + 12, n)
    adc = np.where(rng.random(n) < 0.25, rng.integers(1, 40, n), rng.integers(40, 256, n))
    w, fo, perm = d.stream(mods, r, c, adc)
    mods, r, c, adc = mods[perm], r[perm], c[perm], adc[perm]
    o = oracle.process(d, w, fo, P)
    gain = d.gain.reshape(-1, 416); ped = d.pedestal.reshape(-1, 416)
    b = brute_chain(list(mods), list(r), list(c), list(adc), lambda m, cc: gain[m, cc], lambda m, cc: ped[m, cc], P)
    assert list(o["charge"]) == b["charge"]
    assert list(o["status"]) == b["status"]
    assert list(o["clus"]) == b["clus"]
    cms = o["clus_module_start"]
    assert len(b["clusters"]) == int(o["summary"][13])
    for cl in b["clusters"]:
        g = int(cms[cl["module"]]) + cl["local"]
        assert int(o["c_module"][g]) == cl["module"] and int(o["c_first_digi"][g]) == cl["first_digi"]
        assert int(o["c_n_pix"][g]) == cl["n_pix"] and int(o["c_charge"][g]) == cl["charge"]
        assert o["c_x_col"][g] == cl["x"] and o["c_y_row"][g] == cl["y"]
