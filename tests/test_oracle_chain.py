"""Whole-chain pins for the oracle: invariants, conservation, offsets (Fig. 3), metamorphic.  CPU only."""
import numpy as np
import pytest

import oracle
import pixgen
from helpers import P, check_invariants, partition


@pytest.fixture(scope="module")
def full():
    return pixgen.detector("full")


def test_invariants_cfg0():
    det, b = pixgen.config("cfg0")
    o = oracle.process(det, *b.event(0), P)
    check_invariants(o, P, det.n_modules)
    s = dict(zip(oracle.SUMMARY, (int(x) for x in o["summary"])))
    assert 9000 < s["n_words"] < 12000 and s["n_modules_present"] == 64
    assert s["n_below_threshold"] > 0 and s["n_cut_digis"] > 0      # both cuts are exercised (recipe G3)


@pytest.mark.parametrize("recipe,seed", [("pu50", 0), ("pu50", 7), ("pu200", 0), ("dense", 3), ("dups", 21),
                                         ("errors", 41), ("edges", 61), ("empty", 80), ("oneword", 81),
                                         ("allbad", 82), ("threemods", 83), ("fedempty", 84)])
def test_invariants_full_detector(full, recipe, seed):
    b = pixgen.events(full, recipe, [seed])
    o = oracle.process(full, *b.event(0), P)
    check_invariants(o, P, full.n_modules)
    s = dict(zip(oracle.SUMMARY, (int(x) for x in o["summary"])))
    assert s["flags"] == 0
    if recipe == "pu50":       # ~250 MB / 1000 events => ~62.5k words per event
        assert 55000 < s["n_words"] < 66000 and 13000 < s["n_clusters"] < 16500
    if recipe == "pu200":
        assert 230000 < s["n_words"] < 280000 and o["c_n_pix"].max() >= 50
    if recipe == "dups":
        assert s["n_duplicate"] > 1000
    if recipe == "dense":
        assert s["n_words"] > 100000
    if recipe == "empty":
        assert s["n_words"] == 0 and np.all(o["clus_module_start"] == 0)
    if recipe == "threemods":
        assert s["n_modules_present"] == 3


def test_offsets_clamp_is_fig3(full):
    """clus_module_start[m+1] - clus_module_start[m] == min(cap, n_clus[m]) and the digis keep true ids."""
    b = pixgen.events(full, "pu50", [3])
    w, fo = b.event(0)
    free = oracle.process(full, w, fo, P)
    n_clus = np.diff(free["clus_module_start"].astype(np.int64))
    assert n_clus.max() > 8
    capped = oracle.process(full, w, fo, dict(P, max_clusters_per_module=8))
    assert np.array_equal(np.diff(capped["clus_module_start"].astype(np.int64)), np.minimum(8, n_clus))
    assert int(capped["summary"][14]) == int(np.minimum(8, n_clus).sum())
    assert int(capped["summary"][13]) == int(n_clus.sum())          # n_clusters stays unclamped
    for k in ("module", "row", "col", "charge", "clus", "status"):
        assert np.array_equal(free[k], capped[k])
    # emitted records are the first min(cap, n) of every module, unchanged
    fs, cs = free["clus_module_start"].astype(np.int64), capped["clus_module_start"].astype(np.int64)
    for m in np.nonzero(n_clus)[0][:200]:
        k = cs[m + 1] - cs[m]
        for name in ("c_first_digi", "c_n_pix", "c_charge", "c_x_col", "c_y_row", "c_module"):
            assert np.array_equal(free[name][fs[m]:fs[m] + k], capped[name][cs[m]:cs[m + 1]])


def test_event_capacity_overflow_flag(full):
    b = pixgen.events(full, "pu50", [5])
    w, fo = b.event(0)
    free = oracle.process(full, w, fo, P)
    small = oracle.process(full, w, fo, P, max_clusters_per_event=1000)
    assert int(small["summary"][15]) & 2 and int(small["summary"][14]) == 1000
    assert np.array_equal(small["clus_module_start"], free["clus_module_start"])
    for name in ("c_first_digi", "c_charge"):
        assert np.array_equal(small[name], free[name][:1000])


def test_noncontiguous_flag_and_grouping():
    det = pixgen.detector("tiny")
    inv = det.inverse()
    same_fed = [m for m in range(det.n_modules) if inv["fed"][m] == inv["fed"][0]][:2]
    a, b_ = same_fed
    m = np.array([a, b_, a]); r = np.array([10, 10, 10]); c = np.array([10, 10, 11])
    w, fed = det.encode(m, r, c, np.full(3, 255))
    fo = np.zeros(det.n_feds + 1, np.uint32); fo[inv["fed"][0] + 1:] = 3
    o = oracle.process(det, w, fo, P)
    assert int(o["summary"][15]) & 1
    assert int(o["summary"][13]) == 2 and sorted(o["c_n_pix"]) == [1, 2]   # the oracle still groups by module id
    assert (int(o["module_first"][a]), int(o["module_end"][a])) == (0, 3)
    # interleaved undecodable words do not break a run
    w2 = np.array([w[0], 0, 0xFFFFFFFF, w[2]], np.uint32)
    fo2 = np.zeros(det.n_feds + 1, np.uint32); fo2[inv["fed"][0] + 1:] = 4
    o2 = oracle.process(det, w2, fo2, P)
    assert int(o2["summary"][15]) == 0 and int(o2["summary"][13]) == 1
    assert (int(o2["module_first"][a]), int(o2["module_end"][a])) == (0, 4)


def test_single_fed_without_offsets():
    det = pixgen.detector("tiny")
    one = pixgen.Detector(1, 32, 32, det.cabling[:64 * 32].copy(), det.gain, det.pedestal)
    mods = np.unique((one.cabling[one.cabling & 2 != 0] >> 2) & 0xFFFF)
    m = int(mods[0])
    w, fo, _ = det.stream(np.full(3, m), [1, 2, 50], [1, 2, 50], [255, 255, 255])
    a = oracle.process(det, w, fo, P)
    b = oracle.process(pixgen.Detector(1, 32, det.n_modules, det.cabling[:64 * 32].copy(), det.gain, det.pedestal), w, None, P)
    for k in ("module", "row", "col", "charge", "clus", "status"):
        assert np.array_equal(a[k], b[k])


def _pixel_partition(o):
    sets = partition(o["clus"], o["module"], o["status"])
    return {frozenset((int(o["module"][i]), int(o["row"][i]), int(o["col"][i]), int(o["charge"][i])) for i in s) for s in sets}


def test_metamorphic_permutations_and_recabling():
    det = pixgen.detector("tiny")
    b = pixgen.events(det, "tiny", [11])
    w, fo = b.event(0)
    base = oracle.process(det, w, fo, P)
    ref = _pixel_partition(base)
    rng = np.random.default_rng(5)
    # (1) permute words inside every module run
    w2 = w.copy()
    for m in range(det.n_modules):
        a, e = int(base["module_first"][m]), int(base["module_end"][m])
        w2[a:e] = w2[a:e][rng.permutation(e - a)]
    o2 = oracle.process(det, w2, fo, P)
    assert _pixel_partition(o2) == ref and int(o2["summary"][13]) == int(base["summary"][13])
    # (2) permute the module runs inside each FED
    parts = []
    for f in range(det.n_feds):
        runs = [(int(base["module_first"][m]), int(base["module_end"][m])) for m in range(det.n_modules)
                if base["module_end"][m] > 0 and fo[f] <= base["module_first"][m] < fo[f + 1]]
        for i in rng.permutation(len(runs)):
            parts.append(w[runs[i][0]:runs[i][1]])
    w3 = np.concatenate(parts)
    assert _pixel_partition(oracle.process(det, w3, fo, P)) == ref
    # (3) re-cabling: other cabling seed, same physical pixels
    det2 = pixgen.detector("tiny", cabling_seed=999)
    dec = base["status"] < 4
    mm, rr, cc = base["module"][dec], base["row"][dec], base["col"][dec]
    order = np.argsort(mm, kind="stable")
    w4, fo4, _ = det2.stream(mm[order], rr[order], cc[order], (w[dec] & 255)[order])
    assert _pixel_partition(oracle.process(det2, w4, fo4, P)) == ref
    # (4) one far-away pixel above the cut adds exactly one cluster
    free_mod = 0
    occupied = {(int(r), int(c)) for m_, r, c in zip(mm, rr, cc) if m_ == free_mod}
    spot = next((r, c) for r in range(3, 157) for c in range(3, 413)
                if all((r + dr, c + dc) not in occupied for dr in (-1, 0, 1) for dc in (-1, 0, 1)))
    a, e = int(base["module_first"][free_mod]), int(base["module_end"][free_mod])
    extra, _ = det.encode([free_mod], [spot[0]], [spot[1]], [255])
    w5 = np.concatenate([w[:e], extra, w[e:]])
    fo5 = fo.copy(); fo5[fo5 >= e] += 1
    if a == e == 0:
        pytest.skip("module 0 empty in this event")
    o5 = oracle.process(det, w5, fo5, P)
    assert int(o5["summary"][13]) == int(base["summary"][13]) + 1
