"""Pins of the oracle's legacy digi format and FED error list (pixo_legacy, readings S29-S31; SURVEY 8f
NEXT-4: "optional modules ... to convert the SoA to legacy data formats").  The paper gives no format
and no value, so the pins are: a packed word computed by hand, an independent numpy unpacking, the error list
recomputed with numpy from the (separately pinned) status array, the generator's injected-error tallies, the clamp."""
import numpy as np

import oracle
import pixgen
from helpers import P, hand_event


def raw_ids(det, seed=3):
    return (0x12000000 + np.random.default_rng(seed).permutation(det.n_modules).astype(np.uint32) * 4).astype(np.uint32)


def test_hand_computed_word():
    """module 3, row 5, col 7, adc 200: 5 + 7 * 2048 + 200 * 4194304 = 838875141 (written out by hand)."""
    det = pixgen.detector("tiny")
    w, fo, _ = hand_event(det, [3], [5], [7], [200])
    o = oracle.process(det, w, fo, P)
    rid = raw_ids(det)
    leg = oracle.legacy(det, w, fo, o, rid, 8)
    assert int(leg["pdigi"][0]) == 838875141
    assert int(leg["raw_id"][0]) == int(rid[3]) and int(leg["n_errors"][0]) == 0


def test_unpacks_to_the_digi_fields_and_padding_is_zero():
    det = pixgen.detector("full")
    b = pixgen.events(det, ["errors", "pu50", "dups"], [11, 12, 13])
    rid = raw_ids(det)
    for e in range(b.n_events):
        w, fo = b.event(e)
        o = oracle.process(det, w, fo, P)
        leg = oracle.legacy(det, w, fo, o, rid, len(w))
        dec = o["status"] <= 3
        assert np.array_equal(leg["pdigi"][dec] & 0x7FF, o["row"][dec])
        assert np.array_equal((leg["pdigi"][dec] >> 11) & 0x7FF, o["col"][dec])
        assert np.array_equal(leg["pdigi"][dec] >> 22, w[dec] & 255)          # bits 30-31 stay clear: adc < 256
        assert np.array_equal(leg["raw_id"][dec], rid[o["module"][dec]])
        assert np.all(leg["pdigi"][~dec] == 0) and np.all(leg["raw_id"][~dec] == 0)


def test_error_list_against_numpy_and_the_injected_tallies():
    det = pixgen.detector("full")
    b = pixgen.events(det, ["errors", "errors", "allbad", "pu50"], [21, 22, 23, 24])
    rid = raw_ids(det)
    for e in range(b.n_events):
        w, fo = b.event(e)
        o = oracle.process(det, w, fo, P)
        leg = oracle.legacy(det, w, fo, o, rid, len(w))
        idx = np.nonzero(o["status"] >= 5)[0]                                  # word order
        assert int(leg["n_errors"][0]) == len(idx)
        assert np.array_equal(leg["err_word"], w[idx]) and np.array_equal(leg["err_type"], o["status"][idx])
        assert np.array_equal(leg["err_fed"], np.searchsorted(fo, idx, side="right") - 1)
        assert np.all(leg["err_word"] != 0)                                    # padding words are not errors
        if e < 2:  # the generator's exact tally of injected words per class (link, roc, dcol, pxid)
            assert len(idx) == int(b.tally[e][1:5].sum())
            assert np.array_equal(np.bincount(leg["err_type"], minlength=9)[5:9], b.tally[e][1:5])


def test_capacity_clamp_keeps_the_true_count():
    det = pixgen.detector("full")
    b = pixgen.events(det, "errors", [31])
    w, fo = b.event(0)
    o = oracle.process(det, w, fo, P)
    full = oracle.legacy(det, w, fo, o, raw_ids(det), len(w))
    cut = oracle.legacy(det, w, fo, o, raw_ids(det), 10)
    n = int(full["n_errors"][0])
    assert n > 10 and int(cut["n_errors"][0]) == n and len(cut["err_word"]) == 10
    assert np.array_equal(cut["err_word"], full["err_word"][:10]) and np.array_equal(cut["err_fed"], full["err_fed"][:10])
