"""Pins for oracle O1 (decode) -- DESIGN.md readings S1-S6.  CPU only."""
import numpy as np
import pytest

import oracle
import pixgen
from helpers import P

ST = oracle.STATUS


def entry(module, rocx, rocy, flip_r=0, flip_c=0, roc_valid=1):
    # S3 bit layout of a cabling entry (interface definition, include/pixclus.h)
    return 1 | (roc_valid << 1) | (module << 2) | (rocx << 18) | (rocy << 21) | (flip_r << 22) | (flip_c << 23)


def word(link, roc, dcol, pxid, adc):
    return (link << 26) | (roc << 21) | (dcol << 16) | (pxid << 8) | adc


@pytest.fixture(scope="module")
def hand_cabling():
    cab = np.zeros(2 * 64 * 32, np.uint32)            # F = 2
    base = (0 * 64 + 5) * 32
    cab[base:base + 32] = entry(1, 0, 0, roc_valid=0)  # link 5 of FED 0 mapped, rocs invalid unless set below
    cab[base + 3] = entry(1, 2, 1)
    cab[base + 4] = entry(1, 7, 0, flip_r=1, flip_c=1)
    base = (1 * 64 + 63) * 32
    cab[base:base + 32] = entry(0, 0, 0, roc_valid=0)
    cab[base + 15] = entry(0, 0, 0)
    return cab


def test_hand_computed_positions(hand_cabling):
    # link 5 roc 3 -> module 1, ROC at (rocx 2, rocy 1), no flips.  dcol 4, pxid 9: ROC-local row 9>>1 = 4,
    # ROC-local col 2*4 + (9&1) = 9  ->  row 80 + 4 = 84, col 2*52 + 9 = 113.
    assert oracle.decode_word(word(5, 3, 4, 9, 77), 0, hand_cabling) == (ST["OK"], 1, 84, 113, 77)
    # flipped ROC at (rocx 7, rocy 0): dcol 25 pxid 159 -> local (79, 51) -> flipped (0, 0) -> row 0, col 364
    assert oracle.decode_word(word(5, 4, 25, 159, 1), 0, hand_cabling) == (ST["OK"], 1, 0, 364, 1)
    # dcol 0 pxid 0 -> local (0,0) -> flipped (79, 51) -> row 79, col 7*52 + 51 = 415
    assert oracle.decode_word(word(5, 4, 0, 0, 255), 0, hand_cabling) == (ST["OK"], 1, 79, 415, 255)
    # same word in FED 1 uses FED 1's table: link 63 roc 15 -> module 0 at the origin
    assert oracle.decode_word(word(63, 15, 1, 2, 9), 1, hand_cabling) == (ST["OK"], 0, 1, 2, 9)


def test_error_classes_and_precedence(hand_cabling):
    d = lambda w, fed=0: oracle.decode_word(w, fed, hand_cabling)[0]
    assert d(0) == ST["EMPTY"]
    assert d(word(6, 3, 4, 9, 77)) == ST["ERR_LINK"]                  # unmapped link
    assert d(word(5, 3, 4, 9, 77), fed=1) == ST["ERR_LINK"]           # mapped in FED 0 only
    assert d(word(5, 7, 4, 9, 77)) == ST["ERR_ROC"]                   # roc id unused on a mapped link
    assert d(word(5, 20, 4, 9, 77)) == ST["ERR_ROC"]                  # roc >= 16
    assert d(word(5, 3, 26, 9, 77)) == ST["ERR_DCOL"]
    assert d(word(5, 3, 25, 9, 77)) == ST["OK"]
    assert d(word(5, 3, 4, 160, 77)) == ST["ERR_PXID"]
    assert d(word(5, 3, 4, 159, 77)) == ST["OK"]
    # first failing check wins: link > roc > dcol > pxid
    assert d(word(6, 31, 31, 255, 0)) == ST["ERR_LINK"]
    assert d(word(5, 31, 31, 255, 0)) == ST["ERR_ROC"]
    assert d(word(5, 3, 31, 255, 0)) == ST["ERR_DCOL"]
    # adc 0 with a valid address is a valid word (only the all-zero word is padding)
    assert d(word(5, 3, 0, 0, 0)) == ST["OK"]


def test_address_bijection_full_detector():
    """For a fixed module the 16*26*160 = 66 560 valid addresses hit every (row, col) exactly once."""
    det = pixgen.detector("full")
    inv = det.inverse()
    roc, dcol, pxid = np.meshgrid(np.arange(16), np.arange(26), np.arange(160), indexing="ij")
    for m in (0, 95, 1855):
        link, fed = int(inv["link"][m]), int(inv["fed"][m])
        w = ((link << 26) | (roc.ravel() << 21) | (dcol.ravel() << 16) | (pxid.ravel() << 8) | 200).astype(np.uint32)
        fo = np.zeros(det.n_feds + 1, np.uint32); fo[fed + 1:] = len(w)
        o = oracle.process(det, w, fo, P)
        assert np.all(o["status"] == 0) and np.all(o["module"] == m)
        hit = np.zeros((160, 416), np.int64)
        np.add.at(hit, (o["row"], o["col"]), 1)
        assert np.all(hit == 1)
        assert int(o["summary"][13]) == 1 and int(o["c_n_pix"][0]) == 66560    # full module -> one cluster


def test_round_trip_against_generator_encoder():
    """pixgen's encoder is written in the inverse direction, independently of the oracle."""
    det = pixgen.detector("full")
    rng = np.random.default_rng(1)
    n = 20000
    m = np.sort(rng.integers(0, det.n_modules, n))
    r, c, a = rng.integers(0, 160, n), rng.integers(0, 416, n), rng.integers(1, 256, n)
    w, fo, perm = det.stream(m, r, c, a)
    o = oracle.process(det, w, fo, P)
    assert np.all(o["status"] != 4) and np.all(o["status"] < 5)
    assert np.array_equal(o["module"], m[perm]) and np.array_equal(o["row"], r[perm]) and np.array_equal(o["col"], c[perm])


def test_exhaustive_one_fed_closed_form():
    """All 2^24 address patterns of one FED (adc = 255): error counts and clusters in closed form."""
    det = pixgen.detector("full")
    L = det.links_per_fed
    w = ((np.arange(1 << 24, dtype=np.uint64) << 8) | 255).astype(np.uint32)
    fo = np.zeros(det.n_feds + 1, np.uint32); fo[4:] = len(w)     # everything sits in FED 3
    o = oracle.process(det, w, fo, P, max_clusters_per_event=4096)
    s = dict(zip(oracle.SUMMARY, (int(x) for x in o["summary"])))
    assert s["n_words"] == 1 << 24 and s["n_empty"] == 0
    assert s["n_err_link"] == (64 - L) * 32 * 32 * 256
    assert s["n_err_roc"] == L * 16 * 32 * 256
    assert s["n_err_dcol"] == L * 16 * 6 * 256
    assert s["n_err_pxid"] == L * 16 * 26 * 96
    assert s["n_decoded"] == L * 66560 and s["n_duplicate"] == 0
    assert s["n_modules_present"] == L and s["n_clusters"] == L and s["flags"] == 0
    assert np.all(o["c_n_pix"] == 66560)


def test_generator_error_tallies():
    """cfg4 (c): the generator injects words that are invalid by construction and tallies them."""
    det = pixgen.detector("full")
    b = pixgen.events(det, ["errors", "errors", "allbad"], [40, 41, 82])
    for e in range(3):
        w, fo = b.event(e)
        o = oracle.process(det, w, fo, P)
        assert list(o["summary"][2:7]) == list(b.tally[e]), e
    assert int(oracle.process(det, *b.event(2), P)["summary"][1]) == 0
