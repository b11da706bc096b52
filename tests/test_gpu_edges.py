"""Edge cases of the CUDA path through the C ABI: events that break the one-run-per-module contract (S11),
oversize events (PIX_FLAG_EVENT_TOO_LARGE), NULL outputs of the host entry point, long stretches of undecodable
words, and BASELINE.json configs[3] / configs[4] at their full batch sizes.  Needs a B200."""
import time

import numpy as np
import pytest

import pixgen
from helpers import P

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import gpu_util
    return gpu_util


@pytest.fixture(scope="module")
def full():
    return pixgen.detector("full")


def _batch(det, events):
    """events: list of (module, row, col, adc) -> pixgen.Batch; modules of one FED keep the order given."""
    words, ev_off, fed_off = [], [0], []
    for module, row, col, adc in events:
        w, fo, _ = det.stream(np.asarray(module), np.asarray(row), np.asarray(col), np.asarray(adc))
        words.append(w); ev_off.append(ev_off[-1] + len(w)); fed_off.append(fo)
    return pixgen.Batch(np.concatenate(words).astype(np.uint32), np.array(ev_off, np.uint32),
                        np.array(fed_off, np.uint32).reshape(len(events), det.n_feds + 1),
                        np.zeros((len(events), 5), np.uint32))


def _pixels(rng, n):
    pos = rng.choice(160 * 416, size=n, replace=False)
    return pos // 416, pos % 416, rng.integers(1, 256, size=n)


def _noncontiguous_events(det, rng):
    """Three ways to give a module more than one run (all inside FED 0, so the stream keeps the order)."""
    a, b, c = np.nonzero(det.inverse()["fed"] == 0)[0][:3]
    ev = []
    # A, B, A
    ra, ca, aa = _pixels(rng, 90)
    rb, cb, ab = _pixels(rng, 40)
    ev.append((np.r_[np.full(50, a), np.full(40, b), np.full(40, a)], np.r_[ra[:50], rb, ra[50:]],
               np.r_[ca[:50], cb, ca[50:]], np.r_[aa[:50], ab, aa[50:]]))
    # a run of 300 words, then B, then A again, then a valid module C
    ra, ca, aa = _pixels(rng, 420)
    rc, cc, ac = _pixels(rng, 70)
    ev.append((np.r_[np.full(300, a), np.full(40, b), np.full(120, a), np.full(70, c)], np.r_[ra[:300], rb, ra[300:], rc],
               np.r_[ca[:300], cb, ca[300:], cc], np.r_[aa[:300], ab, aa[300:], ac]))
    # A, B, A, B ... word by word: more runs in one 128-word chunk than a window can own
    ra, ca, aa = _pixels(rng, 400)
    rb2, cb2, ab2 = _pixels(rng, 400)
    m = np.empty(800, np.int64); m[0::2] = a; m[1::2] = b
    r = np.empty(800, np.int64); r[0::2] = ra; r[1::2] = rb2
    cc_ = np.empty(800, np.int64); cc_[0::2] = ca; cc_[1::2] = cb2
    ad = np.empty(800, np.int64); ad[0::2] = aa; ad[1::2] = ab2
    ev.append((m, r, cc_, ad))
    return ev


def _check_noncontiguous(g, o, tag):
    """What DESIGN.md S11 / pixclus.h define for a flagged event."""
    s = g["summary"].astype(np.int64)
    assert s[15] & 1 and int(o["summary"][15]) & 1, f"{tag}: flag"
    for k in ("module", "row", "col", "charge", "module_first", "module_end"):
        assert np.array_equal(g[k], o[k]), f"{tag} {k}"
    assert np.array_equal(s[:7], o["summary"].astype(np.int64)[:7]) and s[11] == int(o["summary"][11]), tag
    und = g["module"] == 0xFFFF
    assert np.array_equal(g["status"][und], o["status"][und]), f"{tag}: undecodable statuses"
    below = g["charge"] < P["pixel_threshold_e"]
    assert np.all(g["status"][~und & below] == 2) and np.all(g["status"][~und & ~below] == 1), f"{tag}: BELOW / CUT"
    assert np.all(g["clus"] == -1), tag
    assert s[7] == 0 and s[9] == 0 and s[12] == 0 and s[13] == 0 and s[14] == 0, tag
    assert s[8] == int((~und & below).sum()) and s[10] == int((~und & ~below).sum()) and s[1] == s[8] + s[10], tag
    assert np.all(g["clus_module_start"] == 0), tag


def test_noncontiguous_alone(gu, full):
    """S11: each flagged event alone (pix_process_batch with one event, and pix_process): flag on both sides, every
    output element written (the buffers are poisoned with 0xCD), counters as pixclus.h states."""
    rng = np.random.default_rng(21)
    for i, ev in enumerate(_noncontiguous_events(full, rng)):
        b = _batch(full, [ev])
        for mode in ("batch", "single"):
            got = gu.run_batch(full, b, P, mode=mode)
            exp = gu.oracle_events(full, b, P)
            _check_noncontiguous(got[0], exp[0], f"noncontiguous {i} {mode}")


def test_noncontiguous_inside_a_batch(gu, full):
    """Flagged events between valid ones in ONE launch group, among them a pathological one (two modules alternating
    word by word, 64k words: 32k runs per module): the valid neighbours stay bit-exact."""
    rng = np.random.default_rng(22)
    bad = _noncontiguous_events(full, rng)
    a, bm = np.nonzero(full.inverse()["fed"] == 0)[0][:2]
    n = 32768
    pa = rng.choice(160 * 416, size=n, replace=False); pb = rng.choice(160 * 416, size=n, replace=False)
    m = np.empty(2 * n, np.int64); m[0::2] = a; m[1::2] = bm
    pos = np.empty(2 * n, np.int64); pos[0::2] = pa; pos[1::2] = pb
    bad.append((m, pos // 416, pos % 416, rng.integers(1, 256, size=2 * n)))
    good = pixgen.events(full, "pu50", np.arange(700, 706))
    hand = _batch(full, bad)
    words, ev_off, fed_off, kinds = [], [0], [], []
    order = [("g", 0), ("b", 0), ("g", 1), ("b", 3), ("g", 2), ("b", 1), ("b", 2), ("g", 3), ("g", 4), ("g", 5)]
    for kind, i in order:
        src = good if kind == "g" else hand
        w, fo = src.event(i)
        words.append(w); ev_off.append(ev_off[-1] + len(w)); fed_off.append(fo); kinds.append(kind)
    b = pixgen.Batch(np.concatenate(words).astype(np.uint32), np.array(ev_off, np.uint32),
                     np.array(fed_off, np.uint32).reshape(len(order), full.n_feds + 1), np.zeros((len(order), 5), np.uint32))
    got = gu.run_batch(full, b, P)  # library-default launch groups: one group
    exp = gu.oracle_events(full, b, P)
    for e, (g, o) in enumerate(zip(got, exp)):
        if kinds[e] == "g":
            gu.assert_event_equal(g, o, tag=f"valid event {e} next to flagged ones")
        else:
            _check_noncontiguous(g, o, f"flagged event {e}")


def test_event_too_large(gu, full):
    """PIX_FLAG_EVENT_TOO_LARGE: an event longer than max_words_per_event that still fits its launch group is flagged
    and processed; events that respect the limit are untouched by it."""
    import paper_2104_06573_b200 as pix
    import torch
    big = dict(pixgen.RECIPES["pu50"], n_clusters=20000)  # about 80k words
    b = pixgen.events(full, ["pu50", big, "pu50", "empty", "pu50", "pu50", "pu50", "pu50", "pu50"], np.arange(40, 49),
                      cap_words_per_event=1 << 19)
    sizes = np.diff(b.event_offsets.astype(np.int64))
    E, M, F, n = b.n_events, full.n_modules, full.n_feds, len(b.words)
    wmax = 64000
    kmax = int(sizes.max())
    assert sizes[1] > wmax and np.delete(sizes, 1).max() <= wmax and sizes.sum() <= E * wmax  # the batch fits one launch group
    h = pix.pix_create(full.cabling, F, M, full.gain, full.pedestal, pix.make_params(P, wmax, kmax, E, 0))
    try:
        words = torch.from_numpy(np.concatenate([b.words, np.zeros(16, np.uint32)]).view(np.int32)).cuda()
        ev_off = torch.from_numpy(b.event_offsets.view(np.int32).copy()).cuda()
        fed_off = torch.from_numpy(b.fed_offsets.view(np.int32).reshape(-1).copy()).cuda()
        digis, cl = pix.alloc_outputs(n, E, M, kmax, "cuda", fill=0xCD)
        pix.pix_process_batch(h, None, E, words, n, ev_off, fed_off, digis, cl)
        got = gu.split_events(full, b, gu.to_numpy(digis), gu.to_numpy(cl), kmax)
    finally:
        torch.cuda.synchronize()
        pix.pix_destroy(h)
    exp = gu.oracle_events(full, b, P, kmax=kmax)
    for e, (g, o) in enumerate(zip(got, exp)):
        flags = int(g["summary"][15])
        assert bool(flags & 4) == (e == 1), (e, flags)
        g = dict(g); g["summary"] = g["summary"].copy(); g["summary"][15] &= ~np.uint32(4)
        gu.assert_event_equal(g, o, tag=f"too-large test, event {e}")


def test_host_entry_null_outputs(gu, full):
    """pix_process_batch_host skips NULL output arrays (clusters only: no digi array travels back) and copies no
    more records than the events emitted."""
    import paper_2104_06573_b200 as pix
    b = pixgen.events(full, ["pu50"] * 5 + ["empty"] + ["pu50"] * 4, np.arange(50, 60))
    sizes = np.diff(b.event_offsets.astype(np.int64))
    E, M, F, n = b.n_events, full.n_modules, full.n_feds, len(b.words)
    kmax = int(sizes.max())
    h = gu.make_handle(full, P, int(sizes.max()), kmax, E, 0)
    try:
        cl = {k: np.full(max(E * kmax, 1), 0xCD, np.dtype(dt)) for k, dt in pix.CLUSTER_DTYPES.items()}
        cl["module_first"] = np.full(E * M, 0xCD, np.uint32); cl["module_end"] = None
        cl["clus_module_start"] = np.full(E * (M + 1), 0xCD, np.uint32); cl["summary"] = np.full(E * 16, 0xCD, np.uint32)
        cl["x_col"] = None
        digis = {k: None for k in pix.DIGI_DTYPES}
        pix.pix_process_batch_host(h, None, E, np.ascontiguousarray(b.words), n, np.ascontiguousarray(b.event_offsets),
                                   np.ascontiguousarray(b.fed_offsets), digis, cl)
        moved = pix.pix_host_bytes_out(h)
    finally:
        import torch
        torch.cuda.synchronize()
        pix.pix_destroy(h)
    exp = gu.oracle_events(full, b, P, kmax=kmax)
    emitted = 0
    for e, o in enumerate(exp):
        k = int(o["summary"][14]); emitted += k
        assert np.array_equal(cl["summary"][e * 16:(e + 1) * 16], o["summary"])
        for name, key in (("module", "c_module"), ("first_digi", "c_first_digi"), ("n_pix", "c_n_pix"), ("charge", "c_charge")):
            assert np.array_equal(cl[name][e * kmax:e * kmax + k], o[key]), (e, name)
        np.testing.assert_allclose(cl["y_row"][e * kmax:e * kmax + k], o["c_y_row"], rtol=1e-5)
        assert np.array_equal(cl["module_first"][e * M:(e + 1) * M], o["module_first"])
        assert np.array_equal(cl["clus_module_start"][e * (M + 1):(e + 1) * (M + 1)], o["clus_module_start"])
    # 18 B per record row element (module 2, first 4, n_pix 4, charge 4, y 4) for at most max-per-group rows + per-event arrays
    assert moved < 18 * (emitted + E * 2000) + E * (2 * M + 1 + 16) * 4 and moved > 18 * emitted


def test_undecodable_stretch_is_linear(gu, full):
    """A batch that is almost all padding (zero words): the look-back for the previous decodable word stops at the
    start of the event, so the cost stays linear (it used to walk back to the start of the launch group)."""
    import paper_2104_06573_b200 as pix
    import torch
    E, nw = 64, 100_000
    w, fo = pixgen.events(full, "pu50", [1]).event(0)
    words = np.zeros(E * nw, np.uint32)
    fed_off = np.zeros((E, full.n_feds + 1), np.uint32)
    for e in range(E):
        fed_off[e, 1:] = nw                       # everything sits in FED 0's block
        if e % 8 == 0:
            words[e * nw + 5:e * nw + 5 + 200] = w[:200]  # a few real words near the start of some events
            fed_off[e] = np.minimum(fo, 205); fed_off[e, 0] = 0; fed_off[e, -1] = nw
            fed_off[e] = np.maximum.accumulate(fed_off[e])
    b = pixgen.Batch(words, (np.arange(E + 1) * nw).astype(np.uint32), fed_off, np.zeros((E, 5), np.uint32))
    t0 = time.perf_counter()
    got = gu.run_batch(full, b, P, kmax=4096)
    dt = time.perf_counter() - t0
    exp = gu.oracle_events(full, b, P, kmax=4096)
    for e in (0, 1, 8, 63):
        gu.assert_event_equal(got[e], exp[e], tag=f"padding batch, event {e}")
    assert all(int(g["summary"][2]) >= nw - 205 for g in got)
    assert dt < 20.0, dt


def test_two_cabling_entries_for_one_roc(gu, full):
    """A cabling table in which two (link, ROC) entries name the same ROC position of a module: the same pixel can then
    arrive twice in words that ascend in (link, roc, dcol, pxid) like ordinary read-out order.  The later word is a
    DUPLICATE (S10) all the same; the tile kernel's short cut for ordered words must be off for such a table."""
    import dataclasses
    inv = full.inverse()
    m = 700
    f, l = int(inv["fed"][m]), int(inv["link"][m])
    ent = full.cabling.reshape(full.n_feds, 64, 32).copy()
    r1 = int(inv["roc"][m, 3])                                  # the ROC at position 3 (rocy 0, rocx 3)
    r2 = int(np.nonzero((ent[f, l] & 2) == 0)[0][-1])           # an unused ROC number of the link, above the used ones
    assert r2 > int(inv["roc"][m].max())
    ent[f, l, r2] = ent[f, l, r1]
    det = dataclasses.replace(full, cabling=ent.reshape(-1), _inv={})
    rng = np.random.default_rng(31)
    rows = np.r_[10, 10, 11, 11, 40, 41, 60]; cols = np.r_[160, 161, 160, 161, 170, 170, 200]   # inside ROC position 3
    adc = rng.integers(60, 250, size=len(rows))
    w, _ = full.encode(np.full(len(rows), m), rows, cols, adc)
    again = (w[[1, 2, 4]] & ~np.uint32(31 << 21)) | np.uint32(r2 << 21)  # the same pixels through the second entry
    again = (again & ~np.uint32(255)) | np.uint32(200)
    other, _ = full.encode(np.full(3, m), np.r_[100, 100, 101], np.r_[20, 21, 21], np.r_[90, 90, 90])
    mine = np.sort(np.concatenate([w, again, other])).astype(np.uint32)
    assert np.all(np.diff(mine >> 8) > 0)                       # read-out order, every (link, roc, dcol, pxid) once
    # forty other modules around it, each in read-out order, so that the module sits in the middle of a work item made of
    # whole, clean 128-word chunks (the short cut is decided per chunk; the chunks at the ends of an event never take it)
    per_fed = [[] for _ in range(full.n_feds)]
    before, after = np.nonzero(inv["fed"] < f)[0], np.nonzero(inv["fed"] > f)[0]
    for mo in np.r_[rng.choice(before, size=20, replace=False), rng.choice(after, size=20, replace=False)]:
        r, c, a = _pixels(rng, 45)
        wo, _ = full.encode(np.full(45, mo), r, c, a)
        per_fed[int(inv["fed"][mo])].append((int(inv["link"][mo]), np.sort(wo)))
    per_fed[f].append((l, mine))
    chunks, fo = [], [0]
    for lst in per_fed:
        for _, wo in sorted(lst, key=lambda t: t[0]):
            chunks.append(wo)
        fo.append(sum(len(x) for x in chunks))
    words = np.concatenate(chunks).astype(np.uint32)
    at = int(np.nonzero(words == mine[0])[0][0])
    assert 256 <= at and at + len(mine) + 256 <= len(words)
    b = pixgen.Batch(words, np.array([0, len(words)], np.uint32), np.array(fo, np.uint32).reshape(1, -1), np.zeros((1, 5), np.uint32))
    got = gu.run_batch(det, b, P)
    exp = gu.oracle_events(det, b, P)
    gu.assert_event_equal(got[0], exp[0], tag="two entries for one ROC")
    assert int(exp[0]["summary"][7]) == 3                       # three DUPLICATE words


def _full_size(gu, full, b, n_sample, seed, tag):
    """One pix_process_batch call with library-default launch groups; identities on every event, n_sample events
    compared element by element with the oracle."""
    import paper_2104_06573_b200 as pix
    import torch
    sizes = np.diff(b.event_offsets.astype(np.int64))
    E, M, F, W = b.n_events, full.n_modules, full.n_feds, int(sizes.sum())
    wmax = (int(sizes.max()) + 1023) // 1024 * 1024
    kmax = max(int(sizes.max()) // 2, 4096)
    h = pix.pix_create(full.cabling, F, M, full.gain, full.pedestal, pix.make_params(P, wmax, kmax, E, 0))
    try:
        words = torch.from_numpy(np.concatenate([b.words, np.zeros(16, np.uint32)]).view(np.int32)).cuda()
        ev_off = torch.from_numpy(b.event_offsets.view(np.int32).copy()).cuda()
        fed_off = torch.from_numpy(b.fed_offsets.view(np.int32).reshape(-1).copy()).cuda()
        digis, cl = pix.alloc_outputs(W, E, M, kmax, "cuda", fill=0xCD)
        pix.pix_process_batch(h, None, E, words, W, ev_off, fed_off, digis, cl)
        got = gu.split_events(full, b, gu.to_numpy(digis), gu.to_numpy(cl), kmax)
    finally:
        torch.cuda.synchronize()
        pix.pix_destroy(h)
    for e, g in enumerate(got):
        s = g["summary"].astype(np.int64)
        assert s[0] == sizes[e] and s[1] == s[0] - s[2:7].sum(), (tag, e)
        assert s[1] == s[7] + s[8] + s[9] + s[10], (tag, e)
        assert s[14] == min(s[13], kmax) and g["clus_module_start"][-1] == s[13] and (s[15] & ~2) == 0, (tag, e)
        assert np.count_nonzero(g["clus"] >= 0) == s[9], (tag, e)
        if not s[15] & 2:
            assert int(g["c_n_pix"].sum()) == s[9], (tag, e)
    rng = np.random.default_rng(seed)
    for e in sorted(set([0, E - 1]) | set(rng.choice(E, n_sample - 2, replace=False).tolist())):
        sub = type(b)(b.words[int(b.event_offsets[e]):int(b.event_offsets[e + 1])], np.array([0, sizes[e]], np.uint32),
                      b.fed_offsets[e:e + 1], b.tally[e:e + 1])
        gu.assert_event_equal(got[e], gu.oracle_events(full, sub, P, kmax=kmax)[0], tag=f"{tag}, event {e}")


def test_cfg3_full_size_sampled(gu, full):
    """BASELINE.json configs[3] at its batch size: 200 PU200-like events (50.8 M words) in one call."""
    _full_size(gu, full, pixgen.events(full, "pu200", np.arange(200), cap_words_per_event=1 << 19), 8, 3, "cfg3 full size")


def test_cfg4_full_size_sampled(gu, full):
    """BASELINE.json configs[4] at its batch size: 100 edge-case events in one call."""
    _, b = pixgen.config("cfg4")
    _full_size(gu, full, b, 30, 4, "cfg4 full size")


def test_legacy_format(gu, full):
    """pix_legacy_format (S29-S31) against the oracle: packed digi words, raw detector ids, the error list in
    word order with its FED index and type, the true count beyond the list capacity; everything bit-exact."""
    import oracle
    import paper_2104_06573_b200 as pix
    import torch
    b = pixgen.events(full, ["pu50", "errors", "allbad", "empty", "dups", "errors", "oneword"], 600 + np.arange(7))
    sizes = np.diff(b.event_offsets.astype(np.int64))
    E, M, F, n = b.n_events, full.n_modules, full.n_feds, len(b.words)
    kmax, cap = int(sizes.max()), 1500  # the "allbad" event has more errors than the list holds
    rid = (0x12000000 + np.random.default_rng(3).permutation(M).astype(np.uint32) * 4).astype(np.uint32)
    h = gu.make_handle(full, P, int(sizes.max()), kmax, E, 3)
    try:
        words = torch.from_numpy(np.concatenate([b.words, np.zeros(16, np.uint32)]).view(np.int32)).cuda()
        ev_off = torch.from_numpy(b.event_offsets.view(np.int32).copy()).cuda()
        fed_off = torch.from_numpy(b.fed_offsets.view(np.int32).reshape(-1).copy()).cuda()
        digis, cl = pix.alloc_outputs(n, E, M, kmax, "cuda", fill=0xCD)
        leg = pix.alloc_legacy(n, E, cap, "cuda", fill=0xCD)
        rid_d = torch.from_numpy(rid.view(np.int32)).cuda()
        pix.pix_process_batch(h, None, E, words, n, ev_off, fed_off, digis, cl)
        pix.pix_legacy_format(h, None, E, words, n, ev_off, fed_off, digis, rid_d, cap, leg)
        got = gu.to_numpy(leg)
    finally:
        torch.cuda.synchronize()
        pix.pix_destroy(h)
    clipped = 0
    for e in range(E):
        w, fo = b.event(e)
        o = oracle.process(full, w, fo, P, max_clusters_per_event=kmax)
        lo = oracle.legacy(full, w, fo, o, rid, cap)
        a, z = int(b.event_offsets[e]), int(b.event_offsets[e + 1])
        assert np.array_equal(got["pdigi"][a:z], lo["pdigi"]) and np.array_equal(got["raw_id"][a:z], lo["raw_id"]), e
        ne = int(lo["n_errors"][0]); k = min(ne, cap); clipped += ne > cap
        assert int(got["n_errors"][e]) == ne, e
        for name in ("err_word", "err_fed", "err_type"):
            assert np.array_equal(got[name][e * cap:e * cap + k], lo[name]), (e, name)
        assert np.all(got["err_type"][e * cap + k:(e + 1) * cap] == 0xCD)  # untouched beyond the count
    assert clipped >= 1


def test_guard_bands_and_repeatability(gu, full):
    """compute-sanitizer is closed on this pool, so bounds and races are checked by hand: every output array sits
    between two poisoned guard bands that must stay untouched, and twelve runs of a batch that exercises every kernel
    (PU200 runs for the block kernels, dense modules, duplicates, invalid words, a flagged event) on alternating
    streams and launch-group sizes must be bit-identical -- a lost update or a read of an unfinished neighbour
    shows up as a run that differs."""
    import paper_2104_06573_b200 as pix
    import torch
    b = pixgen.events(full, ["pu50", "dense", "dups", "errors", "pu200", "edges", "empty", "pu50"], 800 + np.arange(8),
                      cap_words_per_event=1 << 19)
    sizes = np.diff(b.event_offsets.astype(np.int64))
    E, M, F, n = b.n_events, full.n_modules, full.n_feds, len(b.words)
    kmax, G = int(sizes.max()), 4096
    words = torch.from_numpy(np.concatenate([b.words, np.zeros(16, np.uint32)]).view(np.int32)).cuda()
    ev_off = torch.from_numpy(b.event_offsets.view(np.int32).copy()).cuda()
    fed_off = torch.from_numpy(b.fed_offsets.view(np.int32).reshape(-1).copy()).cuda()
    sizes_of = dict(module=n, row=n, col=n, charge=n, clus=n, status=n)
    csz = {k: E * kmax for k in pix.CLUSTER_DTYPES}
    csz.update(module_first=E * M, module_end=E * M, clus_module_start=E * (M + 1), summary=E * 16)
    dts = dict(pix.DIGI_DTYPES); cdt = dict(pix.CLUSTER_DTYPES); cdt.update(pix.PER_EVENT)

    def guarded(size, dt):
        t = torch.empty(size + 2 * G, dtype=getattr(torch, dt), device="cuda")
        t.view(torch.uint8).fill_(0xCD)
        return t

    ref = None
    streams = [None, torch.cuda.Stream(), torch.cuda.Stream()]
    for it in range(12):
        h = gu.make_handle(full, P, int(sizes.max()), kmax, E, (0, 3, 5)[it % 3])
        try:
            raw_d = {k: guarded(v, dts[k]) for k, v in sizes_of.items()}
            raw_c = {k: guarded(v, cdt[k]) for k, v in csz.items()}
            d = {k: v[G:G + sizes_of[k]] for k, v in raw_d.items()}
            c = {k: v[G:G + csz[k]] for k, v in raw_c.items()}
            pix.pix_process_batch(h, streams[it % 3], E, words, n, ev_off, fed_off, d, c)
            torch.cuda.synchronize()
            for k, v, size in [(k, v, sizes_of[k]) for k, v in raw_d.items()] + [(k, v, csz[k]) for k, v in raw_c.items()]:
                u = v.view(torch.uint8); es = v.element_size()
                assert bool((u[:G * es] == 0xCD).all()) and bool((u[(G + size) * es:] == 0xCD).all()), f"guard band of {k} touched"
            out = gu.split_events(full, b, {k: v.cpu().numpy() for k, v in d.items()}, {k: v.cpu().numpy() for k, v in c.items()}, kmax)
        finally:
            torch.cuda.synchronize()
            pix.pix_destroy(h)
        if ref is None:
            ref = out
            for e, (g, o) in enumerate(zip(out, gu.oracle_events(full, b, P, kmax=kmax))):
                gu.assert_event_equal(g, o, tag=f"guarded run, event {e}")
        else:
            for e, (x, y) in enumerate(zip(ref, out)):
                for k in x:
                    assert np.array_equal(x[k], y[k]), (it, e, k)
