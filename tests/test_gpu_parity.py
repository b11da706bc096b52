"""Parity of the CUDA path (through the C ABI) against the oracle, element by element.  Needs a B200."""
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


def check(gu, det, batch, params=P, kmax=None, **kw):
    got = gu.run_batch(det, batch, params, kmax=kmax, **kw)
    exp = gu.oracle_events(det, batch, params, kmax=kmax)
    assert len(got) == len(exp)
    for e, (g, o) in enumerate(zip(got, exp)):
        gu.assert_event_equal(g, o, tag=f"event {e}")
    return got, exp


@pytest.mark.parametrize("mode", ["batch", "single", "host"])
def test_cfg0_tiny(gu, mode):
    det, b = pixgen.config("cfg0")
    check(gu, det, b, mode=mode)


@pytest.mark.parametrize("mode", ["batch", "single"])
def test_cfg1_pu50_event(gu, full, mode):
    b = pixgen.events(full, "pu50", [0])
    got, _ = check(gu, full, b, mode=mode)
    assert 55000 < int(got[0]["summary"][0]) < 66000


def test_cfg2_batch_ragged_chunks(gu, full):
    """24 PU50-like events in chunks of 5 (last chunk ragged): chunk boundaries fall inside vectors and tiles."""
    b = pixgen.events(full, "pu50", np.arange(24))
    check(gu, full, b, chunk_events=5)


def test_cfg2_one_chunk(gu, full):
    b = pixgen.events(full, "pu50", np.arange(100, 112))
    check(gu, full, b)


def test_cfg3_pu200(gu, full):
    b = pixgen.events(full, "pu200", np.arange(3))
    got, _ = check(gu, full, b, chunk_events=2)
    assert max(int(g["c_n_pix"].max()) for g in got) >= 50


def test_cfg4_edge_mix(gu, full):
    """5 events of each class: dense, duplicates, invalid words, edges, degenerate (empty, one word, all bad, ...)."""
    _, b = pixgen.config("cfg4", n_events=25)
    got, _ = check(gu, full, b, chunk_events=4)
    tally = b.tally.astype(np.int64)
    for e, g in enumerate(got):
        s = g["summary"].astype(np.int64)
        assert np.all(s[2:7] >= tally[e])  # injected invalid words are counted exactly (>=: degenerate events add their own)
    assert sum(int(g["summary"][7]) for g in got) > 1000     # duplicates seen
    assert any(int(g["summary"][0]) == 0 for g in got)        # an empty event


def test_cfg4_edge_mix_single_calls(gu, full):
    _, b = pixgen.config("cfg4", n_events=10)
    check(gu, full, b, mode="single")


def test_clamp_and_capacity(gu, full):
    b = pixgen.events(full, "pu50", [3, 4])
    check(gu, full, b, params=dict(P, max_clusters_per_module=8))
    got, _ = check(gu, full, b, kmax=1000)
    assert all(int(g["summary"][15]) & 2 for g in got)


def test_cfg2_full_size_sampled(gu, full):
    """BASELINE.json configs[2] at full size, in the launch configuration bench.py times (1000 events, one
    pix_process_batch call, library-default launch groups): 24 sampled events are compared element by element
    with the oracle; every event must satisfy the counting identities of the summary."""
    import torch
    import paper_2104_06573_b200 as pix
    E, kmax = 1000, 20480
    b = pixgen.events(full, "pu50", np.arange(E), cap_words_per_event=1 << 17)
    sizes = np.diff(b.event_offsets.astype(np.int64))
    W, M, F = int(sizes.sum()), full.n_modules, full.n_feds
    wmax = (int(sizes.max()) + 1023) // 1024 * 1024
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
        assert s[0] == sizes[e] and s[1] == s[0] - s[2:7].sum()
        assert s[1] == s[7] + s[8] + s[9] + s[10]                      # every decoded word has exactly one status
        assert s[14] == s[13] == g["clus_module_start"][-1] and s[15] == 0
        assert np.count_nonzero(g["clus"] >= 0) == s[9]
        assert int(g["c_n_pix"].sum()) == s[9]                         # pixels of surviving clusters = OK digis
    rng = np.random.default_rng(7)
    for e in sorted(set([0, E - 1]) | set(rng.choice(E, 22, replace=False).tolist())):
        o = gu.oracle_events(full, type(b)(b.words[int(b.event_offsets[e]):int(b.event_offsets[e + 1])],
                                           np.array([0, sizes[e]], np.uint32), b.fed_offsets[e:e + 1], b.tally[e:e + 1]),
                             P, kmax=kmax)[0]
        gu.assert_event_equal(got[e], o, tag=f"cfg2 full size, event {e}")


def test_deterministic_and_stream_independent(gu, full):
    """Two runs of the same batch (default stream, then a side stream) are bit-identical (several
    events in flight must give the same physics as one at a time)."""
    import torch
    b = pixgen.events(full, "pu50", np.arange(200, 216))
    a1 = gu.run_batch(full, b, P)
    st = torch.cuda.Stream()
    a2 = gu.run_batch(full, b, P, stream=st, chunk_events=7)
    for x, y in zip(a1, a2):
        for k in x:
            assert np.array_equal(x[k], y[k]), k


def test_cfg2_host_pipelined(gu, full):
    """pix_process_batch_host over several launch groups (input copy, kernels and output copy of consecutive groups
    overlap on three streams): 20 PU50-like events + an empty one, outputs poisoned first."""
    b = pixgen.events(full, ["pu50"] * 10 + ["empty"] + ["pu50"] * 10, np.arange(300, 321))
    check(gu, full, b, mode="host")


def _hand_batch(det, events):
    """events: list of (module, row, col, adc) arrays -> pixgen.Batch (modules emitted in the order given)."""
    words, ev_off, fed_off = [], [0], []
    for module, row, col, adc in events:
        w, fo, _ = det.stream(np.asarray(module), np.asarray(row), np.asarray(col), np.asarray(adc))
        words.append(w); ev_off.append(ev_off[-1] + len(w)); fed_off.append(fo)
    return pixgen.Batch(np.concatenate(words).astype(np.uint32), np.array(ev_off, np.uint32),
                        np.array(fed_off, np.uint32).reshape(len(events), det.n_feds + 1),
                        np.zeros((len(events), 5), np.uint32))


def test_run_lengths_across_kernel_tiers(gu, full):
    """Hand-built events: one long run of n words after a filler run of k words, for n around every size at which
    something changes for a run (a work item of the tile kernel holds at most 1024 words; runs of 256 words or more count
    their pixels differently; longer runs go to the block-per-run kernel, whose shared-memory tier ends at 2048 words)
    and k shifting the start inside the 128-word chunk.  Pixels form staircase lines, blobs and isolated pixels so
    that components span many rounds."""
    rng = np.random.default_rng(11)
    inv = full.inverse()
    fed_of = inv["fed"]
    mods = np.nonzero(fed_of == 0)[0][:2]  # two modules of FED 0: filler run, then the run under test
    events = []
    for n in (1, 31, 32, 33, 127, 128, 129, 130, 200, 255, 256, 257, 300, 511, 512, 513, 700, 1023, 1024, 1025, 1500):
        for k in (0, 1, 64, 127):
            pos = rng.choice(160 * 416, size=n, replace=False)          # scattered pixels ...
            line = (np.arange(n) % 160) * 416 + (np.arange(n) * 3 // 2) % 416
            sel = np.unique(np.where(rng.random(n) < 0.5, pos, line))    # ... mixed with staircase lines
            rng.shuffle(sel)
            sel = sel[:n]
            fr, fc = np.arange(k) % 160, (np.arange(k) * 7) % 416
            module = np.concatenate([np.full(k, mods[0]), np.full(len(sel), mods[1])])
            row = np.concatenate([fr, sel // 416]); col = np.concatenate([fc, sel % 416])
            adc = rng.integers(1, 256, size=len(module))
            events.append((module, row, col, adc))
    b = _hand_batch(full, events)
    check(gu, full, b, chunk_events=9)


def test_random_recipes(gu, full):
    """Seeded sweep over the generator's knobs (cluster count from nearly empty to PU200-dense, long-cluster share,
    read-out or shuffled word order, every edge class), ragged launch groups."""
    rng = np.random.default_rng(5)
    recipes = []
    for _ in range(36):
        recipes.append(dict(n_clusters=int(rng.choice([3, 50, 700, 5000, 15000, 30000, 45000])),
                            inner_modules=int(rng.choice([0, 16, 96])), inner_weight=int(rng.choice([1, 4, 16])),
                            long_permille=int(rng.choice([0, 0, 20, 150])), shuffle_order=int(rng.integers(0, 2)),
                            edge_class=int(rng.choice([0, 0, 0, 1, 2, 3, 4]))))
    b = pixgen.events(full, recipes, 9000 + np.arange(len(recipes)), cap_words_per_event=1 << 19)
    check(gu, full, b, chunk_events=int(rng.integers(3, 9)))


def test_prepass_chunk_and_pair_boundaries(gu, full):
    """The run-start pre-pass (runs.cu) works on 128-word chunks, two at a time when a pair lies inside one (event, FED)
    segment and holds decodable words only.  Events of many small sizes put event and FED boundaries at every
    alignment; all-zero words (EMPTY, transparent to runs) and words with an impossible double column are written at
    and next to chunk and pair boundaries, so that pairs, single chunks and the scan over undecodable words meet in
    every order.  One launch group and ragged ones."""
    rng = np.random.default_rng(77)
    recipes = [dict(n_clusters=int(rng.integers(3, 900)), inner_modules=int(rng.choice([0, 16])), inner_weight=4,
                    long_permille=int(rng.choice([0, 20])), shuffle_order=int(rng.integers(0, 2)), edge_class=0)
               for _ in range(48)]
    b = pixgen.events(full, recipes, 7700 + np.arange(len(recipes)))
    words = b.words.copy()
    n = len(words)
    for base in range(0, n - 600, 512 * int(rng.integers(1, 4))):
        for off in (0, 1, 126, 127, 128, 129, 255, 256, 257, 383, 384):
            if rng.random() < 0.35:
                g = base + off
                words[g] = 0 if rng.random() < 0.5 else (words[g] & ~np.uint32(31 << 16)) | np.uint32(int(rng.integers(26, 32)) << 16)
    b2 = pixgen.Batch(words, b.event_offsets, b.fed_offsets, b.tally)
    check(gu, full, b2)
    check(gu, full, b2, chunk_events=7)


def test_rechits_lite(gu, full):
    """pix_rechits (S25-S28) against the oracle's rechits on PU50, edge, duplicate, dense and PU200 events:
    boxes and flags bit-exact, local positions within 1e-5 relative (they inherit the centroid's tolerance)."""
    import oracle
    import torch
    import paper_2104_06573_b200 as pix
    b = pixgen.events(full, ["pu50", "edges", "dups", "pu200", "dense", "empty", "pu50"], 500 + np.arange(7),
                      cap_words_per_event=1 << 19)
    E, M, F = b.n_events, full.n_modules, full.n_feds
    sizes = np.diff(b.event_offsets.astype(np.int64))
    W, wmax = int(sizes.sum()), int(sizes.max())
    kmax = wmax
    h = pix.pix_create(full.cabling, F, M, full.gain, full.pedestal, pix.make_params(P, wmax, kmax, E, 3))
    try:
        words = torch.from_numpy(np.concatenate([b.words, np.zeros(16, np.uint32)]).view(np.int32)).cuda()
        ev_off = torch.from_numpy(b.event_offsets.view(np.int32).copy()).cuda()
        fed_off = torch.from_numpy(b.fed_offsets.view(np.int32).reshape(-1).copy()).cuda()
        digis, cl = pix.alloc_outputs(W, E, M, kmax, "cuda", fill=0xCD)
        hits = pix.alloc_hits(E, kmax, "cuda", fill=0xCD)
        pix.pix_process_batch(h, None, E, words, W, ev_off, fed_off, digis, cl)
        pix.pix_rechits(h, None, E, ev_off, digis, cl, hits)
        hn = gu.to_numpy(hits)
        summ = gu.to_numpy({"s": cl["summary"]})["s"].reshape(E, 16)
    finally:
        torch.cuda.synchronize()
        pix.pix_destroy(h)
    for e in range(E):
        o = oracle.process(full, *b.event(e), P, max_clusters_per_event=kmax)
        ho = oracle.rechits(full, o)
        k = int(summ[e, 14])
        assert k == len(ho["flags"])
        for name in ("min_row", "max_row", "min_col", "max_col", "flags"):
            assert np.array_equal(hn[name][e * kmax:e * kmax + k], ho[name]), (e, name)
        for name in ("x_local", "y_local"):
            np.testing.assert_allclose(hn[name][e * kmax:e * kmax + k], ho[name], rtol=1e-5, atol=2e-6, err_msg=f"{e} {name}")
        assert np.all(hn["flags"][e * kmax + k:(e + 1) * kmax] == 0xCD)  # untouched beyond n_clusters_emitted


def test_graph_replay_equals_direct_launch(gu, full):
    """pix_process never allocates, synchronises or copies to the host, so it can be captured into a CUDA graph
    (BASELINE.json configs[2]: one graph launch per event); two replays reproduce the direct launch bit by bit."""
    import torch
    import paper_2104_06573_b200 as pix
    b = pixgen.events(full, "pu50", [77])
    n, M, F = len(b.words), full.n_modules, full.n_feds
    h = gu.make_handle(full, P, n, n, 1, 1)
    try:
        words = torch.from_numpy(np.concatenate([b.words, np.zeros(16, np.uint32)]).view(np.int32)).cuda()
        fo = torch.from_numpy(b.fed_offsets.view(np.int32).reshape(-1).copy()).cuda()
        d0, c0 = pix.alloc_outputs(n, 1, M, n, "cuda", fill=0xCD)
        s = torch.cuda.Stream()
        pix.pix_process(h, s, words, fo, n, d0, c0)
        torch.cuda.synchronize()
        d1, c1 = pix.alloc_outputs(n, 1, M, n, "cuda", fill=0xCD)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            pix.pix_process(h, s, words, fo, n, d1, c1)
        for _ in range(2):
            for t in list(d1.values()) + list(c1.values()):
                t.view(torch.uint8).fill_(0xCD)
            torch.cuda.synchronize()
            with torch.cuda.stream(s):
                g.replay()
            torch.cuda.synchronize()
            k = int(c0["summary"][14])
            for name in d0:
                assert torch.equal(d0[name][:n], d1[name][:n]), name
            for name in ("module", "first_digi", "n_pix", "charge", "x_col", "y_row"):
                assert torch.equal(c0[name][:k], c1[name][:k]), name
            for name in ("module_first", "module_end", "clus_module_start", "summary"):
                assert torch.equal(c0[name], c1[name]), name
    finally:
        torch.cuda.synchronize()
        pix.pix_destroy(h)


def test_many_tiny_runs(gu, full):
    """Every module holds one to three pixels, so a 1024-word stretch has far more than 255 module runs: the packing
    of runs into work items has to cut shorter items (runs.cu, ITEM_RUNS).  Valid, contiguous events."""
    rng = np.random.default_rng(5)
    events = []
    for _ in range(3):
        module, row, col = [], [], []
        for m in range(full.n_modules):
            n = int(rng.integers(1, 4))
            r0, c0 = int(rng.integers(0, 158)), int(rng.integers(0, 414))
            cells = [(r0, c0), (r0 + 1, c0 + 1), (r0, c0 + 2)][:n]  # diagonal neighbours and a gap
            for r, c in cells:
                module.append(m); row.append(r); col.append(c)
        adc = rng.integers(1, 256, size=len(module))
        events.append((np.array(module), np.array(row), np.array(col), adc))
    check(gu, full, _hand_batch(full, events))


def _tile_bucket(run, row, col):
    """The tile kernel's position hash (tile.cu): key = run | row | col, h = (key << 7) * 0x9E3779B1 mod 2^32, bucket = top 11 bits."""
    key = (np.uint64(run) << np.uint64(17)) | (row.astype(np.uint64) << np.uint64(9)) | col.astype(np.uint64)
    return (((key << np.uint64(7)) * np.uint64(0x9E3779B1)) & np.uint64(0xFFFFFFFF)) >> np.uint64(21)


@pytest.mark.parametrize("n_same", [5, 8, 9, 24])
def test_hash_bucket_overflow(gu, full, n_same):
    """n_same pixels of one run that all fall into one bucket of the tile kernel's hash (4 entries per bucket, 4 more in
    the second level, beyond that the item goes to the block-per-run kernel), among ordinary pixels and next to a
    second run, with neighbours among the colliding pixels where the bucket has some."""
    rng = np.random.default_rng(17 + n_same)
    inv = full.inverse()
    mods = np.nonzero(inv["fed"] == 0)[0][:2]
    rr, cc = np.divmod(np.arange(160 * 416), 416)
    events = []
    for run in (0, 1):  # the colliding run is the item's first or second run
        bk = _tile_bucket(run, rr, cc)
        target = int(rng.integers(0, 2048))
        same = np.nonzero(bk == target)[0]
        assert len(same) >= n_same
        pick = same[:n_same]
        others = rng.choice(160 * 416, size=150, replace=False)
        near = np.unique(np.clip(np.concatenate([pick + 1, pick + 416, pick - 415]), 0, 160 * 416 - 1))  # neighbours of the colliding pixels
        sel = np.unique(np.concatenate([pick, others, near]))
        rng.shuffle(sel)
        filler = rng.choice(160 * 416, size=60, replace=False)
        if run == 0:
            module = np.concatenate([np.full(len(sel), mods[0]), np.full(len(filler), mods[1])]); pos = np.concatenate([sel, filler])
        else:
            module = np.concatenate([np.full(len(filler), mods[0]), np.full(len(sel), mods[1])]); pos = np.concatenate([filler, sel])
        events.append((module, pos // 416, pos % 416, rng.integers(1, 256, size=len(pos))))
    check(gu, full, _hand_batch(full, events))


def test_cluster_charge_beyond_32_bit_sums(gu, full):
    """One cluster whose charge makes the 32-bit weighted sums wrap (16 x 22 pixels at ADC 255) in a run short enough
    for the tile kernel, next to a run of 400 low-charge pixels in one cluster (more than 255 pixels: the packed
    pixel count does not apply) and an ordinary run: the first goes to the 64-bit block-per-run kernel."""
    rng = np.random.default_rng(23)
    inv = full.inverse()
    a, b, c = np.nonzero(inv["fed"] == 0)[0][:3]
    r1, c1 = np.divmod(np.arange(16 * 22), 22)
    r2, c2 = np.divmod(np.arange(400), 20)
    pos3 = rng.choice(160 * 416, size=100, replace=False)
    module = np.concatenate([np.full(len(r1), a), np.full(len(r2), b), np.full(len(pos3), c)])
    row = np.concatenate([r1 + 40, r2 + 10, pos3 // 416]); col = np.concatenate([c1 + 300, c2 + 100, pos3 % 416])
    adc = np.concatenate([np.full(len(r1), 255), np.full(len(r2), 45), rng.integers(1, 256, size=len(pos3))])
    got, exp = check(gu, full, _hand_batch(full, [(module, row, col, adc)]))
    assert int(exp[0]["c_n_pix"].max()) == 400 and int(exp[0]["c_charge"].max()) > 0xFFFFFFFF // 415
