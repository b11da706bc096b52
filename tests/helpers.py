"""Shared test plumbing: hand-built events and structural checks (no method arithmetic)."""
import numpy as np

import pixgen

P = dict(pixgen.DEFAULT_PARAMS)


def hand_event(det, module, row, col, adc):
    """Pixels (in the order given, which must keep each module's pixels together) -> words, fed_offsets,
    perm (stream position -> input index).  Modules are emitted in FED order, so the caller's
    relative order is kept inside a FED."""
    module, row, col, adc = (np.asarray(x, np.int64) for x in (module, row, col, adc))
    return det.stream(module, row, col, adc)


def partition(clus, module, status):
    """set of frozensets of digi indices, one per surviving cluster."""
    groups = {}
    for i, (c, m, s) in enumerate(zip(clus, module, status)):
        if s == 0:
            groups.setdefault((int(m), int(c)), []).append(i)
    return {frozenset(v) for v in groups.values()}


def check_invariants(o, params, n_modules):
    """Structural invariants of one event's output (DESIGN.md section 3 'whole chain' pins)."""
    mod, row, col, chg, clus, st = (o[k] for k in ("module", "row", "col", "charge", "clus", "status"))
    s = o["summary"].astype(np.int64)
    n = len(mod)
    assert s[0] == n
    assert s[0] == s[1] + s[2] + s[3] + s[4] + s[5] + s[6]
    assert s[1] == s[7] + s[8] + s[9] + s[10]
    for code, idx in ((4, 2), (5, 3), (6, 4), (7, 5), (8, 6), (3, 7), (2, 8), (0, 9), (1, 10)):
        assert int((st == code).sum()) == s[idx], (code, idx)
    assert np.all((clus >= 0) == (st == 0))
    und = st >= 4
    assert np.all(mod[und] == 0xFFFF) and np.all(row[und] == 0xFFFF) and np.all(col[und] == 0xFFFF)
    assert np.all(chg[und] == 0)
    assert np.all(row[~und] < 160) and np.all(col[~und] < 416) and np.all(mod[~und] < n_modules)
    ok = st == 0
    assert np.all(chg[ok] >= params["pixel_threshold_e"])
    assert np.all(chg[st == 2] < params["pixel_threshold_e"])
    # cluster records vs digis
    cms = o["clus_module_start"].astype(np.int64)
    assert cms[0] == 0 and np.all(np.diff(cms) >= 0)
    k = int(s[14])
    assert k == min(cms[-1], len(o["c_module"])) or k == cms[-1]
    if params.get("max_clusters_per_module", 0xFFFFFFFF) == 0xFFFFFFFF and not (s[15] & 2):
        assert cms[-1] == s[13]
        gid = cms[mod[ok].astype(np.int64)] + clus[ok]
        assert gid.max(initial=-1) < k
        q = np.bincount(gid, weights=chg[ok].astype(np.float64), minlength=k).astype(np.int64)
        npx = np.bincount(gid, minlength=k)
        assert np.array_equal(q, o["c_charge"].astype(np.int64))          # charge conservation, exact
        assert np.array_equal(npx, o["c_n_pix"].astype(np.int64))
        assert int(o["c_charge"].astype(np.int64).sum()) == int(chg[ok].astype(np.int64).sum())
        assert np.all(o["c_charge"].astype(np.int64) >= params["cluster_charge_cut_e"])
        first = np.full(k, n, np.int64)
        np.minimum.at(first, gid, np.nonzero(ok)[0])
        assert np.array_equal(first, o["c_first_digi"].astype(np.int64))   # first_digi = min member index
        assert np.array_equal(o["c_module"].astype(np.int64), mod[o["c_first_digi"]].astype(np.int64))
        for m in np.unique(o["c_module"]):
            f = o["c_first_digi"][cms[m]:cms[m + 1]].astype(np.int64)
            assert np.all(np.diff(f) > 0)                                   # ids ordered by first digi index
        # centroid inside the bounding box
        for arr, cen in ((col, "c_x_col"), (row, "c_y_row")):
            lo = np.full(k, 1 << 30, np.int64); hi = np.full(k, -1, np.int64)
            np.minimum.at(lo, gid, arr[ok].astype(np.int64)); np.maximum.at(hi, gid, arr[ok].astype(np.int64))
            assert np.all(o[cen] >= lo - 1e-3) and np.all(o[cen] <= hi + 1e-3)
    # no two distinct components (surviving or cut) 8-adjacent; duplicates own nothing
    live = np.nonzero((st == 0) | (st == 1))[0]
    key = {}
    for i in live:
        key[(int(mod[i]), int(row[i]), int(col[i]))] = i
    assert len(key) == len(live)
    for (m, r, c), i in key.items():
        for dr in (-1, 0, 1):
            for dc in (-1, 0, 1):
                j = key.get((m, r + dr, c + dc))
                if j is None or j == i:
                    continue
                assert st[i] == st[j] and clus[i] == clus[j], (i, j)
    # module ranges
    dec = np.nonzero(~und)[0]
    mf, me = o["module_first"].astype(np.int64), o["module_end"].astype(np.int64)
    exp_f = np.zeros(n_modules, np.int64); exp_e = np.zeros(n_modules, np.int64)
    if len(dec):
        first_seen = np.full(n_modules, n, np.int64)
        np.minimum.at(first_seen, mod[dec].astype(np.int64), dec)
        last_seen = np.full(n_modules, -1, np.int64)
        np.maximum.at(last_seen, mod[dec].astype(np.int64), dec)
        present = last_seen >= 0
        exp_f[present] = first_seen[present]; exp_e[present] = last_seen[present] + 1
        assert s[11] == present.sum()
    else:
        assert s[11] == 0
    assert np.array_equal(mf, exp_f) and np.array_equal(me, exp_e)
