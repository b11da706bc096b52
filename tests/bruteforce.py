"""Brute-force statement of the path on PIXEL-level input, for tiny cases only.

Independent of oracle/ and of the CUDA path: pure Python/numpy, O(n^2) adjacency and repeated
min-label relaxation to a fix-point (no flood fill, no union-find).  Input is already decoded
(module,row,col,adc per digi, in stream order); decoding is pinned separately.  Follows DESIGN.md
readings S7 (calibration, numpy.float32 one op at a time), S9, S10 (first index wins), S13
(8-adjacency: max(|drow|,|dcol|) == 1, same module), S14 (ids by first digi index), S18.
"""
import numpy as np


def calibrate(adc, gain, ped, params):
    f = np.float32
    with np.errstate(all="ignore"):
        f1 = f(f(adc) - f(ped))
        f2 = f(f1 * f(gain))
        f3 = f(f2 * f(params["vcal_gain"]))
        f4 = f(f3 + f(params["vcal_offset"]))
    if not (f4 >= f(0)):
        return 0
    return int(min(f4, f(params["max_electrons"])))  # int() truncates toward zero


def chain(module, row, col, adc, gain_of, ped_of, params):
    """gain_of/ped_of: callables (module, col) -> float32.  Returns dict of per-digi lists + clusters."""
    n = len(module)
    charge = [calibrate(adc[i], gain_of(module[i], col[i]), ped_of(module[i], col[i]), params) for i in range(n)]
    status = [0] * n
    seen = {}
    for i in range(n):
        key = (module[i], row[i], col[i])
        if key in seen:
            status[i] = 3
        else:
            seen[key] = i
            if charge[i] < params["pixel_threshold_e"]:
                status[i] = 2
    live = [i for i in range(n) if status[i] == 0]
    label = {i: i for i in live}
    changed = True
    while changed:
        changed = False
        for a in live:
            for b in live:
                if module[a] == module[b] and max(abs(row[a] - row[b]), abs(col[a] - col[b])) == 1:
                    lo = min(label[a], label[b])
                    if label[a] != lo or label[b] != lo:
                        label[a] = label[b] = lo
                        changed = True
    clus = [-1] * n
    clusters = []
    next_id = {}
    for root in sorted(set(label.values())):
        mem = [i for i in live if label[i] == root]
        q = sum(charge[i] for i in mem)
        if q >= params["cluster_charge_cut_e"]:
            m = module[root]
            lid = next_id.get(m, 0)
            next_id[m] = lid + 1
            for i in mem:
                clus[i] = lid
            sx = sum(charge[i] * col[i] for i in mem)
            sy = sum(charge[i] * row[i] for i in mem)
            clusters.append(dict(module=m, local=lid, first_digi=root, n_pix=len(mem), charge=q,
                                 x=np.float32(sx / q), y=np.float32(sy / q)))
        else:
            for i in mem:
                status[i] = 1
    return dict(charge=charge, status=status, clus=clus, clusters=clusters)
