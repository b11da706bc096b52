"""pix_cluster_module_noalloc (include/pixclus.h): the entry point that allocates nothing, against the existing path.

Collected last on purpose (the file name): the suite runs with pytest -x, and a failure here must not hide another test.
Passes alone in a fresh process and after the other tests: it makes its own inputs and shares no state with them."""
import numpy as np
import pytest

import pixgen
from helpers import P

pytestmark = pytest.mark.gpu


def _module_event(det, rng, module, n_clusters, n_single, n_dup, n_empty):
    """One event whose only module holds random-walk clusters, single pixels (many below threshold), pixels that come
    twice (S10) and a few all-zero words (not pixels), in shuffled order."""
    cells = {}
    for _ in range(n_clusters):
        r, c = int(rng.integers(2, 157)), int(rng.integers(2, 413))
        for _ in range(int(rng.integers(2, 40))):
            cells[(r, c)] = int(rng.integers(40, 256))
            r = min(158, max(1, r + int(rng.integers(-1, 2)))); c = min(414, max(1, c + int(rng.integers(-1, 2))))
    for _ in range(n_single):
        cells[(int(rng.integers(0, 160)), int(rng.integers(0, 416)))] = int(rng.integers(1, 256))
    rc = np.array(list(cells.keys())); adc = np.array(list(cells.values()))
    again = rng.choice(len(rc), size=n_dup, replace=False)
    row = np.r_[rc[:, 0], rc[again, 0]]; col = np.r_[rc[:, 1], rc[again, 1]]; adc = np.r_[adc, rng.integers(1, 256, size=n_dup)]
    order = rng.permutation(len(row))
    w, fo, _ = det.stream(np.full(len(row), module), row[order], col[order], adc[order])
    w = w.copy()
    w[rng.choice(len(w), size=n_empty, replace=False)] = 0
    return pixgen.Batch(w.astype(np.uint32), np.array([0, len(w)], np.uint32), np.asarray(fo, np.uint32).reshape(1, -1),
                        np.zeros((1, 5), np.uint32))


def _compare(pix, torch, exp, tag):
    """exp: the existing path's per-event dict (gpu_util.run_batch).  Feeds its row / col / charge to the new entry point."""
    n = len(exp["row"])
    dev = torch.device("cuda", 0)
    k_exp = len(exp["c_first_digi"])
    kmax = k_exp + 7
    row = torch.from_numpy(exp["row"].astype(np.uint16).view(np.int16).copy()).to(dev)
    col = torch.from_numpy(exp["col"].astype(np.uint16).view(np.int16).copy()).to(dev)
    charge = torch.from_numpy(exp["charge"].astype(np.int32).copy()).to(dev)
    poison = lambda size, dt: torch.full((max(size, 1),), 0xCD, dtype=torch.uint8, device=dev).repeat_interleave(  # noqa: E731
        np.dtype(dt).itemsize).view(getattr(torch, dt))
    out = dict(clus=poison(n, "int32"), status=poison(n, "uint8"), first_digi=poison(kmax, "int32"), n_pix=poison(kmax, "int32"),
               charge=poison(kmax, "int32"), x_col=poison(kmax, "float32"), y_row=poison(kmax, "float32"), counts=poison(8, "int32"))
    pix.pix_cluster_module_noalloc(None, n, row, col, charge, int(P["pixel_threshold_e"]), int(P["cluster_charge_cut_e"]), kmax, out)
    torch.cuda.synchronize()
    got = {k: v.cpu().numpy() for k, v in out.items()}
    pixel = exp["row"] != 0xFFFF
    assert np.array_equal(got["clus"][:n], exp["clus"]), tag
    assert np.array_equal(got["status"][:n][pixel], exp["status"][pixel]), tag
    assert np.all(got["status"][:n][~pixel] == 0xCD), tag               # not pixels: status untouched
    s = exp["summary"].astype(np.int64)
    counts = got["counts"].astype(np.int64)
    assert list(counts) == [s[13], k_exp, s[12], s[7], s[8], s[9], s[10], 0], (tag, counts, s)
    assert np.array_equal(got["first_digi"][:k_exp].view(np.uint32), exp["c_first_digi"]), tag
    assert np.array_equal(got["n_pix"][:k_exp].view(np.uint32), exp["c_n_pix"]), tag
    assert np.array_equal(got["charge"][:k_exp].view(np.uint32), exp["c_charge"]), tag
    np.testing.assert_allclose(got["x_col"][:k_exp], exp["c_x_col"], rtol=1e-5, atol=0, err_msg=tag)  # the tests' centroid tolerance
    np.testing.assert_allclose(got["y_row"][:k_exp], exp["c_y_row"], rtol=1e-5, atol=0, err_msg=tag)
    assert np.all(got["first_digi"][k_exp:].view(np.uint32) == 0xCDCDCDCD), tag   # beyond the emitted records: untouched
    return k_exp


def test_noalloc_entry_point_matches_the_existing_path_twice():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import gpu_util
    import paper_2104_06573_b200 as pix
    det = pixgen.detector("full")
    rng = np.random.default_rng(20260)
    pix.pix_noalloc_setup()
    # two calls in a row on different inputs (the second smaller: what the first left in the scratch array must not show),
    # then the first again
    ev_a = _module_event(det, rng, 301, n_clusters=160, n_single=500, n_dup=40, n_empty=9)
    ev_b = _module_event(det, rng, 1700, n_clusters=25, n_single=60, n_dup=5, n_empty=3)
    exp_a = gpu_util.run_batch(det, ev_a, P)[0]
    exp_b = gpu_util.run_batch(det, ev_b, P)[0]
    assert len(exp_a["row"]) > 2048 > len(exp_b["row"]) > 200
    assert exp_a["summary"][7] >= 30 and exp_a["summary"][8] > 50 and exp_a["summary"][10] > 0  # DUPLICATE, BELOW, CUT all occur
    ka = _compare(pix, torch, exp_a, "first call")
    kb = _compare(pix, torch, exp_b, "second call")
    assert ka > 100 and kb > 10
    _compare(pix, torch, exp_a, "third call")


def test_noalloc_entry_point_rejects_what_does_not_fit():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2104_06573_b200 as pix
    n = pix.NOALLOC_MAX_DIGIS + 1
    dev = torch.device("cuda", 0)
    z16 = torch.zeros(n, dtype=torch.int16, device=dev); z32 = torch.zeros(n, dtype=torch.int32, device=dev)
    out = dict(clus=z32.clone(), status=torch.zeros(n, dtype=torch.uint8, device=dev), first_digi=z32.clone(), n_pix=z32.clone(),
               charge=z32.clone(), x_col=torch.zeros(n, device=dev), y_row=torch.zeros(n, device=dev), counts=z32[:8].clone())
    rc = pix.pix_cluster_module_noalloc(None, n, z16, z16, z32, 1000, 4000, 8, out, raise_on_error=False)
    assert rc == -2 and "PIX_NOALLOC_MAX_DIGIS" in pix.pix_noalloc_last_error()
    with pytest.raises(pix.PixError):
        pix.pix_cluster_module_noalloc(None, 16, None, z16, z32, 1000, 4000, 8, out)
    # the largest size that fits: every pixel of a 128 x 128 block is one cluster
    n = pix.NOALLOC_MAX_DIGIS
    idx = torch.arange(n, device=dev)
    row = (idx // 128).to(torch.int16); col = (idx % 128).to(torch.int16)
    charge = torch.full((n,), 2000, dtype=torch.int32, device=dev)
    pix.pix_cluster_module_noalloc(None, n, row, col, charge, 1000, 4000, 8, out)
    torch.cuda.synchronize()
    assert out["counts"].cpu().tolist() == [1, 1, 1, 0, 0, n, 0, 0]
    assert int(out["n_pix"][0]) == n and int(out["charge"][0]) == 2000 * n and int(out["first_digi"][0]) == 0
    assert abs(float(out["x_col"][0]) - 63.5) < 1e-3 and abs(float(out["y_row"][0]) - 63.5) < 1e-3
    assert bool((out["clus"][:n] == 0).all()) and bool((out["status"][:n] == 0).all())
