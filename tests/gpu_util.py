"""GPU-side test plumbing: run events through the C ABI (via the Python binding) and compare with the oracle."""
from __future__ import annotations

import numpy as np

import oracle
import paper_2104_06573_b200 as pix

DIGI_KEYS = ("module", "row", "col", "charge", "clus", "status")
REC_KEYS = (("c_module", "module"), ("c_first_digi", "first_digi"), ("c_n_pix", "n_pix"), ("c_charge", "charge"),
            ("c_x_col", "x_col"), ("c_y_row", "y_row"))


def make_handle(det, params, max_words_per_event, max_clusters_per_event, max_events_per_batch=1, chunk_events=0):
    p = pix.make_params(params, max_words_per_event, max_clusters_per_event, max_events_per_batch, chunk_events)
    return pix.pix_create(det.cabling, det.n_feds, det.n_modules, det.gain, det.pedestal, p)


def split_events(det, batch, digis, clusters, kmax):
    """Batch outputs (numpy) -> list of per-event dicts shaped like oracle.process()."""
    M = det.n_modules
    out = []
    for e in range(batch.n_events):
        a, b = int(batch.event_offsets[e]), int(batch.event_offsets[e + 1])
        o = {k: digis[k][a:b] for k in DIGI_KEYS}
        s = clusters["summary"][e * 16:(e + 1) * 16]
        k = int(s[14])
        for ok, gk in REC_KEYS:
            o[ok] = clusters[gk][e * kmax:e * kmax + k]
        o["module_first"] = clusters["module_first"][e * M:(e + 1) * M]
        o["module_end"] = clusters["module_end"][e * M:(e + 1) * M]
        o["clus_module_start"] = clusters["clus_module_start"][e * (M + 1):(e + 1) * (M + 1)]
        o["summary"] = s
        out.append(o)
    return out


def to_numpy(d):
    import torch
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in d.items()}


def run_batch(det, batch, params, kmax=None, mode="batch", chunk_events=0, poison=0xCD, handle=None, stream=None):
    """Runs a pixgen.Batch on the GPU.  mode: 'batch' (pix_process_batch), 'single' (pix_process per event on
    slices of the same buffers), 'host' (pix_process_batch_host).  Returns per-event dicts."""
    import torch
    E, M, F = batch.n_events, det.n_modules, det.n_feds
    n = len(batch.words)
    sizes = np.diff(batch.event_offsets.astype(np.int64))
    wmax = max(int(sizes.max(initial=1)), 1)
    kmax = int(kmax if kmax is not None else wmax)
    own = handle is None
    h = handle or make_handle(det, params, wmax, kmax, max(E, 1), chunk_events)
    try:
        if mode == "host":
            words = np.ascontiguousarray(batch.words)
            digis = {k: np.full(n + 16, poison, np.dtype(dt)) for k, dt in pix.DIGI_DTYPES.items()}
            cl = {k: np.full(max(E * kmax, 1), poison, np.dtype(dt)) for k, dt in pix.CLUSTER_DTYPES.items()}
            cl["module_first"] = np.full(E * M, poison, np.uint32); cl["module_end"] = np.full(E * M, poison, np.uint32)
            cl["clus_module_start"] = np.full(E * (M + 1), poison, np.uint32); cl["summary"] = np.full(E * 16, poison, np.uint32)
            pix.pix_process_batch_host(h, stream, E, words, n, np.ascontiguousarray(batch.event_offsets),
                                       np.ascontiguousarray(batch.fed_offsets) if F > 1 else None, digis, cl)
            return split_events(det, batch, digis, cl, kmax)
        dev = "cuda"
        words = torch.from_numpy(np.concatenate([batch.words, np.zeros(16, np.uint32)]).view(np.int32)).to(dev)
        ev_off = torch.from_numpy(batch.event_offsets.view(np.int32).copy()).to(dev)
        fed_off = torch.from_numpy(batch.fed_offsets.view(np.int32).reshape(-1).copy()).to(dev) if F > 1 else None
        digis, cl = pix.alloc_outputs(n, E, M, kmax, dev, fill=poison)
        if mode == "batch":
            pix.pix_process_batch(h, stream, E, words, n, ev_off, fed_off, digis, cl)
            return split_events(det, batch, to_numpy(digis), to_numpy(cl), kmax)
        assert mode == "single"
        outs = []
        for e in range(E):
            a, b = int(batch.event_offsets[e]), int(batch.event_offsets[e + 1])
            nw = b - a
            w_e = torch.empty(nw + 16, dtype=torch.int32, device=dev)  # fresh, aligned buffer per event
            w_e[:nw] = words[a:b]
            fo = fed_off[e * (F + 1):(e + 1) * (F + 1)].clone() if F > 1 else None
            d_e, c_e = pix.alloc_outputs(nw, 1, M, kmax, dev, fill=poison)
            pix.pix_process(h, stream, w_e, fo, nw, d_e, c_e)
            sub = type(batch)(batch.words[a:b], np.array([0, nw], np.uint32), batch.fed_offsets[e:e + 1], batch.tally[e:e + 1])
            outs.extend(split_events(det, sub, to_numpy(d_e), to_numpy(c_e), kmax))
        return outs
    finally:
        if own:
            import torch as _t
            _t.cuda.synchronize()
            pix.pix_destroy(h)


def oracle_events(det, batch, params, kmax=None):
    sizes = np.diff(batch.event_offsets.astype(np.int64))
    kmax = int(kmax if kmax is not None else max(int(sizes.max(initial=1)), 1))
    return [oracle.process(det, *batch.event(e), params, max_clusters_per_event=kmax) for e in range(batch.n_events)]


def assert_event_equal(g, o, tag=""):
    """Bit-exact on every integer array; centroids within 1e-5 relative (BASELINE.json north_star)."""
    for k in DIGI_KEYS + ("module_first", "module_end", "clus_module_start", "summary"):
        if not np.array_equal(g[k], o[k]):
            bad = np.nonzero(np.asarray(g[k]) != np.asarray(o[k]))[0]
            raise AssertionError(f"{tag} {k}: {len(bad)} mismatches, first at {bad[:5]}: gpu {np.asarray(g[k])[bad[:5]]} "
                                 f"oracle {np.asarray(o[k])[bad[:5]]}; summary gpu {g['summary']} oracle {o['summary']}")
    for k in ("c_module", "c_first_digi", "c_n_pix", "c_charge"):
        assert np.array_equal(g[k], o[k]), f"{tag} {k}"
    for k in ("c_x_col", "c_y_row"):
        assert g[k].shape == o[k].shape, f"{tag} {k} shape"
        np.testing.assert_allclose(g[k], o[k], rtol=1e-5, atol=0, err_msg=f"{tag} {k}")
