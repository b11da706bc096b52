"""paper_2104_06573_b200 -- thin Python binding of libpixclus.so (include/pixclus.h).

Argument marshalling only: every step of the path (unpack, calibrate, cluster per module;
Fig. 3 offsets) runs in the CUDA kernels behind the C ABI.  There is no CPU fallback: if the library is
missing or does not load, importing the binding's functions raises.  torch is used for device memory and
streams only.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpixclus.so")

PIX_OK, PIX_ERR_INVALID_ARG, PIX_ERR_CAPACITY, PIX_ERR_CUDA, PIX_ERR_ALLOC = 0, -1, -2, -3, -4
ROWS, COLS = 160, 416
STATUS = dict(OK=0, CUT=1, BELOW_THRESHOLD=2, DUPLICATE=3, EMPTY=4, ERR_LINK=5, ERR_ROC=6, ERR_DCOL=7, ERR_PXID=8)
SUMMARY = ("n_words", "n_decoded", "n_empty", "n_err_link", "n_err_roc", "n_err_dcol", "n_err_pxid", "n_duplicate",
           "n_below_threshold", "n_ok_digis", "n_cut_digis", "n_modules_present", "n_clusters_precut", "n_clusters",
           "n_clusters_emitted", "flags")
FLAG_NONCONTIGUOUS, FLAG_CLUSTER_CAPACITY_OVERFLOW, FLAG_EVENT_TOO_LARGE = 1, 2, 4
EXPORTS = ("pix_create", "pix_clone", "pix_destroy", "pix_process", "pix_process_batch", "pix_process_batch_host",
           "pix_rechits", "pix_kernel_launches", "pix_last_error", "pix_set_profiling", "pix_read_profile",
           "pix_overflow_runs", "pix_host_bytes_out", "pix_legacy_format", "pix_noalloc_setup",
           "pix_cluster_module_noalloc", "pix_noalloc_last_error")
NOALLOC_MAX_DIGIS = 16384  # PIX_NOALLOC_MAX_DIGIS of include/pixclus.h

_vp, _u32 = ctypes.c_void_p, ctypes.c_uint32


class CablingMap(ctypes.Structure):
    _fields_ = [("n_feds", _u32), ("n_modules", _u32), ("entry", _vp)]


class GainTable(ctypes.Structure):
    _fields_ = [("n_modules", _u32), ("gain", _vp), ("pedestal", _vp)]


class Params(ctypes.Structure):
    _fields_ = [("vcal_gain", ctypes.c_float), ("vcal_offset", ctypes.c_float), ("pixel_threshold_e", ctypes.c_int32),
                ("cluster_charge_cut_e", ctypes.c_int32), ("max_electrons", ctypes.c_int32),
                ("max_clusters_per_module", _u32), ("max_words_per_event", _u32), ("max_clusters_per_event", _u32),
                ("max_events_per_batch", _u32), ("chunk_events", _u32)]


class Digis(ctypes.Structure):
    _fields_ = [(n, _vp) for n in ("module", "row", "col", "charge", "clus", "status")]


class Clusters(ctypes.Structure):
    _fields_ = [(n, _vp) for n in ("module", "first_digi", "n_pix", "charge", "x_col", "y_row", "module_first",
                                   "module_end", "clus_module_start", "summary")]


class Legacy(ctypes.Structure):
    _fields_ = [(n, _vp) for n in ("pdigi", "raw_id", "err_word", "err_fed", "err_type", "n_errors")]


class Hits(ctypes.Structure):
    _fields_ = [(n, _vp) for n in ("x_local", "y_local", "min_row", "max_row", "min_col", "max_col", "flags")]


_lib = None


def load() -> ctypes.CDLL:
    """Loads libpixclus.so (built in-tree by paper_2104_06573_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2104_06573_b200.build` "
                               "(there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        pp = ctypes.POINTER
        lib.pix_create.argtypes = [pp(CablingMap), pp(GainTable), pp(Params), pp(_vp)]
        lib.pix_clone.argtypes = [_vp, pp(_vp)]
        lib.pix_destroy.argtypes = [_vp]
        lib.pix_process.argtypes = [_vp, _vp, _vp, _vp, _u32, pp(Digis), pp(Clusters)]
        batch = [_vp, _vp, _u32, _vp, _u32, _vp, _vp, pp(Digis), pp(Clusters)]
        lib.pix_process_batch.argtypes = batch
        lib.pix_process_batch_host.argtypes = batch
        for f in ("pix_create", "pix_clone", "pix_destroy", "pix_process", "pix_process_batch",
                  "pix_process_batch_host"):
            getattr(lib, f).restype = ctypes.c_int
        lib.pix_kernel_launches.argtypes = [_vp]
        lib.pix_kernel_launches.restype = ctypes.c_uint64
        lib.pix_host_bytes_out.argtypes = [_vp]
        lib.pix_host_bytes_out.restype = ctypes.c_uint64
        lib.pix_set_profiling.argtypes = [_vp, ctypes.c_int]
        lib.pix_set_profiling.restype = ctypes.c_int
        lib.pix_read_profile.argtypes = [_vp, pp(ctypes.c_float), pp(_u32)]
        lib.pix_read_profile.restype = ctypes.c_int
        lib.pix_overflow_runs.argtypes = [_vp, pp(_u32)]
        lib.pix_overflow_runs.restype = ctypes.c_int
        lib.pix_last_error.argtypes = [_vp]
        lib.pix_last_error.restype = ctypes.c_char_p
        _lib = lib
    return _lib


class PixError(RuntimeError):
    def __init__(self, code: int, text: str = ""):
        super().__init__(f"pixclus error {code}: {text}")
        self.code = code


def _ptr(t) -> int | None:
    """Address of a torch tensor / numpy array / None."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags.c_contiguous
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


def _stream_ptr(stream) -> int | None:
    if stream is None:
        return None
    return stream if isinstance(stream, int) else stream.cuda_stream


@dataclass
class Handle:
    ptr: int
    n_feds: int
    n_modules: int
    params: dict


def make_params(params: dict, max_words_per_event: int, max_clusters_per_event: int, max_events_per_batch: int = 1,
                chunk_events: int = 0) -> Params:
    return Params(params["vcal_gain"], params["vcal_offset"], params["pixel_threshold_e"],
                  params["cluster_charge_cut_e"], params["max_electrons"],
                  params.get("max_clusters_per_module", 0xFFFFFFFF), max_words_per_event, max_clusters_per_event,
                  max_events_per_batch, chunk_events)


def pix_create(cabling: np.ndarray, n_feds: int, n_modules: int, gain: np.ndarray, pedestal: np.ndarray,
               params: Params) -> Handle:
    """pix_create(cabling_map, gain_table, params): host tables -> handle (device tables + workspace)."""
    cabling = np.ascontiguousarray(cabling, np.uint32)
    gain = np.ascontiguousarray(gain, np.float32)
    pedestal = np.ascontiguousarray(pedestal, np.float32)
    assert cabling.size == n_feds * 64 * 32 and gain.size == n_modules * COLS == pedestal.size
    cm = CablingMap(n_feds, n_modules, cabling.ctypes.data)
    gt = GainTable(n_modules, gain.ctypes.data, pedestal.ctypes.data)
    out = _vp()
    rc = load().pix_create(ctypes.byref(cm), ctypes.byref(gt), ctypes.byref(params), ctypes.byref(out))
    if rc != PIX_OK:
        raise PixError(rc, "pix_create")
    return Handle(out.value, n_feds, n_modules, {f: getattr(params, f) for f, _ in Params._fields_})


def pix_clone(h: Handle) -> Handle:
    out = _vp()
    rc = load().pix_clone(h.ptr, ctypes.byref(out))
    if rc != PIX_OK:
        raise PixError(rc, "pix_clone")
    return Handle(out.value, h.n_feds, h.n_modules, dict(h.params))


def pix_destroy(h: Handle) -> None:
    if h.ptr:
        load().pix_destroy(h.ptr)
        h.ptr = 0


def pix_last_error(h: Handle) -> str:
    return load().pix_last_error(h.ptr).decode()


def pix_kernel_launches(h: Handle) -> int:
    return int(load().pix_kernel_launches(h.ptr))


def pix_host_bytes_out(h: Handle) -> int:
    return int(load().pix_host_bytes_out(h.ptr))


def pix_overflow_runs(h: Handle) -> int:
    """Diagnostic: runs the last internal chunk left to the overflow kernel (synchronises the device)."""
    n = _u32()
    rc = load().pix_overflow_runs(h.ptr, ctypes.byref(n))
    if rc != PIX_OK:
        raise PixError(rc, pix_last_error(h))
    return int(n.value)


KERNEL_FAMILIES = ("init", "runs", "tile", "overflow", "finalize")


def pix_set_profiling(h: Handle, enable: bool) -> None:
    rc = load().pix_set_profiling(h.ptr, int(enable))
    if rc != PIX_OK:
        raise PixError(rc, "pix_set_profiling")


def pix_read_profile(h: Handle):
    """-> ({kernel family: accumulated ms}, chunks covered) since the last read."""
    ms = (ctypes.c_float * 8)()
    n = _u32()
    rc = load().pix_read_profile(h.ptr, ms, ctypes.byref(n))
    if rc != PIX_OK:
        raise PixError(rc, pix_last_error(h))
    return dict(zip(KERNEL_FAMILIES, (float(x) for x in ms))), int(n.value)


def _structs(digis: dict, clusters: dict):
    d = Digis(*[_ptr(digis.get(n)) for n, _ in Digis._fields_])
    c = Clusters(*[_ptr(clusters.get(n)) for n, _ in Clusters._fields_])
    return d, c


def _check(h: Handle, rc: int, raise_on_error: bool) -> int:
    if rc != PIX_OK and raise_on_error:
        raise PixError(rc, pix_last_error(h))
    return rc


def pix_process(h: Handle, stream, raw_words, fed_offsets, n_words: int, out_digis: dict, out_clusters: dict,
                raise_on_error: bool = True) -> int:
    """One event, device pointers, asynchronous on `stream` (a torch.cuda.Stream, a raw handle or None)."""
    d, c = _structs(out_digis, out_clusters)
    rc = load().pix_process(h.ptr, _stream_ptr(stream), _ptr(raw_words), _ptr(fed_offsets), n_words,
                            ctypes.byref(d), ctypes.byref(c))
    return _check(h, rc, raise_on_error)


def pix_process_batch(h: Handle, stream, n_events: int, raw_words, n_words_total: int, event_word_offsets,
                      fed_offsets, out_digis: dict, out_clusters: dict, raise_on_error: bool = True) -> int:
    """n_events events in one call, device pointers, asynchronous on `stream`."""
    d, c = _structs(out_digis, out_clusters)
    rc = load().pix_process_batch(h.ptr, _stream_ptr(stream), n_events, _ptr(raw_words), n_words_total,
                                  _ptr(event_word_offsets), _ptr(fed_offsets), ctypes.byref(d), ctypes.byref(c))
    return _check(h, rc, raise_on_error)


def pix_process_batch_host(h: Handle, stream, n_events: int, raw_words, n_words_total: int, event_word_offsets,
                           fed_offsets, out_digis: dict, out_clusters: dict, raise_on_error: bool = True) -> int:
    """Same with HOST pointers (numpy arrays or pinned torch CPU tensors); copies in and out, synchronous."""
    d, c = _structs(out_digis, out_clusters)
    rc = load().pix_process_batch_host(h.ptr, _stream_ptr(stream), n_events, _ptr(raw_words), n_words_total,
                                       _ptr(event_word_offsets), _ptr(fed_offsets), ctypes.byref(d), ctypes.byref(c))
    return _check(h, rc, raise_on_error)


def pix_rechits(h: Handle, stream, n_events: int, event_word_offsets, digis: dict, clusters: dict, out_hits: dict,
                raise_on_error: bool = True) -> int:
    """RecHits-lite over the outputs of pix_process_batch (device pointers, asynchronous on `stream`)."""
    d, c = _structs(digis, clusters)
    hh = Hits(*[_ptr(out_hits.get(n)) for n, _ in Hits._fields_])
    lib = load()
    lib.pix_rechits.argtypes = [_vp, _vp, _u32, _vp, ctypes.POINTER(Digis), ctypes.POINTER(Clusters), ctypes.POINTER(Hits)]
    lib.pix_rechits.restype = ctypes.c_int
    rc = lib.pix_rechits(h.ptr, _stream_ptr(stream), n_events, _ptr(event_word_offsets), ctypes.byref(d), ctypes.byref(c),
                         ctypes.byref(hh))
    return _check(h, rc, raise_on_error)


def pix_legacy_format(h: Handle, stream, n_events: int, raw_words, n_words_total: int, event_word_offsets, fed_offsets,
                      digis: dict, module_raw_id, max_errors_per_event: int, out: dict, raise_on_error: bool = True) -> int:
    """Legacy digi format + FED error words over the outputs of pix_process_batch (device pointers, asynchronous)."""
    d = Digis(*[_ptr(digis.get(n)) for n, _ in Digis._fields_])
    o = Legacy(*[_ptr(out.get(n)) for n, _ in Legacy._fields_])
    lib = load()
    lib.pix_legacy_format.argtypes = [_vp, _vp, _u32, _vp, _u32, _vp, _vp, ctypes.POINTER(Digis), _vp, _u32, ctypes.POINTER(Legacy)]
    lib.pix_legacy_format.restype = ctypes.c_int
    rc = lib.pix_legacy_format(h.ptr, _stream_ptr(stream), n_events, _ptr(raw_words), n_words_total, _ptr(event_word_offsets),
                               _ptr(fed_offsets), ctypes.byref(d), _ptr(module_raw_id), max_errors_per_event, ctypes.byref(o))
    return _check(h, rc, raise_on_error)


def pix_noalloc_last_error() -> str:
    lib = load()
    lib.pix_noalloc_last_error.restype = ctypes.c_char_p
    return (lib.pix_noalloc_last_error() or b"").decode()


def pix_noalloc_setup() -> None:
    """Looks up the static scratch array's address for the current device (allocates nothing)."""
    lib = load()
    lib.pix_noalloc_setup.restype = ctypes.c_int
    rc = lib.pix_noalloc_setup()
    if rc != 0:
        raise PixError(rc, pix_noalloc_last_error())


def pix_cluster_module_noalloc(stream, n_digis: int, row, col, charge, pixel_threshold_e: int, cluster_charge_cut_e: int,
                               max_clusters: int, out: dict, raise_on_error: bool = True) -> int:
    """One module's decoded digis -> clus, status, cluster records, counts, with no allocation anywhere (device
    pointers, asynchronous).  out: clus, status, first_digi, n_pix, charge, x_col, y_row, counts."""
    lib = load()
    lib.pix_cluster_module_noalloc.argtypes = [_vp, _u32, _vp, _vp, _vp, ctypes.c_int32, ctypes.c_int32, _u32] + [_vp] * 8
    lib.pix_cluster_module_noalloc.restype = ctypes.c_int
    rc = lib.pix_cluster_module_noalloc(_stream_ptr(stream), n_digis, _ptr(row), _ptr(col), _ptr(charge), pixel_threshold_e,
                                        cluster_charge_cut_e, max_clusters,
                                        *[_ptr(out.get(k)) for k in ("clus", "status", "first_digi", "n_pix", "charge",
                                                                     "x_col", "y_row", "counts")])
    if rc != 0 and raise_on_error:
        raise PixError(rc, pix_noalloc_last_error())
    return rc


def alloc_legacy(n_words: int, n_events: int, max_errors_per_event: int, device="cuda", fill: int | None = None):
    import torch
    shapes = dict(pdigi=(n_words + 16, "uint32"), raw_id=(n_words + 16, "uint32"),
                  err_word=(n_events * max_errors_per_event, "uint32"), err_fed=(n_events * max_errors_per_event, "uint16"),
                  err_type=(n_events * max_errors_per_event, "uint8"), n_errors=(n_events, "uint32"))
    out = {}
    for k, (n, dt) in shapes.items():
        t = torch.empty(max(int(n), 1), dtype=getattr(torch, dt), device=device)
        if fill is not None:
            t.view(torch.uint8).fill_(fill)
        out[k] = t
    return out


HIT_DTYPES = dict(x_local="float32", y_local="float32", min_row="uint16", max_row="uint16", min_col="uint16",
                  max_col="uint16", flags="uint8")


def alloc_hits(n_events: int, max_clusters_per_event: int, device="cuda", fill: int | None = None):
    import torch
    out = {}
    for k, dt in HIT_DTYPES.items():
        t = torch.empty(max(n_events * max_clusters_per_event, 1), dtype=getattr(torch, dt), device=device)
        if fill is not None:
            t.view(torch.uint8).fill_(fill)
        out[k] = t
    return out


# ---------------------------------------------------------------- output buffers (torch: device memory only)
DIGI_DTYPES = dict(module="uint16", row="uint16", col="uint16", charge="int32", clus="int32", status="uint8")
CLUSTER_DTYPES = dict(module="uint16", first_digi="uint32", n_pix="uint32", charge="uint32", x_col="float32",
                      y_row="float32")
PER_EVENT = dict(module_first="uint32", module_end="uint32", clus_module_start="uint32", summary="uint32")


def alloc_outputs(n_words: int, n_events: int, n_modules: int, max_clusters_per_event: int, device="cuda",
                  fill: int | None = None, pinned: bool = False):
    """(digis, clusters) dicts of tensors laid out as include/pixclus.h says.  fill: poison byte for tests."""
    import torch
    kw = dict(device=device) if device != "cpu" else dict(pin_memory=pinned)

    def mk(n, dt):
        t = torch.empty(max(int(n), 1), dtype=getattr(torch, dt), **kw)
        if fill is not None:
            t.view(torch.uint8).fill_(fill)
        return t

    digis = {k: mk(n_words + 16, dt) for k, dt in DIGI_DTYPES.items()}
    clusters = {k: mk(n_events * max_clusters_per_event, dt) for k, dt in CLUSTER_DTYPES.items()}
    clusters["module_first"] = mk(n_events * n_modules, "uint32")
    clusters["module_end"] = mk(n_events * n_modules, "uint32")
    clusters["clus_module_start"] = mk(n_events * (n_modules + 1), "uint32")
    clusters["summary"] = mk(n_events * 16, "uint32")
    return digis, clusters
