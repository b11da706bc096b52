"""oracle -- ctypes wrapper around oracle/pix_oracle.cpp.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  Nothing here touches the CUDA path; nothing in the CUDA path touches this.
The arithmetic lives entirely in pix_oracle.cpp (see its header for citations and pins).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pix_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

STATUS = dict(OK=0, CUT=1, BELOW_THRESHOLD=2, DUPLICATE=3, EMPTY=4, ERR_LINK=5, ERR_ROC=6, ERR_DCOL=7, ERR_PXID=8)
SUMMARY = ("n_words", "n_decoded", "n_empty", "n_err_link", "n_err_roc", "n_err_dcol", "n_err_pxid", "n_duplicate",
           "n_below_threshold", "n_ok_digis", "n_cut_digis", "n_modules_present", "n_clusters_precut", "n_clusters",
           "n_clusters_emitted", "flags")


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (no FMA contraction: DESIGN.md reading S7)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_SRC) > os.path.getmtime(_LIB):
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", _LIB, _SRC])
    return _LIB


class Params(ctypes.Structure):
    _fields_ = [("vcal_gain", ctypes.c_float), ("vcal_offset", ctypes.c_float),
                ("pixel_threshold_e", ctypes.c_int32), ("cluster_charge_cut_e", ctypes.c_int32),
                ("max_electrons", ctypes.c_int32), ("max_clusters_per_module", ctypes.c_uint32),
                ("max_clusters_per_event", ctypes.c_uint32)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp = ctypes.c_void_p
        lib.pixo_process.argtypes = [ctypes.c_uint32, ctypes.c_uint32, vp, vp, vp, ctypes.POINTER(Params), vp, vp,
                                     ctypes.c_uint32] + [vp] * 16
        lib.pixo_process.restype = ctypes.c_int
        lib.pixo_decode_word.argtypes = [ctypes.c_uint32, ctypes.c_uint32, vp] + [vp] * 4
        lib.pixo_decode_word.restype = ctypes.c_int
        lib.pixo_calibrate.argtypes = [ctypes.c_uint8, ctypes.c_float, ctypes.c_float, ctypes.POINTER(Params)]
        lib.pixo_calibrate.restype = ctypes.c_int32
        lib.pixo_rechits.argtypes = [ctypes.c_uint32, ctypes.c_uint32] + [vp] * 6 + [ctypes.c_uint32] + [vp] * 10
        lib.pixo_rechits.restype = ctypes.c_int
        lib.pixo_legacy.argtypes = [ctypes.c_uint32, ctypes.c_uint32] + [vp] * 7 + [ctypes.c_uint32, ctypes.c_uint32] + [vp] * 6
        lib.pixo_legacy.restype = ctypes.c_int
        _lib = lib
    return _lib


def make_params(params: dict, max_clusters_per_event: int) -> Params:
    return Params(params["vcal_gain"], params["vcal_offset"], params["pixel_threshold_e"],
                  params["cluster_charge_cut_e"], params["max_electrons"],
                  params.get("max_clusters_per_module", 0xFFFFFFFF), max_clusters_per_event)


def decode_word(word: int, fed: int, cabling: np.ndarray):
    """O1 for one word -> (status, module, row, col, adc)."""
    m, r, c = (ctypes.c_uint16() for _ in range(3))
    a = ctypes.c_uint8()
    st = _load().pixo_decode_word(int(word), int(fed), cabling.ctypes.data, ctypes.addressof(m), ctypes.addressof(r),
                                  ctypes.addressof(c), ctypes.addressof(a))
    return st, m.value, r.value, c.value, a.value


def calibrate(adc: int, gain: float, pedestal: float, params: dict) -> int:
    """O2 for one pixel."""
    p = make_params(params, 0)
    return _load().pixo_calibrate(int(adc), float(gain), float(pedestal), ctypes.byref(p))


def process(det, words: np.ndarray, fed_offsets, params: dict, max_clusters_per_event: int | None = None) -> dict:
    """The whole path for one event.  det: anything with n_feds, n_modules, cabling, gain, pedestal."""
    words = np.ascontiguousarray(words, np.uint32)
    n = len(words)
    M = det.n_modules
    kmax = int(max_clusters_per_event if max_clusters_per_event is not None else max(n, 1))
    p = make_params(params, kmax)
    fo = None if fed_offsets is None else np.ascontiguousarray(fed_offsets, np.uint32)
    out = dict(
        module=np.empty(n, np.uint16), row=np.empty(n, np.uint16), col=np.empty(n, np.uint16),
        charge=np.empty(n, np.int32), clus=np.empty(n, np.int32), status=np.empty(n, np.uint8),
        c_module=np.zeros(kmax, np.uint16), c_first_digi=np.zeros(kmax, np.uint32), c_n_pix=np.zeros(kmax, np.uint32),
        c_charge=np.zeros(kmax, np.uint32), c_x_col=np.zeros(kmax, np.float32), c_y_row=np.zeros(kmax, np.float32),
        module_first=np.empty(M, np.uint32), module_end=np.empty(M, np.uint32),
        clus_module_start=np.empty(M + 1, np.uint32), summary=np.empty(16, np.uint32))
    order = ("module", "row", "col", "charge", "clus", "status", "c_module", "c_first_digi", "c_n_pix", "c_charge",
             "c_x_col", "c_y_row", "module_first", "module_end", "clus_module_start", "summary")
    rc = _load().pixo_process(det.n_feds, M, det.cabling.ctypes.data, det.gain.ctypes.data, det.pedestal.ctypes.data,
                              ctypes.byref(p), words.ctypes.data, None if fo is None else fo.ctypes.data, n,
                              *[out[k].ctypes.data for k in order])
    if rc != 0:
        raise ValueError(f"pixo_process returned {rc}")
    k = int(out["summary"][14])
    for name in ("c_module", "c_first_digi", "c_n_pix", "c_charge", "c_x_col", "c_y_row"):
        out[name] = out[name][:k]
    return out


def rechits(det, o: dict) -> dict:
    """RecHits-lite (S25-S28) from one event's process() output -> hit arrays, one per emitted record."""
    k = int(o["summary"][14])
    h = dict(x_local=np.zeros(k, np.float32), y_local=np.zeros(k, np.float32), min_row=np.zeros(k, np.uint16),
             max_row=np.zeros(k, np.uint16), min_col=np.zeros(k, np.uint16), max_col=np.zeros(k, np.uint16),
             flags=np.zeros(k, np.uint8))
    ins = [np.ascontiguousarray(o[n]) for n in ("module", "row", "col", "clus", "status", "clus_module_start")]
    recs = [np.ascontiguousarray(o[n]) for n in ("c_n_pix", "c_x_col", "c_y_row")]
    rc = _load().pixo_rechits(len(o["module"]), det.n_modules, *[a.ctypes.data for a in ins], k,
                              *[a.ctypes.data for a in recs],
                              *[h[n].ctypes.data for n in ("x_local", "y_local", "min_row", "max_row", "min_col", "max_col", "flags")])
    if rc != 0:
        raise ValueError(f"pixo_rechits returned {rc}")
    return h


def legacy(det, words: np.ndarray, fed_offsets, o: dict, module_raw_id: np.ndarray, max_errors: int) -> dict:
    """Legacy digi format + FED error words (S29-S31) from one event's raw words and process() output."""
    words = np.ascontiguousarray(words, np.uint32)
    n = len(words)
    rid = np.ascontiguousarray(module_raw_id, np.uint32)
    fo = None if fed_offsets is None else np.ascontiguousarray(fed_offsets, np.uint32)
    out = dict(pdigi=np.zeros(n, np.uint32), raw_id=np.zeros(n, np.uint32), err_word=np.zeros(max_errors, np.uint32),
               err_fed=np.zeros(max_errors, np.uint16), err_type=np.zeros(max_errors, np.uint8), n_errors=np.zeros(1, np.uint32))
    ins = [np.ascontiguousarray(o[k]) for k in ("module", "row", "col", "status")]
    rc = _load().pixo_legacy(n, det.n_feds, words.ctypes.data, None if fo is None else fo.ctypes.data,
                             *[a.ctypes.data for a in ins], rid.ctypes.data, det.n_modules, max_errors,
                             *[out[k].ctypes.data for k in ("pdigi", "raw_id", "err_word", "err_fed", "err_type", "n_errors")])
    if rc != 0:
        raise ValueError(f"pixo_legacy returned {rc}")
    k = min(int(out["n_errors"][0]), max_errors)
    for name in ("err_word", "err_fed", "err_type"):
        out[name] = out[name][:k]
    return out
