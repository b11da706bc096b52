"""pixgen -- seeded synthetic inputs (tables + raw-word events) for the pixel Clusters path.

Serves both the oracle tests and the CUDA tests / bench.  Holds none of the method's arithmetic:
it only builds input bytes (see pixgen.c header and DESIGN.md "Input recipe").  The synthetic
events stand in for the paper's dataset (CMS Open Data ttbar <PU>=50), which is
not available on the box; sizes and distributions follow BASELINE.json configs[0..4].
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pixgen.c")
_LIB = os.path.join(_HERE, "libpixgen.so")

ROWS, COLS = 160, 416
CABLING_SEED = 0xCAB1E
GAIN_SEED = 0x6A15

# BASELINE.json configs[0]: pixel threshold 1000 e, cluster-charge cut 4000 e.  vcal_* and
# max_electrons: DESIGN.md reading S7/S15 (the config gives no VCAL->electron map).
DEFAULT_PARAMS = dict(vcal_gain=47.0, vcal_offset=-60.0, pixel_threshold_e=1000,
                      cluster_charge_cut_e=4000, max_electrons=64000,
                      max_clusters_per_module=0xFFFFFFFF)


def build(force: bool = False) -> str:
    """Compiles pixgen.c into libpixgen.so (in-tree) if missing or older than its sources."""
    deps = [_SRC, os.path.join(_HERE, "adc_cdf.h")]
    if force or not os.path.exists(_LIB) or any(os.path.getmtime(d) > os.path.getmtime(_LIB) for d in deps):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC])
    return _LIB


class _Cfg(ctypes.Structure):
    _fields_ = [(n, ctypes.c_uint32) for n in (
        "clusters_per_module", "n_clusters", "inner_modules", "inner_weight", "long_permille",
        "shuffle_order", "edge_class", "edge_sub")]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u32p, f32p, u64p = (ctypes.POINTER(t) for t in (ctypes.c_uint32, ctypes.c_float, ctypes.c_uint64))
        lib.pixgen_cabling.argtypes = [ctypes.c_uint32] * 3 + [ctypes.c_uint64, u32p]
        lib.pixgen_cabling.restype = ctypes.c_int
        lib.pixgen_gains.argtypes = [ctypes.c_uint32, ctypes.c_uint64, f32p, f32p]
        lib.pixgen_gains.restype = None
        lib.pixgen_batch.argtypes = [ctypes.POINTER(_Cfg), u64p, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32,
                                     u32p, u32p, ctypes.c_uint64, u32p, u32p, u32p]
        lib.pixgen_batch.restype = ctypes.c_int64
        _lib = lib
    return _lib


def _p(a, t):
    return a.ctypes.data_as(ctypes.POINTER(t))


@dataclass
class Detector:
    """Conditions: cabling map + gain table (the two pix_create inputs)."""
    n_feds: int
    links_per_fed: int
    n_modules: int
    cabling: np.ndarray      # uint32 [F*64*32]
    gain: np.ndarray         # float32 [M*416]
    pedestal: np.ndarray     # float32 [M*416]
    _inv: dict = field(default_factory=dict, repr=False)

    def inverse(self):
        """module -> (fed, link, roc id at placement p, flips at placement p), from the entry table."""
        if not self._inv:
            e = self.cabling.reshape(self.n_feds, 64, 32)
            M = self.n_modules
            fed = np.full(M, -1, np.int64); link = np.full(M, -1, np.int64)
            roc = np.zeros((M, 16), np.int64); flip = np.zeros((M, 16), np.int64)
            f, l, r = np.nonzero((e & 2) != 0)
            v = e[f, l, r]
            m = (v >> 2) & 0xFFFF
            p = ((v >> 21) & 1) * 8 + ((v >> 18) & 7)
            fed[m] = f; link[m] = l; roc[m, p] = r; flip[m, p] = (v >> 22) & 3
            self._inv = dict(fed=fed, link=link, roc=roc, flip=flip)
        return self._inv

    def encode(self, module, row, col, adc):
        """(module,row,col,adc) -> raw words, plus the FED each word belongs to (encode direction only)."""
        inv = self.inverse()
        module, row, col, adc = (np.asarray(x, np.int64) for x in (module, row, col, adc))
        p = (row // 80) * 8 + col // 52
        rloc, cloc = row % 80, col % 52
        roc, flip = inv["roc"][module, p], inv["flip"][module, p]
        rr = np.where(flip & 1, 79 - rloc, rloc)
        cc = np.where(flip & 2, 51 - cloc, cloc)
        w = (inv["link"][module] << 26) | (roc << 21) | ((cc >> 1) << 16) | ((rr * 2 + (cc & 1)) << 8) | adc
        return w.astype(np.uint32), inv["fed"][module]

    def stream(self, module, row, col, adc):
        """Hand-built event: encodes the pixels and orders them FED-ascending (stable), returning
        (words, fed_offsets, perm) where perm maps stream position -> index into the inputs."""
        w, fed = self.encode(module, row, col, adc)
        perm = np.argsort(fed, kind="stable")
        counts = np.bincount(fed[perm], minlength=self.n_feds) if len(w) else np.zeros(self.n_feds, np.int64)
        fed_offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.uint32)
        return w[perm], fed_offsets, perm


def detector(kind: str = "full", cabling_seed: int = CABLING_SEED, gain_seed: int = GAIN_SEED) -> Detector:
    """'tiny': F=2 x 32 links = 64 modules (cfg0).  'full': F=32 x 58 links = 1856 modules (cfg1-4)."""
    F, L = {"tiny": (2, 32), "full": (32, 58)}[kind]
    M = F * L
    lib = _load()
    cab = np.zeros(F * 64 * 32, np.uint32)
    if lib.pixgen_cabling(F, L, M, cabling_seed, _p(cab, ctypes.c_uint32)) != 0:
        raise RuntimeError("pixgen_cabling failed")
    gain = np.zeros(M * COLS, np.float32); ped = np.zeros(M * COLS, np.float32)
    lib.pixgen_gains(M, gain_seed, _p(gain, ctypes.c_float), _p(ped, ctypes.c_float))
    return Detector(F, L, M, cab, gain, ped)


@dataclass
class Batch:
    """Raw input of n_events events, concatenated."""
    words: np.ndarray           # uint32 [n_words_total]
    event_offsets: np.ndarray   # uint32 [E+1]
    fed_offsets: np.ndarray     # uint32 [E, F+1], event-relative
    tally: np.ndarray           # uint32 [E, 5]: injected n_empty, n_err_link, n_err_roc, n_err_dcol, n_err_pxid

    @property
    def n_events(self):
        return len(self.event_offsets) - 1

    def event(self, e):
        a, b = int(self.event_offsets[e]), int(self.event_offsets[e + 1])
        return self.words[a:b], self.fed_offsets[e]


# event recipes; values are pixgen_cfg fields
RECIPES = {
    "tiny":   dict(clusters_per_module=40, shuffle_order=1),                                   # cfg0
    "pu50":   dict(n_clusters=15000, inner_modules=96, inner_weight=4),                        # cfg1 / cfg2
    "pu200":  dict(n_clusters=40000, inner_modules=96, inner_weight=4, long_permille=20),      # cfg3
    "dense":  dict(n_clusters=15000, inner_modules=96, inner_weight=4, shuffle_order=1, edge_class=1),  # cfg4 (a)
    "dups":   dict(n_clusters=15000, inner_modules=96, inner_weight=4, shuffle_order=1, edge_class=2),  # cfg4 (b)
    "errors": dict(n_clusters=15000, inner_modules=96, inner_weight=4, shuffle_order=1, edge_class=3),  # cfg4 (c)
    "edges":  dict(n_clusters=15000, inner_modules=96, inner_weight=4, shuffle_order=1, edge_class=4),  # cfg4 (d)
}
for _s, _n in enumerate(("empty", "oneword", "allbad", "threemods", "fedempty")):                # cfg4 (e)
    RECIPES[_n] = dict(n_clusters=15000, inner_modules=96, inner_weight=4, shuffle_order=1, edge_class=5, edge_sub=_s)


def events(det: Detector, recipes, seeds, cap_words_per_event: int = 1 << 18) -> Batch:
    """Generates len(seeds) events; recipes is one recipe name/dict or a list of them (one per event)."""
    seeds = np.asarray(seeds, np.uint64)
    E = len(seeds)
    if isinstance(recipes, (str, dict)):
        recipes = [recipes] * E
    cfgs = (_Cfg * max(E, 1))()
    for i, r in enumerate(recipes):
        r = RECIPES[r] if isinstance(r, str) else r
        for k, v in r.items():
            setattr(cfgs[i], k, v)
    cap = int(cap_words_per_event) * max(E, 1)
    words = np.zeros(cap, np.uint32)
    ev_off = np.zeros(E + 1, np.uint32)
    fed_off = np.zeros((E, det.n_feds + 1), np.uint32)
    tally = np.zeros((E, 5), np.uint32)
    n = _load().pixgen_batch(cfgs, _p(seeds, ctypes.c_uint64), E, det.n_feds, det.n_modules,
                             _p(det.cabling, ctypes.c_uint32), _p(words, ctypes.c_uint32), cap,
                             _p(ev_off, ctypes.c_uint32), _p(fed_off, ctypes.c_uint32), _p(tally, ctypes.c_uint32))
    if n < 0:
        raise RuntimeError(f"pixgen_batch failed ({n})")
    return Batch(words[:n].copy(), ev_off, fed_off, tally)


def config(name: str, n_events: int | None = None):
    """The five BASELINE.json configs -> (detector kind, Batch).  n_events truncates cfg2/3/4."""
    if name == "cfg0":
        det = detector("tiny")
        return det, events(det, "tiny", [0])
    det = detector("full")
    if name == "cfg1":
        return det, events(det, "pu50", [0])
    if name == "cfg2":
        return det, events(det, "pu50", np.arange(n_events or 1000))
    if name == "cfg3":
        return det, events(det, "pu200", np.arange(n_events or 200))
    if name == "cfg4":
        E = n_events or 100
        per = max(E // 5, 1)
        rec = []
        for e in range(E):
            k = min(e // per, 4)
            rec.append(("dense", "dups", "errors", "edges")[k] if k < 4 else
                       ("empty", "oneword", "allbad", "threemods", "fedempty")[(e - 4 * per) % 5])
        return det, events(det, rec, np.arange(E))
    raise KeyError(name)
