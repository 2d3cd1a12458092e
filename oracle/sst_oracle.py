"""ctypes front end of the CPU ORACLE (oracle/sst_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  It never imports the CUDA package and the CUDA package
never imports it.  All arithmetic lives in sst_oracle.c; this file only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sst_oracle.c")
_SRC_OMP = os.path.join(_HERE, "sst_oracle_omp.c")
_LIB = os.path.join(_HERE, "liboracle_sst.so")
_LIB_OMP = os.path.join(_HERE, "liboracle_sst_omp.so")
CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]

N_CHAN, N_STRIP = 96, 256
FLAG_CL_CAP, FLAG_ADC_CAP, FLAG_MALFORMED, FLAG_OVERRUN = 1, 2, 4, 8


def _stale(lib: str, srcs) -> bool:
    return (not os.path.exists(lib)) or any(os.path.getmtime(s) > os.path.getmtime(lib) for s in srcs)


def build(force: bool = False) -> None:
    """Compile the oracle (and its OpenMP timing build) with gcc."""
    if force or _stale(_LIB, [_SRC]):
        subprocess.check_call(["gcc", *CFLAGS, "-o", _LIB, _SRC, "-lm"])
    if os.path.exists(_SRC_OMP) and (force or _stale(_LIB_OMP, [_SRC, _SRC_OMP])):
        subprocess.check_call(["gcc", *CFLAGS, "-fopenmp", "-o", _LIB_OMP, _SRC_OMP, _SRC, "-lm"])


_lib = None
_lib_omp = None


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.sst_oracle_unpack.restype = None
        L.sst_oracle_unpack.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint32,
                                        C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.sst_oracle_flags.restype = C.c_uint32
        L.sst_oracle_flags.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64, C.c_float,
                                       C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]
        L.sst_oracle_gain_correct.restype = C.c_int32
        L.sst_oracle_gain_correct.argtypes = [C.c_uint8, C.c_float]
        L.sst_oracle_cluster.restype = None
        L.sst_oracle_cluster.argtypes = [C.c_void_p] * 6 + [C.c_uint32, C.c_float, C.c_uint32,
                                                            C.c_uint32] + [C.c_void_p] * 10
        L.sst_oracle_compact.restype = C.c_uint64
        L.sst_oracle_compact.argtypes = [C.c_void_p] * 4 + [C.c_uint64, C.c_uint64] + [C.c_void_p] * 5
        L.sst_oracle_hits.restype = None
        L.sst_oracle_hits.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint32] + [C.c_void_p] * 3
        _lib = L
    return _lib


def lib_omp():
    global _lib_omp
    if _lib_omp is None:
        build()
        L = C.CDLL(_LIB_OMP)
        L.sst_oracle_events_omp.restype = C.c_int
        _lib_omp = L
    return _lib_omp


@dataclass
class OracleResult:
    chan_off: np.ndarray
    chan_len: np.ndarray
    adc: np.ndarray          # dense uint8 [N]
    active: np.ndarray       # uint8 [N]
    seed: np.ndarray         # uint8 [N]
    seed_idx: np.ndarray     # uint32 [n_seeds]
    n_clusters: int
    cl_module: np.ndarray
    cl_first: np.ndarray
    cl_width: np.ndarray
    cl_charge: np.ndarray
    cl_bary: np.ndarray
    cl_adc_off: np.ndarray
    cl_adc: np.ndarray
    cl_snr: np.ndarray
    status: np.ndarray       # uint32 [8]: flags, n_malformed, n_cl_needed, n_adc_needed, n_overrun, n_seeds


def unpack(raw: np.ndarray, fed_offsets: np.ndarray, n_feds: int):
    raw = np.ascontiguousarray(raw, dtype=np.uint8)
    fo = np.ascontiguousarray(fed_offsets, dtype=np.uint32)
    assert fo.size == n_feds + 1
    nch = n_feds * N_CHAN
    chan_off = np.zeros(nch, np.uint32)
    chan_len = np.zeros(nch, np.uint16)
    adc = np.zeros(nch * N_STRIP, np.uint8)
    status = np.zeros(8, np.uint32)
    lib().sst_oracle_unpack(_p(raw), raw.size, _p(fo), n_feds, _p(chan_off), _p(chan_len), _p(adc),
                            _p(status))
    return chan_off, chan_len, adc, status


def flags(adc, noise, bad, t_ch: float, t_seed: float):
    n = adc.size
    active = np.zeros(n, np.uint8)
    seed = np.zeros(n, np.uint8)
    seed_idx = np.zeros(n, np.uint32)
    ns = lib().sst_oracle_flags(_p(adc), _p(noise), _p(bad), n, t_ch, t_seed, _p(active), _p(seed),
                                _p(seed_idx))
    return active, seed, seed_idx[:ns].copy()


def gain_correct(adc: int, gain) -> int:
    return int(lib().sst_oracle_gain_correct(int(adc), float(np.float32(gain))))


def cluster(adc, gain, noise, active, seed, chan_module, n_feds, t_cl: float,
            cap_clusters: Optional[int] = None, cap_adc: Optional[int] = None, status=None):
    nz = int(np.count_nonzero(active))
    capc = nz if cap_clusters is None else int(cap_clusters)
    capa = nz if cap_adc is None else int(cap_adc)
    st = np.zeros(8, np.uint32) if status is None else status
    n_cl = np.zeros(1, np.uint32)
    m = max(capc, 1)
    cl_module = np.zeros(m, np.uint32)
    cl_first = np.zeros(m, np.uint16)
    cl_width = np.zeros(m, np.uint16)
    cl_charge = np.zeros(m, np.int32)
    cl_bary = np.zeros(m, np.float32)
    cl_adc_off = np.zeros(m, np.uint32)
    cl_adc = np.zeros(max(capa, 1), np.uint8)
    cl_snr = np.zeros(m, np.float32)
    lib().sst_oracle_cluster(_p(adc), _p(gain), _p(noise), _p(active), _p(seed), _p(chan_module),
                             n_feds, t_cl, capc, capa, _p(n_cl), _p(cl_module), _p(cl_first),
                             _p(cl_width), _p(cl_charge), _p(cl_bary), _p(cl_adc_off), _p(cl_adc),
                             _p(cl_snr), _p(st))
    k = int(n_cl[0])
    na = int(cl_adc_off[k - 1]) + int(cl_width[k - 1]) if k else 0
    return dict(n_clusters=k, cl_module=cl_module[:k], cl_first=cl_first[:k], cl_width=cl_width[:k],
                cl_charge=cl_charge[:k], cl_bary=cl_bary[:k], cl_adc_off=cl_adc_off[:k],
                cl_adc=cl_adc[:na], cl_snr=cl_snr[:k], status=st)


def run(raw, fed_offsets, n_feds, gain, noise, bad, chan_module, thresholds,
        cap_clusters: Optional[int] = None, cap_adc: Optional[int] = None) -> OracleResult:
    """The whole path on one event: walk + decode, flags + seed-index array, clustering."""
    t_ch, t_seed, t_cl = (float(np.float32(t)) for t in thresholds)
    if not all(np.isfinite(t) and t > 0 for t in (t_ch, t_seed, t_cl)):
        raise ValueError("thresholds must be finite and > 0")
    gain = np.ascontiguousarray(gain, np.float32)
    noise = np.ascontiguousarray(noise, np.float32)
    bad = np.ascontiguousarray(bad, np.uint8)
    chan_module = np.ascontiguousarray(chan_module, np.uint32)
    chan_off, chan_len, adc, status = unpack(raw, fed_offsets, n_feds)
    active, seed, seed_idx = flags(adc, noise, bad, t_ch, t_seed)
    status[5] = seed_idx.size
    c = cluster(adc, gain, noise, active, seed, chan_module, n_feds, t_cl, cap_clusters, cap_adc,
                status)
    return OracleResult(chan_off, chan_len, adc, active, seed, seed_idx, c["n_clusters"],
                        c["cl_module"], c["cl_first"], c["cl_width"], c["cl_charge"], c["cl_bary"],
                        c["cl_adc_off"], c["cl_adc"], c["cl_snr"], status)


def compact(adc, gain, noise, bad, cap: Optional[int] = None):
    """Compact SoA (sst_oracle_compact): one entry per recorded strip, ascending strip id.
    Returns (n_present, dict of arrays trimmed to min(n_present, cap))."""
    adc = np.ascontiguousarray(adc, np.uint8)
    gain = np.ascontiguousarray(gain, np.float32)
    noise = np.ascontiguousarray(noise, np.float32)
    bad = np.ascontiguousarray(bad, np.uint8)
    capn = int(np.count_nonzero(adc)) if cap is None else int(cap)
    m = max(capn, 1)
    out = dict(strip=np.zeros(m, np.uint32), adc=np.zeros(m, np.uint8), noise=np.zeros(m, np.float32),
               gain=np.zeros(m, np.float32), bad=np.zeros(m, np.uint8))
    k = int(lib().sst_oracle_compact(_p(adc), _p(gain), _p(noise), _p(bad), adc.size, capn, _p(out["strip"]),
                                     _p(out["adc"]), _p(out["noise"]), _p(out["gain"]), _p(out["bad"])))
    w = min(k, capn)
    return k, {key: v[:w] for key, v in out.items()}


def hits(cl_module, cl_bary, geom):
    """Global hit coordinates of clusters (sst_oracle_hits); geom float32 [n_modules, 6]."""
    cm = np.ascontiguousarray(cl_module, np.uint32)
    cb = np.ascontiguousarray(cl_bary, np.float32)
    g = np.ascontiguousarray(geom, np.float32).reshape(-1, 6)
    n = cm.size
    x, y, z = (np.zeros(max(n, 1), np.float32) for _ in range(3))
    lib().sst_oracle_hits(_p(cm), _p(cb), n, _p(g), g.shape[0], _p(x), _p(y), _p(z))
    return x[:n], y[:n], z[:n]


def events_omp(raws, fed_offsets_list, n_feds, gain, noise, bad, chan_module, thresholds,
               n_outer: int, n_inner: int):
    """OpenMP timing build (sst_oracle_omp.c): N events x M FED ranges.  Returns per event
    (n_clusters, n_seeds, FNV-1a hash of the outputs)."""
    L = lib_omp()
    ne = len(raws)
    raws = [np.ascontiguousarray(r, np.uint8) for r in raws]
    fos = [np.ascontiguousarray(f, np.uint32) for f in fed_offsets_list]
    rp = (C.c_void_p * ne)(*[r.ctypes.data for r in raws])
    fp = (C.c_void_p * ne)(*[f.ctypes.data for f in fos])
    rb = np.asarray([r.size for r in raws], np.uint64)
    ncl = np.zeros(ne, np.uint32)
    nsd = np.zeros(ne, np.uint32)
    hh = np.zeros(ne, np.uint64)
    t = [C.c_float(float(np.float32(x))) for x in thresholds]
    L.sst_oracle_events_omp(C.c_uint32(ne), rp, _p(rb), fp, C.c_uint32(n_feds), _p(gain), _p(noise),
                            _p(bad), _p(chan_module), t[0], t[1], t[2], C.c_int(n_outer),
                            C.c_int(n_inner), _p(ncl), _p(nsd), _p(hh))
    return ncl, nsd, hh


def result_hash(res: OracleResult) -> int:
    """The FNV-1a hash sst_oracle_events_omp computes, from a sequential OracleResult."""
    rec = np.zeros(res.n_clusters, dtype=np.dtype([("m", "<u4"), ("f", "<u2"), ("w", "<u2"),
                                                   ("q", "<i4"), ("b", "<f4"), ("o", "<u4")]))
    rec["m"], rec["f"], rec["w"] = res.cl_module, res.cl_first, res.cl_width
    rec["q"], rec["b"], rec["o"] = res.cl_charge, res.cl_bary, res.cl_adc_off
    h = 14695981039346656037
    for b in rec.tobytes() + res.cl_adc.tobytes():
        h = ((h ^ b) * 1099511628211) & 0xFFFFFFFFFFFFFFFF
    return h
