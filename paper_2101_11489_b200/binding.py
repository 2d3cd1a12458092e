"""Thin Python binding of libsst (include/sst.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/sst.cu.  There is NO CPU fallback: if
csrc/libsst.so is missing or cannot be loaded, ``load()`` raises.  torch is used for device
memory and streams only (``tensor.data_ptr()``, ``torch.cuda.Stream.cuda_stream``).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "csrc", "libsst.so")

N_CHAN, N_STRIP, FED_STRIPS = 96, 256, 96 * 256
ST_WORDS = 8
ST_FLAGS, ST_N_MALFORMED, ST_N_CLUSTERS, ST_N_ADC, ST_N_OVERRUN, ST_N_SEEDS, ST_N_PRESENT = range(7)
FLAG_CLUSTER_CAP, FLAG_ADC_CAP, FLAG_MALFORMED, FLAG_OVERRUN, FLAG_COMPACT_CAP = 1, 2, 4, 8, 16
SST_OK, SST_ERR_INVALID_ARG, SST_ERR_CUDA, SST_ERR_NO_CALIB, SST_ERR_BAD_CALIB, SST_ERR_TOO_LARGE = range(6)
NOALLOC_SCRATCH_BYTES = 32 << 20

EXPORTS = ["sst_create", "sst_upload_calib", "sst_upload_geometry", "sst_unpack_cluster", "sst_unpack_cluster_noalloc",
           "sst_unpack_cluster_batch", "sst_unpack_cluster_host",
           "sst_unpack_cluster_host_batch", "sst_unpack_cluster_host_packed",
           "sst_event_alloc", "sst_event_free", "sst_event_upload", "sst_event_download", "sst_destroy", "sst_last_cuda_error",
           "sst_status_string", "sst_get_info", "sst_trace_read"]


class sst_config(C.Structure):
    _fields_ = [("n_feds", C.c_uint32), ("device", C.c_int32), ("max_raw_bytes", C.c_uint32),
                ("max_events_in_flight", C.c_uint32), ("fed_strips_hint", C.c_uint32), ("move_mode", C.c_uint32),
                ("trace", C.c_uint32)]


class sst_thresholds(C.Structure):
    _fields_ = [("channel", C.c_float), ("seed", C.c_float), ("cluster", C.c_float)]


class sst_output(C.Structure):
    _fields_ = [("strip_adc", C.c_void_p), ("chan_off", C.c_void_p), ("chan_len", C.c_void_p),
                ("seed_idx", C.c_void_p), ("cap_seeds", C.c_uint32), ("cap_clusters", C.c_uint32),
                ("cap_adc", C.c_uint32), ("n_clusters", C.c_void_p), ("cl_module", C.c_void_p),
                ("cl_first", C.c_void_p), ("cl_width", C.c_void_p), ("cl_charge", C.c_void_p),
                ("cl_bary", C.c_void_p), ("cl_adc_off", C.c_void_p), ("cl_snr", C.c_void_p),
                ("cl_adc", C.c_void_p), ("dev_status", C.c_void_p),
                ("compact_strip", C.c_void_p), ("compact_adc", C.c_void_p), ("compact_noise", C.c_void_p),
                ("compact_gain", C.c_void_p), ("compact_bad", C.c_void_p), ("cap_compact", C.c_uint32),
                ("hit_x", C.c_void_p), ("hit_y", C.c_void_p), ("hit_z", C.c_void_p)]


class sst_info(C.Structure):
    _fields_ = [("smem_bytes", C.c_uint32), ("threads", C.c_uint32), ("ctas_per_sm", C.c_uint32),
                ("sm_count", C.c_uint32), ("kernels_per_event", C.c_uint32), ("slot_bytes", C.c_uint32),
                ("events_per_launch", C.c_uint32), ("pieces", C.c_uint32)]


class SSTError(RuntimeError):
    pass


_lib = None


def load():
    """dlopen csrc/libsst.so and declare the C ABI.  Raises if the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise SSTError(f"{LIB_PATH} is not built; run `python -m paper_2101_11489_b200.build` "
                       "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    L.sst_create.argtypes = [C.POINTER(sst_config), C.POINTER(vp)]
    L.sst_upload_calib.argtypes = [vp, vp, vp, vp, vp]
    L.sst_upload_geometry.argtypes = [vp, vp, C.c_uint32]
    L.sst_unpack_cluster.argtypes = [vp, vp, vp, C.POINTER(sst_thresholds), C.POINTER(sst_output), vp]
    L.sst_unpack_cluster_noalloc.argtypes = [vp, vp, vp, C.POINTER(sst_thresholds), C.POINTER(sst_output), vp]
    L.sst_unpack_cluster_batch.argtypes = [vp, C.c_uint32, vp, vp, C.POINTER(sst_thresholds), vp, vp, C.c_uint32]
    L.sst_unpack_cluster_host.argtypes = [vp, vp, C.c_uint32, vp, C.POINTER(sst_thresholds),
                                          C.POINTER(sst_output), vp]
    L.sst_unpack_cluster_host_batch.argtypes = [vp, C.c_uint32, vp, vp, vp, C.POINTER(sst_thresholds), vp, vp, C.c_uint32]
    L.sst_unpack_cluster_host_packed.argtypes = [vp, C.c_uint32, vp, vp, vp, C.POINTER(sst_thresholds), C.c_uint32,
                                                 C.c_uint32, vp, vp, C.c_uint32]
    L.sst_event_alloc.argtypes = [vp, C.c_uint64, vp, C.POINTER(vp)]
    L.sst_event_free.argtypes = [vp, vp, vp]
    L.sst_event_upload.argtypes = [vp, vp, C.c_uint32, vp, vp, C.POINTER(vp), C.POINTER(vp)]
    L.sst_event_download.argtypes = [vp, vp, vp, C.c_uint64, vp]
    L.sst_destroy.argtypes = [vp]
    L.sst_last_cuda_error.argtypes = [vp]
    L.sst_last_cuda_error.restype = C.c_int32
    L.sst_status_string.argtypes = [C.c_int]
    L.sst_status_string.restype = C.c_char_p
    L.sst_get_info.argtypes = [vp, C.POINTER(sst_info)]
    L.sst_trace_read.argtypes = [vp, vp, C.POINTER(C.c_uint64)]
    for name in EXPORTS:
        if name not in ("sst_last_cuda_error", "sst_status_string"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _check(ctx, rc: int, what: str):
    if rc != SST_OK:
        L = load()
        msg = L.sst_status_string(rc).decode()
        cu = L.sst_last_cuda_error(ctx) if ctx else 0
        raise SSTError(f"{what}: {msg}" + (f" (cudaError {cu})" if rc == SST_ERR_CUDA else ""))


def _ptr(t) -> Optional[int]:
    """Device (or pinned host) pointer of a torch tensor / numpy array / int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def sst_create(n_feds: int, device: int = 0, max_raw_bytes: int = 1 << 22, max_events_in_flight: int = 8,
               fed_strips_hint: int = 0, move_mode: int = 0, trace: int = 0):
    L = load()
    cfg = sst_config(n_feds, device, max_raw_bytes, max_events_in_flight, fed_strips_hint, move_mode, trace)
    ctx = C.c_void_p()
    _check(None, L.sst_create(C.byref(cfg), C.byref(ctx)), "sst_create")
    return ctx


def sst_upload_calib(ctx, gain, noise, bad, chan_module):
    """HOST numpy arrays: gain/noise float32 [N], bad uint8 [N], chan_module uint32 [n_feds*96]."""
    import numpy as np
    g = np.ascontiguousarray(gain, np.float32)
    n = np.ascontiguousarray(noise, np.float32)
    b = np.ascontiguousarray(bad, np.uint8)
    m = np.ascontiguousarray(chan_module, np.uint32)
    _check(ctx, load().sst_upload_calib(ctx, _ptr(g), _ptr(n), _ptr(b), _ptr(m)), "sst_upload_calib")


def sst_upload_geometry(ctx, geom):
    """HOST float32 array [n_modules, 6] = {pitch, u0, r, cos phi, sin phi, z} per module id."""
    import numpy as np
    g = np.ascontiguousarray(geom, np.float32).reshape(-1, 6)
    _check(ctx, load().sst_upload_geometry(ctx, _ptr(g), g.shape[0]), "sst_upload_geometry")


def make_output(*, n_clusters, cl_module, cl_first, cl_width, cl_charge, cl_bary, cl_adc_off, cl_adc,
                dev_status, cap_clusters: int, cap_adc: int, strip_adc=None, chan_off=None,
                chan_len=None, seed_idx=None, cap_seeds: int = 0, cl_snr=None, compact_strip=None,
                compact_adc=None, compact_noise=None, compact_gain=None, compact_bad=None,
                cap_compact: int = 0, hit_x=None, hit_y=None, hit_z=None) -> sst_output:
    return sst_output(_ptr(strip_adc), _ptr(chan_off), _ptr(chan_len), _ptr(seed_idx), cap_seeds,
                      cap_clusters, cap_adc, _ptr(n_clusters), _ptr(cl_module), _ptr(cl_first),
                      _ptr(cl_width), _ptr(cl_charge), _ptr(cl_bary), _ptr(cl_adc_off), _ptr(cl_snr),
                      _ptr(cl_adc), _ptr(dev_status), _ptr(compact_strip), _ptr(compact_adc),
                      _ptr(compact_noise), _ptr(compact_gain), _ptr(compact_bad), cap_compact,
                      _ptr(hit_x), _ptr(hit_y), _ptr(hit_z))


def sst_unpack_cluster(ctx, raw, fed_offsets, thresholds, out: sst_output, stream: int = 0):
    """raw / fed_offsets: DEVICE tensors; stream: cudaStream_t as int.  Does not synchronise."""
    thr = thresholds if isinstance(thresholds, sst_thresholds) else sst_thresholds(*map(float, thresholds))
    rc = load().sst_unpack_cluster(ctx, _ptr(raw), _ptr(fed_offsets), C.byref(thr), C.byref(out),
                                   C.c_void_p(stream))
    _check(ctx, rc, "sst_unpack_cluster")


def sst_unpack_cluster_noalloc(ctx, raw, fed_offsets, thresholds, out: sst_output, stream: int = 0):
    """sst_unpack_cluster for callers that must not allocate device memory while they run (real-time
    loops with a fixed memory budget, hosts whose own allocator owns the GPU): the kernels' scratch is
    the library's built-in 32 MiB array, one per GPU and shared by all calls, so calls that could
    overlap on the GPU must be ordered by the caller.  Raises SSTError (SST_ERR_TOO_LARGE) for a
    context whose one-event scratch does not fit.  Same arguments and results as sst_unpack_cluster;
    does not synchronise."""
    thr = thresholds if isinstance(thresholds, sst_thresholds) else sst_thresholds(*map(float, thresholds))
    rc = load().sst_unpack_cluster_noalloc(ctx, _ptr(raw), _ptr(fed_offsets), C.byref(thr), C.byref(out),
                                           C.c_void_p(stream))
    _check(ctx, rc, "sst_unpack_cluster_noalloc")


class Batch:
    """Marshalled arguments of sst_unpack_cluster_batch, built once and reused every step."""

    def __init__(self, raws, fed_offsets, thresholds, outs, streams):
        n = len(raws)
        self.n = n
        self.raw = (C.c_void_p * n)(*[_ptr(r) for r in raws])
        self.fo = (C.c_void_p * n)(*[_ptr(f) for f in fed_offsets])
        self.outs = (sst_output * n)(*outs)
        self.streams = (C.c_void_p * len(streams))(*streams)
        self.n_streams = len(streams)
        self.thr = thresholds if isinstance(thresholds, sst_thresholds) else sst_thresholds(*map(float, thresholds))


def sst_unpack_cluster_batch(ctx, batch: Batch):
    """Enqueue batch.n events, event e on batch.streams[e % n_streams].  Does not synchronise."""
    rc = load().sst_unpack_cluster_batch(ctx, batch.n, batch.raw, batch.fo, C.byref(batch.thr), batch.outs,
                                         batch.streams, batch.n_streams)
    _check(ctx, rc, "sst_unpack_cluster_batch")


def sst_unpack_cluster_host(ctx, raw, raw_bytes: int, fed_offsets, thresholds, out: sst_output,
                            stream: int = 0):
    """HOST buffers in and out (see sst.h); returns after the stream has completed."""
    thr = thresholds if isinstance(thresholds, sst_thresholds) else sst_thresholds(*map(float, thresholds))
    rc = load().sst_unpack_cluster_host(ctx, _ptr(raw), raw_bytes, _ptr(fed_offsets), C.byref(thr),
                                        C.byref(out), C.c_void_p(stream))
    _check(ctx, rc, "sst_unpack_cluster_host")


class HostBatch:
    """Marshalled arguments of sst_unpack_cluster_host_batch (HOST buffers), built once."""

    def __init__(self, raws, raw_bytes, fed_offsets, thresholds, outs, streams):
        n = len(raws)
        self.n = n
        self.keep = (list(raws), list(fed_offsets), list(outs))
        self.raw = (C.c_void_p * n)(*[_ptr(r) for r in raws])
        self.raw_bytes = (C.c_uint32 * n)(*[int(x) for x in raw_bytes])
        self.fo = (C.c_void_p * n)(*[_ptr(f) for f in fed_offsets])
        self.outs = (sst_output * n)(*outs)
        self.streams = (C.c_void_p * len(streams))(*streams)
        self.n_streams = len(streams)
        self.thr = thresholds if isinstance(thresholds, sst_thresholds) else sst_thresholds(*map(float, thresholds))


def sst_unpack_cluster_host_batch(ctx, batch: HostBatch):
    """batch.n events with HOST buffers, chunked over batch.streams; returns when all are done."""
    rc = load().sst_unpack_cluster_host_batch(ctx, batch.n, batch.raw, batch.raw_bytes, batch.fo, C.byref(batch.thr),
                                              batch.outs, batch.streams, batch.n_streams)
    _check(ctx, rc, "sst_unpack_cluster_host_batch")


class sst_packed_result(C.Structure):
    _fields_ = [("block", C.c_void_p), ("block_bytes", C.c_uint64), ("view", sst_output)]


class PackedBatch:
    """Marshalled arguments of sst_unpack_cluster_host_packed: one HOST result block per event."""

    def __init__(self, raws, raw_bytes, fed_offsets, thresholds, cap_clusters, cap_adc, blocks, streams):
        n = len(raws)
        self.n = n
        self.keep = (list(raws), list(fed_offsets), list(blocks))
        self.raw = (C.c_void_p * n)(*[_ptr(r) for r in raws])
        self.raw_bytes = (C.c_uint32 * n)(*[int(x) for x in raw_bytes])
        self.fo = (C.c_void_p * n)(*[_ptr(f) for f in fed_offsets])
        self.cap_clusters, self.cap_adc = int(cap_clusters), int(cap_adc)
        self.results = (sst_packed_result * n)()
        for i, blk in enumerate(blocks):
            self.results[i].block = _ptr(blk)
            self.results[i].block_bytes = int(blk.nbytes if hasattr(blk, "nbytes") else blk.numel() * blk.element_size())
        self.streams = (C.c_void_p * len(streams))(*streams)
        self.n_streams = len(streams)
        self.thr = thresholds if isinstance(thresholds, sst_thresholds) else sst_thresholds(*map(float, thresholds))

    def view(self, i: int):
        """numpy views of event i's arrays inside its block (valid after the call)."""
        import numpy as np
        r = self.results[i]
        blk = self.keep[2][i]
        a = blk.numpy() if hasattr(blk, "numpy") and not isinstance(blk, np.ndarray) else blk
        a = a.view(np.uint8).reshape(-1)
        st = a[:32].view(np.uint32)
        k = int(a[32:36].view(np.uint32)[0])
        K = min(int(st[ST_N_CLUSTERS]), self.cap_clusters)
        na = min(int(st[ST_N_ADC]), self.cap_adc)
        o = 64
        out = {"status": st, "n_clusters": k}
        for name, dt, w in (("cl_module", np.uint32, 4), ("cl_charge", np.int32, 4), ("cl_bary", np.float32, 4),
                            ("cl_adc_off", np.uint32, 4), ("cl_first", np.uint16, 2), ("cl_width", np.uint16, 2)):
            out[name] = a[o:o + w * K].view(dt)[:k]
            o += w * K
        out["cl_adc"] = a[o:o + na]
        return out


def sst_unpack_cluster_host_packed(ctx, batch: PackedBatch):
    """batch.n events with HOST buffers and packed HOST result blocks; returns when all are done."""
    rc = load().sst_unpack_cluster_host_packed(ctx, batch.n, batch.raw, batch.raw_bytes, batch.fo, C.byref(batch.thr),
                                               batch.cap_clusters, batch.cap_adc, batch.results, batch.streams,
                                               batch.n_streams)
    _check(ctx, rc, "sst_unpack_cluster_host_packed")


def sst_event_alloc(ctx, nbytes: int, stream: int = 0) -> int:
    p = C.c_void_p()
    _check(ctx, load().sst_event_alloc(ctx, nbytes, C.c_void_p(stream), C.byref(p)), "sst_event_alloc")
    return p.value


def sst_event_free(ctx, ptr: int, stream: int = 0):
    _check(ctx, load().sst_event_free(ctx, C.c_void_p(ptr), C.c_void_p(stream)), "sst_event_free")


def sst_event_upload(ctx, raw, raw_bytes: int, fed_offsets, stream: int = 0):
    """HOST (pinned) raw / fed_offsets -> pooled device buffers on `stream`; returns the two
    device pointers (ints).  Free both with sst_event_free."""
    d_raw, d_fo = C.c_void_p(), C.c_void_p()
    rc = load().sst_event_upload(ctx, _ptr(raw), raw_bytes, _ptr(fed_offsets), C.c_void_p(stream),
                                 C.byref(d_raw), C.byref(d_fo))
    _check(ctx, rc, "sst_event_upload")
    return d_raw.value, d_fo.value


def sst_event_download(ctx, dst, src: int, nbytes: int, stream: int = 0):
    """DEVICE pointer `src` (int) -> HOST buffer `dst` (pinned tensor / numpy array) on `stream`;
    does not synchronise."""
    _check(ctx, load().sst_event_download(ctx, _ptr(dst), C.c_void_p(src), nbytes, C.c_void_p(stream)),
           "sst_event_download")


def sst_destroy(ctx):
    _check(None, load().sst_destroy(ctx), "sst_destroy")


def sst_get_info(ctx) -> dict:
    info = sst_info()
    _check(ctx, load().sst_get_info(ctx, C.byref(info)), "sst_get_info")
    return {k: getattr(info, k) for k, _ in sst_info._fields_}


TRACE_WORDS = 32


def sst_trace_read(ctx, stream: int):
    """The stream's 32 trace words (include/sst.h) as a list; waits for the stream."""
    out = (C.c_uint64 * TRACE_WORDS)()
    _check(ctx, load().sst_trace_read(ctx, stream, out), "sst_trace_read")
    return list(out)
