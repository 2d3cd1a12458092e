"""Device-memory plumbing around the binding: torch tensors for the buffers of one event.

Nothing here computes anything about the method; it allocates, copies and calls libsst.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Optional, Sequence

import numpy as np

from . import binding as B


@dataclass
class EventOutputs:
    tensors: Dict[str, "object"]
    out: B.sst_output
    cap_clusters: int
    cap_adc: int

    def numpy(self) -> Dict[str, np.ndarray]:
        """Synchronising read-back, trimmed to the counts the device reported."""
        t = {k: v.cpu().numpy() for k, v in self.tensors.items()}
        st = t["dev_status"]
        k = int(t["n_clusters"][0])
        overflow = bool(st[B.ST_FLAGS] & (B.FLAG_CLUSTER_CAP | B.FLAG_ADC_CAP))
        res = {"n_clusters": k, "status": st}
        for name in ("cl_module", "cl_first", "cl_width", "cl_charge", "cl_bary", "cl_adc_off", "cl_snr"):
            if name in t:
                res[name] = t[name][:k]
        na = int(res["cl_adc_off"][-1]) + int(res["cl_width"][-1]) if k else 0
        if not overflow:
            assert na == int(st[B.ST_N_ADC])
        res["cl_adc"] = t["cl_adc"][:na]
        for name in ("strip_adc", "chan_off", "chan_len"):
            if name in t:
                res[name] = t[name]
        if "seed_idx" in t:
            res["seed_idx"] = t["seed_idx"][:min(int(st[B.ST_N_SEEDS]), t["seed_idx"].size)]
        if "compact_strip" in t:
            npres = min(int(st[B.ST_N_PRESENT]), t["compact_strip"].size)
            for name in ("compact_strip", "compact_adc", "compact_noise", "compact_gain", "compact_bad"):
                res[name] = t[name][:npres]
        for name in ("hit_x", "hit_y", "hit_z"):
            if name in t:
                res[name] = t[name][:k]
        return res


class Detector:
    """A libsst context bound to one calibration (calibration is per strip, uploaded
    once and shared by all events)."""

    def __init__(self, n_feds: int, gain, noise, bad, chan_module, device: int = 0,
                 max_raw_bytes: int = 1 << 22, max_events_in_flight: int = 8, fed_strips_hint: int = 0,
                 move_mode: int = 0, trace: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise B.SSTError("no CUDA device: libsst has no CPU fallback")
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.n_feds = n_feds
        self.n_strips = n_feds * B.FED_STRIPS
        self.max_raw_bytes = int(max_raw_bytes)
        self.ctx = B.sst_create(n_feds, device, self.max_raw_bytes, max_events_in_flight, fed_strips_hint, move_mode, trace)
        B.sst_upload_calib(self.ctx, gain, noise, bad, chan_module)

    def upload_geometry(self, geom):
        B.sst_upload_geometry(self.ctx, geom)

    def close(self):
        if self.ctx is not None:
            B.sst_destroy(self.ctx)
            self.ctx = None

    def info(self) -> dict:
        return B.sst_get_info(self.ctx)

    def upload_raw(self, raw: np.ndarray, fed_offsets: np.ndarray):
        """Device copies of one event's raw bytes (padded to max_raw_bytes) and FED offsets."""
        torch = self.torch
        assert raw.size <= self.max_raw_bytes
        d_raw = torch.zeros(self.max_raw_bytes, dtype=torch.uint8, device=self.device)
        d_raw[:raw.size] = torch.from_numpy(np.ascontiguousarray(raw, np.uint8)).to(self.device)
        d_fo = torch.from_numpy(np.ascontiguousarray(fed_offsets, np.uint32).view(np.int32)).to(self.device)
        return d_raw, d_fo

    def alloc_outputs(self, cap_clusters: int, cap_adc: int, dense: bool = True, chan_map: bool = False,
                      seeds: bool = False, snr: bool = False, cap_seeds: Optional[int] = None,
                      compact: bool = False, cap_compact: Optional[int] = None, hits: bool = False) -> EventOutputs:
        torch = self.torch
        dev = self.device
        cc, ca = max(int(cap_clusters), 1), max(int(cap_adc), 1)
        t = {
            "n_clusters": torch.zeros(1, dtype=torch.int32, device=dev),
            "dev_status": torch.zeros(B.ST_WORDS, dtype=torch.int32, device=dev),
            "cl_module": torch.empty(cc, dtype=torch.int32, device=dev),
            "cl_first": torch.empty(cc, dtype=torch.int16, device=dev),
            "cl_width": torch.empty(cc, dtype=torch.int16, device=dev),
            "cl_charge": torch.empty(cc, dtype=torch.int32, device=dev),
            "cl_bary": torch.empty(cc, dtype=torch.float32, device=dev),
            "cl_adc_off": torch.empty(cc, dtype=torch.int32, device=dev),
            "cl_adc": torch.empty(ca, dtype=torch.uint8, device=dev),
        }
        if dense:
            t["strip_adc"] = torch.empty(self.n_strips, dtype=torch.uint8, device=dev)
        if chan_map:
            t["chan_off"] = torch.empty(self.n_feds * B.N_CHAN, dtype=torch.int32, device=dev)
            t["chan_len"] = torch.empty(self.n_feds * B.N_CHAN, dtype=torch.int16, device=dev)
        ncs = 0
        if seeds:
            ncs = self.n_strips if cap_seeds is None else int(cap_seeds)
            t["seed_idx"] = torch.empty(max(ncs, 1), dtype=torch.int32, device=dev)
        if snr:
            t["cl_snr"] = torch.empty(cc, dtype=torch.float32, device=dev)
        ncc = 0
        if compact:
            ncc = self.max_raw_bytes if cap_compact is None else int(cap_compact)
            m = max(ncc, 1)
            t["compact_strip"] = torch.empty(m, dtype=torch.int32, device=dev)
            t["compact_adc"] = torch.empty(m, dtype=torch.uint8, device=dev)
            t["compact_noise"] = torch.empty(m, dtype=torch.float32, device=dev)
            t["compact_gain"] = torch.empty(m, dtype=torch.float32, device=dev)
            t["compact_bad"] = torch.empty(m, dtype=torch.uint8, device=dev)
        if hits:
            for name in ("hit_x", "hit_y", "hit_z"):
                t[name] = torch.empty(cc, dtype=torch.float32, device=dev)
        out = B.make_output(cap_clusters=int(cap_clusters), cap_adc=int(cap_adc), cap_seeds=ncs, cap_compact=ncc,
                            **{k: v for k, v in t.items()})
        return EventOutputs(t, out, int(cap_clusters), int(cap_adc))

    def run(self, d_raw, d_fo, thresholds: Sequence[float], outputs: EventOutputs, stream=None):
        """Enqueue one event on `stream` (a torch.cuda.Stream; default: the current stream)."""
        st = self.torch.cuda.current_stream(self.device) if stream is None else stream
        B.sst_unpack_cluster(self.ctx, d_raw, d_fo, thresholds, outputs.out, st.cuda_stream)

    def run_noalloc(self, d_raw, d_fo, thresholds: Sequence[float], outputs: EventOutputs, stream=None):
        """The same event through sst_unpack_cluster_noalloc (scratch in the library's static array)."""
        st = self.torch.cuda.current_stream(self.device) if stream is None else stream
        B.sst_unpack_cluster_noalloc(self.ctx, d_raw, d_fo, thresholds, outputs.out, st.cuda_stream)


_FIELDS = (("strip_adc", np.uint8, "N"), ("chan_off", np.uint32, "C"), ("chan_len", np.uint16, "C"),
           ("seed_idx", np.uint32, "S"), ("cl_module", np.uint32, "K"), ("cl_first", np.uint16, "K"),
           ("cl_width", np.uint16, "K"), ("cl_charge", np.int32, "K"), ("cl_bary", np.float32, "K"),
           ("cl_adc_off", np.uint32, "K"), ("cl_snr", np.float32, "K"), ("cl_adc", np.uint8, "A"),
           ("n_clusters", np.uint32, 1), ("dev_status", np.uint32, B.ST_WORDS))


class PooledOutputs:
    """The output arrays of one event carved out of ONE block of the library's stream-ordered pool
    (sst_event_alloc; PAPER.md:41 uses a caching allocator for the same purpose), read back with
    sst_event_download."""

    def __init__(self, det: "Detector", cap_clusters: int, cap_adc: int, stream: int = 0, dense: bool = True,
                 chan_map: bool = False, seeds: bool = False, snr: bool = False, cap_seeds: Optional[int] = None):
        self.det, self.cap_clusters, self.cap_adc = det, int(cap_clusters), int(cap_adc)
        self.cap_seeds = (det.n_strips if cap_seeds is None else int(cap_seeds)) if seeds else 0
        dims = {"N": det.n_strips, "C": det.n_feds * B.N_CHAN, "S": max(self.cap_seeds, 1),
                "K": max(self.cap_clusters, 1), "A": max(self.cap_adc, 1)}
        want = {"strip_adc": dense, "chan_off": chan_map, "chan_len": chan_map, "seed_idx": seeds, "cl_snr": snr}
        self.layout, off = {}, 0
        for name, dt, dim in _FIELDS:
            if not want.get(name, True):
                continue
            n = dims[dim] if isinstance(dim, str) else dim
            self.layout[name] = (off, np.dtype(dt), n)
            off += (n * np.dtype(dt).itemsize + 255) // 256 * 256
        self.nbytes = off
        self.base = B.sst_event_alloc(det.ctx, self.nbytes, stream)
        self.out = B.make_output(cap_clusters=self.cap_clusters, cap_adc=self.cap_adc, cap_seeds=self.cap_seeds,
                                 **{k: self.base + v[0] for k, v in self.layout.items()})

    def numpy(self, stream: int = 0, skip: Sequence[str] = ()) -> Dict[str, np.ndarray]:
        """Downloads the block on `stream`, synchronises, and trims the arrays to the counts the
        device reported (same dictionary as EventOutputs.numpy() after unsigned_view)."""
        torch = self.det.torch
        host = torch.empty(self.nbytes, dtype=torch.uint8).pin_memory()
        lo = 0   # the dense array is the block's first region: skipping it shortens the copy
        if "strip_adc" in skip and "strip_adc" in self.layout:
            lo = (self.layout["strip_adc"][2] + 255) // 256 * 256
        B.sst_event_download(self.det.ctx, host.data_ptr() + lo, self.base + lo, self.nbytes - lo, stream)
        torch.cuda.synchronize(self.det.device)
        a = host.numpy()
        t = {k: a[o:o + n * dt.itemsize].view(dt) for k, (o, dt, n) in self.layout.items()}
        st = t["dev_status"]
        k = int(t["n_clusters"][0])
        res = {"n_clusters": k, "status": st}
        for name in ("cl_module", "cl_first", "cl_width", "cl_charge", "cl_bary", "cl_adc_off", "cl_snr"):
            if name in t:
                res[name] = t[name][:k]
        na = int(res["cl_adc_off"][-1]) + int(res["cl_width"][-1]) if k else 0
        res["cl_adc"] = t["cl_adc"][:na]
        for name in ("strip_adc", "chan_off", "chan_len"):
            if name in t and name not in skip:
                res[name] = t[name]
        if "seed_idx" in t:
            res["seed_idx"] = t["seed_idx"][:min(int(st[B.ST_N_SEEDS]), self.cap_seeds)]
        return res

    def free(self, stream: int = 0):
        if self.base:
            B.sst_event_free(self.det.ctx, self.base, stream)
            self.base = 0


def unsigned_view(res: Dict[str, np.ndarray]) -> Dict[str, np.ndarray]:
    """torch has no uint16/uint32 tensors everywhere; reinterpret the signed storage."""
    conv = {"cl_module": np.uint32, "cl_first": np.uint16, "cl_width": np.uint16, "cl_adc_off": np.uint32,
            "chan_off": np.uint32, "chan_len": np.uint16, "seed_idx": np.uint32, "status": np.uint32,
            "compact_strip": np.uint32}
    return {k: (v.view(conv[k]) if k in conv and isinstance(v, np.ndarray) else v) for k, v in res.items()}
