"""Seeded synthetic inputs for the strip-tracker unpack + clustering path.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's
tests/bench.  It holds none of the method's arithmetic (no decode, no threshold
tests, no clustering): it draws a module map, a calibration and events, applies the
detector-side zero suppression and *encodes* the raw FED byte stream.  The paper's
own input (a simulated CMS TTBar PU70 sample, section 2) is not
available; these events stand in for it with the shapes BASELINE.json's configs give
(96 channels x 256 strips per FED, section 2).

Raw format (BASELINE.json config 0; reading s1-s3): per FED 96 channels
back to back; each channel is a little-endian uint16 payload length L followed by L
bytes of runs ``(uint8 first strip, uint8 run length, run-length x uint8 ADC)``; a run
length byte of 0 encodes 256; every FED is zero-padded to a multiple of 16 bytes.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Iterable, List, Optional, Sequence, Tuple

import numpy as np

N_CHAN = 96      # optical channels per FED
N_STRIP = 256    # strips per channel
FED_STRIPS = N_CHAN * N_STRIP
FED_ALIGN = 16   # reading s3: FED payloads padded to 16 bytes

TAG_MODULES, TAG_CALIB, TAG_EVENT = 1, 2, 3


def _rng(tag: int, seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([tag, seed])))


# --------------------------------------------------------------------------------------
# configs of BASELINE.json
# --------------------------------------------------------------------------------------
@dataclass(frozen=True)
class SynthConfig:
    name: str
    n_feds: int
    occupancy: float
    geom_p: float
    width_cap: int
    bad_frac: float
    saturate_frac: float = 0.0     # config 4: fraction of true clusters whose peak is set to 254/255
    empty_chan_frac: float = 0.0   # config 4: channels forced empty
    full_chan_frac: float = 0.0    # config 4: channels forced fully occupied
    thresholds: Tuple[Tuple[float, float, float], ...] = ((2.0, 3.0, 5.0),)
    event_seeds: Tuple[int, ...] = (1,)


CONFIGS = {
    0: SynthConfig("tiny", 24, 0.01, 0.5, 8, 0.005),
    1: SynthConfig("full_pu50", 440, 0.02, 0.5, 8, 0.005),
    2: SynthConfig("full_pu200", 440, 0.06, 0.35, 16, 0.01),
    3: SynthConfig("multi_event", 440, 0.02, 0.5, 8, 0.005, event_seeds=tuple(range(1, 65))),
    4: SynthConfig("stress", 440, 0.15, 0.5, 8, 0.02, saturate_frac=0.05, empty_chan_frac=0.01,
                   full_chan_frac=0.005,
                   thresholds=((2.0, 3.0, 5.0), (1.5, 2.5, 4.0), (3.0, 5.0, 8.0))),
}


# --------------------------------------------------------------------------------------
# module map and calibration (shared by every event of every config)
# --------------------------------------------------------------------------------------
def make_module_map(n_feds: int, seed: int = 1) -> np.ndarray:
    """chan_module[n_feds*96]: module id of every channel; modules are 2 or 3 consecutive
    channels, never cross a FED, ids ascend in channel order (BASELINE.json config 0)."""
    rng = _rng(TAG_MODULES, seed)
    out = np.empty(n_feds * N_CHAN, dtype=np.uint32)
    mod = 0
    for f in range(n_feds):
        c = 0
        while c < N_CHAN:
            rem = N_CHAN - c
            if rem <= 3:
                w = rem
            elif rem == 4:
                w = 2
            else:
                w = 2 + int(rng.integers(0, 2))
            out[f * N_CHAN + c: f * N_CHAN + c + w] = mod
            mod += 1
            c += w
    return out


@dataclass
class Calibration:
    n_feds: int
    gain: np.ndarray         # float32 [N]
    noise: np.ndarray        # float32 [N]
    bad: np.ndarray          # uint8   [N]
    chan_module: np.ndarray  # uint32  [n_feds*96]

    @property
    def n_strips(self) -> int:
        return self.n_feds * FED_STRIPS


def make_calibration(n_feds: int, bad_frac: float, seed: int = 1) -> Calibration:
    n = n_feds * FED_STRIPS
    rng = _rng(TAG_CALIB, seed)
    noise = (3.0 + 3.0 * rng.random(n, dtype=np.float32)).astype(np.float32)
    noise = np.minimum(noise, np.nextafter(np.float32(6.0), np.float32(0.0))).astype(np.float32)
    gain = np.clip(rng.normal(1.0, 0.05, n), 0.8, 1.2).astype(np.float32)
    # the same uniform draws for every bad fraction => nested bad-strip sets across configs
    bad = (rng.random(n) < bad_frac).astype(np.uint8)
    return Calibration(n_feds, gain, noise, bad, make_module_map(n_feds, seed))


TAG_GEOM = 4


def make_geometry(chan_module: np.ndarray, seed: int = 1) -> np.ndarray:
    """Synthetic module geometry, float32 [n_modules, 6] = {pitch, u0, r, cos phi, sin phi, z}
    (reading s23; the paper names the hit conversion as its next step, and
    gives no geometry).  Module ids must be 0..n_modules-1 (as make_module_map gives them).  Pitch
    80-200 um, the sensor centred on u = 0, radii of a barrel-like tracker (20-110 cm), any azimuth,
    |z| < 110 cm; lengths in cm."""
    cm = np.asarray(chan_module, np.int64)
    n_mod = int(cm.max()) + 1
    n_strips = np.bincount(cm, minlength=n_mod).astype(np.float64) * N_STRIP
    rng = _rng(TAG_GEOM, seed)
    pitch = rng.uniform(0.008, 0.020, n_mod)
    phi = rng.uniform(-np.pi, np.pi, n_mod)
    r = rng.choice(np.array([25.5, 33.9, 41.9, 49.8, 60.8, 69.2, 78.0, 86.8, 96.5, 108.0]), n_mod)
    z = rng.uniform(-110.0, 110.0, n_mod)
    u0 = -pitch * (n_strips - 1.0) / 2.0
    return np.stack([pitch, u0, r, np.cos(phi), np.sin(phi), z], axis=1).astype(np.float32)


# --------------------------------------------------------------------------------------
# raw encoder
# --------------------------------------------------------------------------------------
def encode_dense(z: np.ndarray, n_feds: int, keep: Optional[np.ndarray] = None
                 ) -> Tuple[np.ndarray, np.ndarray]:
    """Encode a dense strip array into the raw FED byte stream.

    ``z`` uint8 [n_feds*96*256]; ``keep`` bool mask of recorded strips (default z > 0).
    Runs are the maximal runs of kept strips inside a channel; a 256-strip run gets
    length byte 0.  Returns (raw uint8, fed_offsets uint32 [n_feds+1])."""
    z = np.ascontiguousarray(z, dtype=np.uint8)
    n_chan = n_feds * N_CHAN
    assert z.size == n_chan * N_STRIP
    k = (z > 0) if keep is None else np.asarray(keep, dtype=bool).reshape(-1)
    k2 = k.reshape(n_chan, N_STRIP)
    prev = np.zeros_like(k2)
    prev[:, 1:] = k2[:, :-1]
    nxt = np.zeros_like(k2)
    nxt[:, :-1] = k2[:, 1:]
    starts = np.flatnonzero((k2 & ~prev).reshape(-1))          # global strip ids, ascending
    ends = np.flatnonzero((k2 & ~nxt).reshape(-1))
    lens = (ends - starts + 1).astype(np.int64)
    run_chan = starts // N_STRIP
    run_bytes = 2 + lens
    chan_len = np.bincount(run_chan, weights=run_bytes, minlength=n_chan).astype(np.int64)
    chan_bytes = 2 + chan_len
    fed_bytes = chan_bytes.reshape(n_feds, N_CHAN).sum(axis=1)
    fed_padded = (fed_bytes + FED_ALIGN - 1) // FED_ALIGN * FED_ALIGN
    fed_offsets = np.zeros(n_feds + 1, dtype=np.int64)
    np.cumsum(fed_padded, out=fed_offsets[1:])
    # channel base = FED base + bytes of the earlier channels of the same FED
    cb = chan_bytes.reshape(n_feds, N_CHAN)
    within = np.cumsum(cb, axis=1) - cb
    chan_base = (fed_offsets[:-1, None] + within).reshape(-1)
    # run base = channel base + 2 + bytes of the earlier runs of the same channel
    run_cum = np.cumsum(run_bytes) - run_bytes
    chan_run_cum0 = np.cumsum(chan_len) - chan_len            # run bytes in all earlier channels
    run_base = chan_base[run_chan] + 2 + (run_cum - chan_run_cum0[run_chan])
    raw = np.zeros(int(fed_offsets[-1]), dtype=np.uint8)
    raw[chan_base] = (chan_len & 0xFF).astype(np.uint8)
    raw[chan_base + 1] = (chan_len >> 8).astype(np.uint8)
    raw[run_base] = (starts % N_STRIP).astype(np.uint8)
    raw[run_base + 1] = (lens & 0xFF).astype(np.uint8)        # 256 -> 0
    kept = np.flatnonzero(k)
    run_of = np.repeat(np.arange(starts.size), lens)
    raw[run_base[run_of] + 2 + (kept - starts[run_of])] = z[kept]
    assert fed_offsets[-1] < 2 ** 32
    return raw, fed_offsets.astype(np.uint32)


def assemble_feds(feds: Sequence[Sequence[bytes]], pad: bool = True
                  ) -> Tuple[np.ndarray, np.ndarray]:
    """Build raw from explicit per-channel byte strings (each INCLUDING its 2 length
    bytes).  Hand-built and malformed test inputs use this; nothing is validated."""
    chunks: List[bytes] = []
    offs = [0]
    pos = 0
    for chans in feds:
        b = b"".join(chans)
        if pad and len(b) % FED_ALIGN:
            b += bytes(FED_ALIGN - len(b) % FED_ALIGN)
        chunks.append(b)
        pos += len(b)
        offs.append(pos)
    raw = np.frombuffer(b"".join(chunks), dtype=np.uint8).copy()
    return raw, np.asarray(offs, dtype=np.uint32)


def channel_bytes(runs: Iterable[Tuple[int, Sequence[int]]]) -> bytes:
    """One channel's bytes (length prefix + runs) from [(first, [adc, ...]), ...]."""
    body = bytearray()
    for first, adcs in runs:
        body += bytes([first & 0xFF, len(adcs) & 0xFF]) + bytes(int(a) & 0xFF for a in adcs)
    return len(body).to_bytes(2, "little") + bytes(body)


EMPTY_CHANNEL = b"\x00\x00"


# --------------------------------------------------------------------------------------
# events
# --------------------------------------------------------------------------------------
@dataclass
class Event:
    n_feds: int
    raw: np.ndarray          # uint8
    fed_offsets: np.ndarray  # uint32 [n_feds+1]
    z: np.ndarray            # uint8 [N]: the dense array the encoder started from
    seed: int = 0
    meta: dict = field(default_factory=dict)


def make_event(cfg: SynthConfig, calib: Calibration, seed: int) -> Event:
    """One synthetic event: true clusters + per-strip Gaussian noise, digitised to uint8,
    zero-suppressed at adc >= 2*noise, encoded (BASELINE.json configs 0-4)."""
    n = calib.n_strips
    n_chan = calib.n_feds * N_CHAN
    rng = _rng(TAG_EVENT, seed)
    p, cap = cfg.geom_p, cfg.width_cap
    # E[min(cap, G)], G geometric on 1,2,...
    mean_w = sum((1 - p) ** (j - 1) for j in range(1, cap + 1))
    k = int(round(cfg.occupancy * n / mean_w))
    width = np.minimum(cap, rng.geometric(p, k)).astype(np.int64)
    start = rng.integers(0, n, k, dtype=np.int64)
    charge = rng.lognormal(5.3, 0.4, k)
    cl_of = np.repeat(np.arange(k), width)
    i_in = np.arange(cl_of.size) - np.repeat(np.cumsum(width) - width, width)
    w_rep = width[cl_of]
    tri = np.minimum(i_in + 1, w_rep - i_in).astype(np.float64)
    tri_sum = np.bincount(cl_of, weights=tri, minlength=k)
    strip = start[cl_of] + i_in
    chan_mod = calib.chan_module.astype(np.int64)
    inside = strip < n
    strip_c = np.minimum(strip, n - 1)
    inside &= chan_mod[strip_c // N_STRIP] == chan_mod[start[cl_of] // N_STRIP]
    signal = np.bincount(strip_c[inside], weights=(charge[cl_of] * tri / tri_sum[cl_of])[inside],
                         minlength=n)
    full = np.zeros(n_chan, dtype=bool)
    empty = np.zeros(n_chan, dtype=bool)
    if cfg.full_chan_frac > 0 or cfg.empty_chan_frac > 0:
        u = rng.random(n_chan)
        empty = u < cfg.empty_chan_frac
        full = (u >= cfg.empty_chan_frac) & (u < cfg.empty_chan_frac + cfg.full_chan_frac)
        signal += np.repeat(full, N_STRIP) * 60.0
    x = signal + rng.standard_normal(n) * calib.noise
    adc = np.clip(np.floor(x + 0.5), 0, 255).astype(np.uint8)
    if cfg.saturate_frac > 0:
        sat = rng.random(k) < cfg.saturate_frac
        val = np.where(rng.random(k) < 0.5, 254, 255).astype(np.uint8)
        peak = start + (width - 1) // 2
        ok = sat & (peak < n)
        ok &= chan_mod[np.minimum(peak, n - 1) // N_STRIP] == chan_mod[start // N_STRIP]
        adc[peak[ok]] = val[ok]
    keep = adc.astype(np.float32) >= np.float32(2.0) * calib.noise
    keep &= adc > 0
    if full.any():
        keep |= np.repeat(full, N_STRIP)
        adc = np.where(np.repeat(full, N_STRIP) & (adc == 0), 1, adc).astype(np.uint8)
    if empty.any():
        keep &= ~np.repeat(empty, N_STRIP)
    z = np.where(keep, adc, 0).astype(np.uint8)
    raw, fed_offsets = encode_dense(z, calib.n_feds, keep)
    meta = {"true_clusters": k, "present": int(keep.sum()), "raw_bytes": int(raw.size),
            "full_channels": int(full.sum()), "empty_channels": int(empty.sum())}
    return Event(calib.n_feds, raw, fed_offsets, z, seed, meta)


def make_config(config_id: int, n_feds: Optional[int] = None, event_seeds: Optional[Sequence[int]] = None
                ) -> Tuple[SynthConfig, Calibration, List[Event]]:
    """Calibration + events of a BASELINE.json config (optionally at fewer FEDs/events)."""
    cfg = CONFIGS[config_id]
    nf = cfg.n_feds if n_feds is None else n_feds
    calib = make_calibration(nf, cfg.bad_frac, seed=1)
    seeds = cfg.event_seeds if event_seeds is None else tuple(event_seeds)
    return cfg, calib, [make_event(cfg, calib, s) for s in seeds]
