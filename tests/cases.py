"""Builders of small hand-made inputs shared by the oracle pins and the GPU parity tests.
No method arithmetic here: only placing ADC values / calibration overrides and encoding."""
from __future__ import annotations

import json
import os
from dataclasses import dataclass
from typing import Dict, Optional, Sequence

import numpy as np

from paper_2101_11489_b200 import synth

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def module_map_from_sizes(n_feds: int, sizes: Sequence[int], default: int = 2) -> np.ndarray:
    out = np.empty(n_feds * synth.N_CHAN, np.uint32)
    mod = 0
    for f in range(n_feds):
        c, i = 0, 0
        while c < synth.N_CHAN:
            w = sizes[i] if i < len(sizes) else default
            w = min(w, synth.N_CHAN - c)
            out[f * synth.N_CHAN + c: f * synth.N_CHAN + c + w] = mod
            mod += 1
            c += w
            i += 1
    return out


@dataclass
class Case:
    n_feds: int
    raw: np.ndarray
    fed_offsets: np.ndarray
    z: np.ndarray
    gain: np.ndarray
    noise: np.ndarray
    bad: np.ndarray
    chan_module: np.ndarray
    thresholds: tuple


def _g(key: str) -> int:
    c, s = key.split(":")
    return int(c) * synth.N_STRIP + int(s)


def build_case(strips: Dict[str, int], n_feds: int = 1, module_sizes=(2, 3), noise=4.0, gain=1.0,
               gain_over: Optional[Dict[str, str]] = None, noise_over: Optional[Dict[str, float]] = None,
               bad: Sequence[str] = (), full_channels: Optional[Dict[str, int]] = None,
               thresholds=(2.0, 3.0, 5.0)) -> Case:
    n = n_feds * synth.FED_STRIPS
    z = np.zeros(n, np.uint8)
    for k, v in strips.items():
        z[_g(k)] = v
    for c, v in (full_channels or {}).items():
        z[int(c) * 256:(int(c) + 1) * 256] = v
    ga = np.full(n, gain, np.float32)
    no = np.full(n, noise, np.float32)
    for k, v in (gain_over or {}).items():
        ga[_g(k)] = np.float32(float.fromhex(v) if isinstance(v, str) else v)
    for k, v in (noise_over or {}).items():
        no[_g(k)] = np.float32(float.fromhex(v) if isinstance(v, str) else v)
    bd = np.zeros(n, np.uint8)
    for k in bad:
        bd[_g(k)] = 1
    raw, fo = synth.encode_dense(z, n_feds)
    return Case(n_feds, raw, fo, z, ga, no, bd, module_map_from_sizes(n_feds, module_sizes),
                tuple(thresholds))


def load_worked_examples():
    with open(os.path.join(GOLDEN, "worked_examples.json")) as f:
        return json.load(f)


def worked_case(doc, case) -> Case:
    d = doc["defaults"]
    return build_case(case.get("strips", {}), d["n_feds"], d["module_sizes"], d["noise"], d["gain"],
                      case.get("gain"), None, case.get("bad", ()), case.get("full_channels"),
                      d["thresholds"])


def move_fed_padding(raw: np.ndarray, fo: np.ndarray, f: int, used: int, k: int):
    """FED f loses k of its trailing pad bytes, FED f+1 gains them behind its last channel: both
    keep their content, FED f gets an unaligned size and FED f+1 an unaligned start (the non-TMA
    path of the kernel).  `used` = bytes of FED f up to the end of its channel 95."""
    fo = fo.astype(np.int64)
    assert 0 < k <= fo[f + 1] - fo[f] - used and f + 2 < fo.size
    a = raw[:fo[f + 1] - k]
    b = raw[fo[f + 1]:fo[f + 2]]
    out = np.concatenate([a, b, np.zeros(k, np.uint8), raw[fo[f + 2]:]])
    fo2 = fo.copy()
    fo2[f + 1] -= k
    assert out.size == raw.size
    return out, fo2.astype(np.uint32)
