"""The seeded generator: determinism, format, and the workload shape DESIGN.md section 4 states."""
import numpy as np

from paper_2101_11489_b200 import synth


def test_module_map_rules():
    m = synth.make_module_map(24)
    assert m.size == 24 * 96 and m[0] == 0
    assert np.all(np.diff(m.astype(np.int64)) >= 0) and np.all(np.diff(m.astype(np.int64)) <= 1)
    sizes = np.bincount(m)
    assert set(sizes.tolist()) <= {2, 3}
    # a module never crosses a FED
    assert np.all(m[96::96] != m[95:-1:96])


def test_deterministic_and_shaped_like_config0():
    cfg, cal, evs = synth.make_config(0)
    cfg2, cal2, evs2 = synth.make_config(0)
    ev = evs[0]
    assert np.array_equal(ev.raw, evs2[0].raw) and np.array_equal(cal.gain, cal2.gain)
    assert cal.noise.dtype == np.float32 and cal.noise.min() >= 3.0 and cal.noise.max() < 6.0
    assert cal.gain.min() >= np.float32(0.8) and cal.gain.max() <= np.float32(1.2)
    assert 0.003 < cal.bad.mean() < 0.007
    assert ev.fed_offsets[0] == 0 and np.all(ev.fed_offsets % 16 == 0) and ev.fed_offsets[-1] == ev.raw.size
    occ = ev.meta["present"] / cal.n_strips
    assert 0.028 < occ < 0.037                     # ~1 % signal + ~2.3 % noise survivors of the 2 sigma cut
    assert 50_000 < ev.raw.size < 62_000


def test_nested_bad_sets_and_shared_calibration():
    a = synth.make_calibration(4, 0.005)
    b = synth.make_calibration(4, 0.02)
    assert np.array_equal(a.noise, b.noise) and np.array_equal(a.gain, b.gain)
    assert np.all(b.bad[a.bad == 1] == 1) and b.bad.sum() > a.bad.sum()


def test_config4_extras():
    cfg, cal, evs = synth.make_config(4, n_feds=40)
    ev = evs[0]
    z = ev.z.reshape(-1, 256)
    assert ev.meta["full_channels"] > 0 and ev.meta["empty_channels"] > 0
    assert int(np.all(z > 0, axis=1).sum()) >= ev.meta["full_channels"]
    assert np.any(ev.z >= 254)
    # fully occupied channels use the single-run form: length 258, header (0, 0)
    full = np.flatnonzero(np.all(z > 0, axis=1))
    raw = ev.raw
    pos_of = {}
    for f in range(40):
        p = int(ev.fed_offsets[f])
        for c in range(96):
            L = int(raw[p]) | int(raw[p + 1]) << 8
            pos_of[f * 96 + c] = (p, L)
            p += 2 + L
    for ch in full:
        p, L = pos_of[int(ch)]
        assert L == 258 and raw[p + 2] == 0 and raw[p + 3] == 0


def test_different_seeds_differ():
    cfg, cal, evs = synth.make_config(3, n_feds=2, event_seeds=(1, 2))
    assert not np.array_equal(evs[0].z, evs[1].z)
