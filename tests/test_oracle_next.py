"""Pins of the oracle functions behind SURVEY.md section 8(f) NEXT-2 (compact SoA)
and NEXT-4 (clusters -> global hit coordinates).  No GPU."""
import numpy as np
import pytest

from paper_2101_11489_b200 import synth
from tests import cases


# ------------------------------------------------------------------ compact SoA
def test_compact_hand_rows(oracle):
    """W5 of the worked examples (bad strips keep their raw ADC in the SoA): entries by hand."""
    doc = cases.load_worked_examples()
    w5 = next(c for c in doc["cases"] if c["id"] == "W5")
    cs = cases.worked_case(doc, w5)
    _, _, adc, _ = oracle.unpack(cs.raw, cs.fed_offsets, 1)
    k, c = oracle.compact(adc, cs.gain, cs.noise, cs.bad)
    # module-local strips 400..402 and 410..412 sit in channel 1 (strips 144.. of it): global = 256 + local - 256
    want_strip = [400, 401, 402, 410, 411, 412]
    assert k == 6 and c["strip"].tolist() == want_strip
    assert c["adc"].tolist() == [30, 50, 30, 9, 50, 9]
    assert c["bad"].tolist() == [0, 1, 0, 0, 1, 0]
    assert np.all(c["noise"] == np.float32(4.0)) and np.all(c["gain"] == np.float32(1.0))


@pytest.mark.parametrize("cid,nf", [(0, 24), (2, 5), (4, 5)])
def test_compact_equals_nonzero_dense_plus_gather(oracle, cid, nf):
    """Library special case: numpy flatnonzero of the dense array and a fancy-index gather of the
    calibration; and the count is the generator's number of kept strips."""
    cfg, cal, evs = synth.make_config(cid, n_feds=nf)
    ev = evs[0]
    _, _, adc, _ = oracle.unpack(ev.raw, ev.fed_offsets, nf)
    k, c = oracle.compact(adc, cal.gain, cal.noise, cal.bad)
    idx = np.flatnonzero(ev.z)
    assert k == idx.size == ev.meta["present"]
    assert np.array_equal(c["strip"], idx.astype(np.uint32))
    assert np.array_equal(c["adc"], ev.z[idx])
    assert np.array_equal(c["noise"], cal.noise[idx]) and np.array_equal(c["gain"], cal.gain[idx])
    assert np.array_equal(c["bad"], cal.bad[idx])
    assert np.all(np.diff(c["strip"].astype(np.int64)) > 0)
    # capacity: a prefix is written, the needed count is still reported
    k2, c2 = oracle.compact(adc, cal.gain, cal.noise, cal.bad, cap=100)
    assert k2 == k and np.array_equal(c2["strip"], c["strip"][:100])


def test_compact_skips_recorded_zero(oracle):
    """Reading s9: an ADC of 0 present in the raw data carries nothing."""
    chans = [synth.channel_bytes([(5, [0, 7, 0])])] + [synth.EMPTY_CHANNEL] * 95
    raw, fo = synth.assemble_feds([chans])
    _, _, adc, _ = oracle.unpack(raw, fo, 1)
    n = synth.FED_STRIPS
    k, c = oracle.compact(adc, np.ones(n, np.float32), np.ones(n, np.float32), np.zeros(n, np.uint8))
    assert k == 1 and c["strip"].tolist() == [6] and c["adc"].tolist() == [7]


# ------------------------------------------------------------------ hits
def geom_rows(rows):
    return np.asarray(rows, np.float32).reshape(-1, 6)


def test_hits_hand_values(oracle):
    """phi = 0: the sensor measures y; phi = 90 deg: it measures -x.  Values by hand."""
    g = geom_rows([[0.0078125, -1.99609375, 50.0, 1.0, 0.0, 12.5],   # 512 strips of 2^-7 cm centred: u0 = -pitch * 255.5
                   [0.02, 0.0, 30.0, 0.0, 1.0, -7.0],
                   [0.01, 0.0, 10.0, 0.6, 0.8, 1.0]])
    x, y, z = oracle.hits([0, 0, 1, 2], [255.5, 0.0, 100.0, 50.0], g)
    # module 0: bary 255.5 is the sensor centre (u = 0); bary 0 is u = u0 (all values exact in binary)
    assert (x[0], y[0], z[0]) == (50.0, 0.0, 12.5)
    assert (x[1], y[1], z[1]) == (50.0, -1.99609375, 12.5)
    # module 1: u = 2.0 -> x = -u, y = r
    assert x[2] == pytest.approx(-2.0, rel=1e-6) and y[2] == 30.0 and z[2] == -7.0
    # module 2: u = 0.5: x = 10*0.6 - 0.5*0.8 = 5.6, y = 10*0.8 + 0.5*0.6 = 8.3
    assert x[3] == pytest.approx(5.6, rel=1e-6) and y[3] == pytest.approx(8.3, rel=1e-6)


def test_hits_of_the_worked_example_barycenters(oracle):
    """W2/W3/W7 barycenters (tests/golden/worked_examples.json) through a hand-checkable geometry:
    pitch 0.01, u0 = 0, r = 100, phi = 0 -> (x, y) = (100, bary / 100)."""
    doc = cases.load_worked_examples()
    g = geom_rows([[0.01, 0.0, 100.0, 1.0, 0.0, 0.0]])
    for cid in ("W2", "W3", "W7"):
        case = next(c for c in doc["cases"] if c["id"] == cid)
        b = np.float32(case["clusters"][0]["bary"])
        x, y, z = oracle.hits([0], [b], g)
        assert x[0] == 100.0 and z[0] == 0.0
        assert y[0] == pytest.approx(float(b) / 100.0, rel=1e-6)


def test_hits_invariants(oracle):
    """x^2 + y^2 = r^2 + u^2; one strip moves the hit by one pitch along (-sin, cos); unknown module -> NaN."""
    cfg, cal, evs = synth.make_config(0, n_feds=3)
    geom = synth.make_geometry(cal.chan_module)
    r = oracle.run(evs[0].raw, evs[0].fed_offsets, 3, cal.gain, cal.noise, cal.bad, cal.chan_module, (2, 3, 5))
    x, y, z = oracle.hits(r.cl_module, r.cl_bary, geom)
    gm = geom[r.cl_module.astype(np.int64)].astype(np.float64)
    u = gm[:, 1] + gm[:, 0] * r.cl_bary.astype(np.float64)
    np.testing.assert_allclose(x.astype(np.float64) ** 2 + y.astype(np.float64) ** 2, gm[:, 2] ** 2 + u ** 2, rtol=1e-6)
    assert np.array_equal(z, gm[:, 5].astype(np.float32))
    x1, y1, _ = oracle.hits(r.cl_module, r.cl_bary + np.float32(1.0), geom)
    np.testing.assert_allclose(x1 - x, -gm[:, 0] * gm[:, 4], atol=2e-5)
    np.testing.assert_allclose(y1 - y, gm[:, 0] * gm[:, 3], atol=2e-5)
    xn, yn, zn = oracle.hits([geom.shape[0]], [1.0], geom)
    assert np.isnan(xn[0]) and np.isnan(yn[0]) and np.isnan(zn[0])


def test_geometry_recipe():
    cm = synth.make_module_map(4)
    g = synth.make_geometry(cm)
    assert g.shape == (int(cm.max()) + 1, 6) and g.dtype == np.float32
    np.testing.assert_allclose(g[:, 3].astype(np.float64) ** 2 + g[:, 4].astype(np.float64) ** 2, 1.0, atol=1e-6)
    assert np.array_equal(g, synth.make_geometry(cm))        # seeded
