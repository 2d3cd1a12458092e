"""Pins of the oracle's FED walk + decode (oracle/sst_oracle.c: sst_oracle_unpack).

Pinned by: (i) the encode -> decode round trip against the dense array the generator started
from (the encoder shares no code with the decoder); (ii) hand-typed byte strings with
hand-typed expectations; (iii) malformed inputs (readings s2b, s3b).
Format: section 2 (96 channels x 256 strips, CSR-like) + BASELINE.json config 0.
"""
import numpy as np
import pytest

from paper_2101_11489_b200 import synth
from tests import cases

E = synth.EMPTY_CHANNEL


def fed_with(chans: dict, n=96):
    return [chans.get(c, E) for c in range(n)]


def test_round_trip_config0(oracle):
    cfg, cal, evs = synth.make_config(0)
    ev = evs[0]
    off, ln, adc, st = oracle.unpack(ev.raw, ev.fed_offsets, cal.n_feds)
    assert np.array_equal(adc, ev.z)
    assert st[0] == 0 and st[1] == 0 and st[4] == 0
    # sum of run lengths = number of recorded strips; lengths chain to the FED ends
    assert int(ln.sum()) == ev.raw.size - 2 * ln.size - int(_pad_bytes(ev, ln))
    assert int(np.count_nonzero(adc)) == ev.meta["present"]
    # channel map: off[c+1] = off[c] + len[c] + 2 inside a FED, off[first] = fed_offset + 2
    o = off.reshape(cal.n_feds, 96).astype(np.int64)
    l = ln.reshape(cal.n_feds, 96).astype(np.int64)
    assert np.array_equal(o[:, 0], ev.fed_offsets[:-1].astype(np.int64) + 2)
    assert np.array_equal(o[:, 1:], o[:, :-1] + l[:, :-1] + 2)


def _pad_bytes(ev, ln):
    used = (ln.reshape(ev.n_feds, 96).astype(np.int64) + 2).sum(axis=1)
    return (np.diff(ev.fed_offsets.astype(np.int64)) - used).sum()


@pytest.mark.parametrize("cid,nf", [(2, 6), (4, 12)])
def test_round_trip_dense_configs(oracle, cid, nf):
    cfg, cal, evs = synth.make_config(cid, n_feds=nf)
    ev = evs[0]
    _, _, adc, st = oracle.unpack(ev.raw, ev.fed_offsets, nf)
    assert np.array_equal(adc, ev.z)
    assert st[1] == 0


def test_hand_built_byte_strings(oracle):
    chans = {
        0: bytes.fromhex("0000"),                                  # empty channel
        1: bytes.fromhex("0300") + bytes([100, 1, 40]),            # strip 100 = 40
        2: bytes.fromhex("0400") + bytes([254, 2, 7, 9]),          # run ending at strip 255
        3: bytes.fromhex("0300") + bytes([255, 1, 11]),            # first = 255, len = 1
        4: bytes.fromhex("0700") + bytes([10, 1, 5, 11, 2, 6, 7]),  # abutting runs 10 | 11-12
        5: (258).to_bytes(2, "little") + bytes([0, 0]) + bytes([60] * 256),   # full channel, len byte 0
        6: (260).to_bytes(2, "little") + bytes([0, 255]) + bytes([9] * 255) + bytes([255, 1, 8]),  # 255 + 1
    }
    raw, fo = synth.assemble_feds([fed_with(chans)])
    assert raw.size % 16 == 0
    off, ln, adc, st = oracle.unpack(raw, fo, 1)
    a = adc.reshape(96, 256)
    exp = np.zeros((96, 256), np.uint8)
    exp[1, 100] = 40
    exp[2, 254], exp[2, 255] = 7, 9
    exp[3, 255] = 11
    exp[4, 10], exp[4, 11], exp[4, 12] = 5, 6, 7
    exp[5, :] = 60
    exp[6, :255] = 9
    exp[6, 255] = 8
    assert np.array_equal(a, exp)
    assert list(ln[:7]) == [0, 3, 4, 3, 7, 258, 260]
    assert off[0] == 2 and off[1] == 4 and off[2] == 9
    assert st[0] == 0 and st[1] == 0


def test_all_empty_fed(oracle):
    raw, fo = synth.assemble_feds([fed_with({})])
    assert raw.size == 192
    off, ln, adc, st = oracle.unpack(raw, fo, 1)
    assert not adc.any() and not ln.any() and st[0] == 0
    assert np.array_equal(off, 2 + 2 * np.arange(96))


@pytest.mark.parametrize("name,body", [
    ("first+len>256", bytes([250, 10]) + bytes([1] * 10)),
    ("descending first", bytes([20, 1, 5, 10, 1, 6])),
    ("overlap", bytes([20, 2, 5, 6, 21, 1, 7])),
    ("L one byte short", bytes([20, 3, 5, 6])),                # header says 3 ADCs, payload has 2
    ("L one byte long", bytes([20, 1, 5, 9])),                 # trailing byte cannot hold a header
    ("len0 with first>0", bytes([1, 0]) + bytes([3] * 255)),   # 256 strips starting at 1
])
def test_malformed_channel_is_empty_and_counted(oracle, name, body):
    good = synth.channel_bytes([(7, [33, 34])])
    bad = len(body).to_bytes(2, "little") + body
    raw, fo = synth.assemble_feds([fed_with({0: good, 1: bad, 2: good})])
    off, ln, adc, st = oracle.unpack(raw, fo, 1)
    a = adc.reshape(96, 256)
    assert not a[1].any(), name
    assert a[0, 7] == 33 and a[2, 8] == 34          # neighbours unaffected: chain uses L only
    assert st[1] == 1 and st[0] & oracle.FLAG_MALFORMED
    assert ln[1] == len(body)


def test_chain_overrun(oracle):
    good = synth.channel_bytes([(7, [33])])
    # channel 2 claims 4000 bytes: passes the FED end -> channels 2.. are empty, FED flagged
    over = (4000).to_bytes(2, "little") + bytes([1, 1, 9])
    raw, fo = synth.assemble_feds([fed_with({0: good, 1: good, 2: over, 3: good}),
                                   fed_with({5: good})])
    off, ln, adc, st = oracle.unpack(raw, fo, 2)
    a = adc.reshape(2 * 96, 256)
    assert a[0, 7] == 33 and a[1, 7] == 33
    assert not a[2:96].any()
    assert a[96 + 5, 7] == 33                       # the next FED is unaffected
    assert st[4] == 1 and st[0] & oracle.FLAG_OVERRUN
    assert np.all(off[2:96] == fo[1]) and not ln[2:96].any()


def test_truncated_fed_and_bad_offsets(oracle):
    good = synth.channel_bytes([(7, [33])])
    raw, fo = synth.assemble_feds([fed_with({0: good})])
    fo2 = fo.copy()
    fo2[1] = 3 + 2                                   # FED ends inside channel 1's length bytes
    _, ln, adc, st = oracle.unpack(raw, fo2, 1)
    assert adc.reshape(96, 256)[0, 7] == 33 and st[4] == 1
    fo3 = np.array([16, 0], np.uint32)               # end < start
    _, _, adc, st = oracle.unpack(raw, fo3, 1)
    assert not adc.any() and st[4] == 1
    fo4 = np.array([0, raw.size + 16], np.uint32)    # end beyond the buffer
    _, _, adc, st = oracle.unpack(raw, fo4, 1)
    assert not adc.any() and st[4] == 1


def test_offsets_that_step_back_are_flagged_and_empty(oracle):
    """Reading s3c: a FED whose start lies below an earlier entry of fed_offsets is flagged and
    empty, so decoded FEDs never overlap.  Offsets [0, n, 0, n]: FED 0 decodes, FED 1 has end <
    start, FED 2 would re-read FED 0's bytes and is refused."""
    good = synth.channel_bytes([(7, [33])])
    raw, fo = synth.assemble_feds([fed_with({0: good})])
    n = int(fo[1])
    off, ln, adc, st = oracle.unpack(raw, np.array([0, n, 0, n], np.uint32), 3)
    a = adc.reshape(3 * 96, 256)
    assert a[0, 7] == 33 and not a[96:].any()
    assert st[4] == 2 and st[0] & oracle.FLAG_OVERRUN
    assert np.all(off[96:192] == n) and np.all(off[192:] == 0) and not ln[96:].any()   # (start as given, 0)
    # [0, n, n/2.., 2n] with the middle FED starting inside FED 0: refused; a later FED that starts
    # at or above every earlier offset is decoded again
    raw2 = np.concatenate([raw, raw])
    off, ln, adc, st = oracle.unpack(raw2, np.array([0, n, 16, n, 2 * n], np.uint32), 4)
    a = adc.reshape(4 * 96, 256)
    assert a[0, 7] == 33 and not a[96:3 * 96].any() and a[3 * 96, 7] == 33
    assert st[4] == 2


def test_worked_example_dense_holds_bad_strips(oracle):
    doc = cases.load_worked_examples()
    w5 = next(c for c in doc["cases"] if c["id"] == "W5")
    cs = cases.worked_case(doc, w5)
    _, _, adc, _ = oracle.unpack(cs.raw, cs.fed_offsets, 1)
    assert adc[256 + 145] == 50 and adc[256 + 155] == 50
    assert np.array_equal(adc, cs.z)
