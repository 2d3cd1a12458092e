"""sst_unpack_cluster_noalloc: the one entry point of libsst that allocates nothing when called.

Some users of the library cannot let it allocate device memory once their job is running: a trigger
or data-acquisition loop whose memory budget is fixed at start-up (an allocation there can stall the
device or fail in the middle of a run), a host program whose own allocator has taken the whole GPU,
a plug-in living under a framework that forbids allocation calls.  For them the kernels' scratch is
a 32 MiB array built into the library (one per GPU, shared by every call) instead of a block from
the context's pool.  The checks here: the results are those of the pooled path (sst_unpack_cluster,
itself compared with the oracle in test_gpu_parity.py) on calls made back to back, although the
array still holds what earlier calls -- also of a context with another layout -- left in it; the
free device memory does not move across the calls; a context that does not fit is refused before
anything runs.

This file sorts last on purpose (pytest -x stops at the first failure).  It passes alone in a fresh
process, where its first call is the one that looks up the array's address, and after all the others.
"""
import numpy as np
import pytest

from paper_2101_11489_b200 import synth

pytestmark = pytest.mark.gpu

REL = 1e-6   # the tolerance of test_gpu_parity.py for barycenter and S/N; everything else bit-exact

INT_FIELDS = ("strip_adc", "chan_off", "chan_len", "seed_idx", "cl_module", "cl_first", "cl_width", "cl_charge",
              "cl_adc_off", "cl_adc", "status")


def same(a, b):
    """a: noalloc result, b: pooled-path result (dictionaries of EventOutputs.numpy())."""
    assert a["n_clusters"] == b["n_clusters"]
    for name in INT_FIELDS:
        assert np.array_equal(a[name], b[name]), name
    for name in ("cl_bary", "cl_snr"):
        np.testing.assert_allclose(a[name], b[name], rtol=REL, atol=0)
    for name in ("compact_strip", "compact_adc", "compact_noise", "compact_gain", "compact_bad", "hit_z"):
        if name in b:
            assert np.array_equal(a[name], b[name]), name
    for name in ("hit_x", "hit_y"):
        if name in b:
            np.testing.assert_allclose(a[name], b[name], rtol=REL, atol=1e-6)


class _Case:
    """A context, its events on the device and the pooled path's results for them."""

    def __init__(self, harness, cid, nf, seeds, move_mode, extras=False, hint=0):
        self.h = harness
        cfg, cal, evs = synth.make_config(cid, n_feds=nf, event_seeds=seeds)
        self.thr = cfg.thresholds[0]
        nf = cal.n_feds
        mrb = max(int(e.raw.size) for e in evs)
        self.det = harness.Detector(nf, cal.gain, cal.noise, cal.bad, cal.chan_module, max_raw_bytes=mrb,
                                    move_mode=move_mode, fed_strips_hint=hint)
        if extras:
            self.det.upload_geometry(synth.make_geometry(cal.chan_module))
        self.kw = dict(chan_map=True, seeds=True, snr=True, compact=extras, hits=extras)
        self.caps = (mrb // 3 + 1, mrb + 1)
        self.inputs = [self.det.upload_raw(e.raw, e.fed_offsets) for e in evs]
        self.want = []
        for d_raw, d_fo in self.inputs:
            o = self.det.alloc_outputs(*self.caps, **self.kw)
            self.det.run(d_raw, d_fo, self.thr, o)
            self.det.torch.cuda.synchronize()
            self.want.append(harness.unsigned_view(o.numpy()))
            assert self.want[-1]["n_clusters"] > 0

    def outputs(self):
        o = self.det.alloc_outputs(*self.caps, **self.kw)
        for t in o.tensors.values():   # nothing of an earlier result may survive in them
            t.fill_(0x55 if t.dtype == self.det.torch.uint8 else 0)
        return o

    def close(self):
        self.det.close()


@pytest.mark.parametrize("move_mode", [0, 1], ids=["move-in-kernel", "move-kernel"])
def test_noalloc_matches_the_pooled_path_on_calls_in_a_row(move_mode):
    from paper_2101_11489_b200 import harness
    import torch
    a = _Case(harness, 1, 37, [11, 12], move_mode)                  # whole-FED slots, two different events
    b = _Case(harness, 4, 11, [13], move_mode, hint=6000)           # another layout of the array; FEDs in pieces
    try:
        outs = [a.outputs(), a.outputs(), b.outputs(), a.outputs()]
        torch.cuda.synchronize()
        # two calls in a row on one stream, no synchronisation in between; then a context with
        # another scratch layout; then the first again, over what that one left behind
        a.det.run_noalloc(*a.inputs[0], a.thr, outs[0])
        a.det.run_noalloc(*a.inputs[1], a.thr, outs[1])
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        b.det.run_noalloc(*b.inputs[0], b.thr, outs[2])
        a.det.run_noalloc(*a.inputs[0], a.thr, outs[3])
        a.det.run_noalloc(*a.inputs[1], a.thr, outs[1])
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before, "device memory was allocated or freed by the calls"
        got = [harness.unsigned_view(o.numpy()) for o in outs]
        same(got[0], a.want[0])
        same(got[1], a.want[1])
        same(got[2], b.want[0])
        same(got[3], a.want[0])
    finally:
        a.close()
        b.close()


def test_noalloc_with_the_second_kernel_and_a_full_detector_event():
    """Compact SoA and hit coordinates (sst_emit_kernel behind sst_event_kernel), and one event of
    BASELINE.json config 1 at 440 FEDs: the largest context the 32 MiB hold."""
    from paper_2101_11489_b200 import harness
    import torch
    x = _Case(harness, 0, 24, [5, 6], 0, extras=True)
    full = _Case(harness, 1, None, [1], 0)
    try:
        o0, o1, of = x.outputs(), x.outputs(), full.outputs()
        x.det.run_noalloc(*x.inputs[0], x.thr, o0)
        x.det.run_noalloc(*x.inputs[1], x.thr, o1)
        full.det.run_noalloc(*full.inputs[0], full.thr, of)
        full.det.run_noalloc(*full.inputs[0], full.thr, of)
        torch.cuda.synchronize()
        same(harness.unsigned_view(o0.numpy()), x.want[0])
        same(harness.unsigned_view(o1.numpy()), x.want[1])
        same(harness.unsigned_view(of.numpy()), full.want[0])
    finally:
        x.close()
        full.close()


def test_noalloc_on_its_own_stream_beside_pooled_calls_on_another():
    """sst.h: the other entry points use pool scratch and may run beside the no-allocation call.  A
    batch of the pooled path on one stream and no-allocation calls on a second stream, enqueued
    alternately without synchronising, several rounds."""
    from paper_2101_11489_b200 import binding as B, harness
    import torch
    a = _Case(harness, 1, 37, [21, 22, 23], 0)
    try:
        s_pool, s_static = torch.cuda.Stream(), torch.cuda.Stream()
        pooled = [a.outputs() for _ in range(3)]
        static = [a.outputs() for _ in range(3)]
        batch = B.Batch([d[0] for d in a.inputs], [d[1] for d in a.inputs], a.thr, [o.out for o in pooled], [s_pool.cuda_stream])
        torch.cuda.synchronize()
        for _ in range(5):
            B.sst_unpack_cluster_batch(a.det.ctx, batch)
            for i in range(3):
                a.det.run_noalloc(*a.inputs[i], a.thr, static[i], stream=s_static)
        torch.cuda.synchronize()
        for i in range(3):
            same(harness.unsigned_view(pooled[i].numpy()), a.want[i])
            same(harness.unsigned_view(static[i].numpy()), a.want[i])
    finally:
        a.close()


def test_noalloc_refuses_a_context_beyond_the_limit():
    from paper_2101_11489_b200 import binding as B, harness
    import torch
    cfg, cal, evs = synth.make_config(0, n_feds=2, event_seeds=[3])
    ev = evs[0]
    det = harness.Detector(2, cal.gain, cal.noise, cal.bad, cal.chan_module, max_raw_bytes=4 << 20)   # ~100 MiB of scratch
    try:
        d_raw, d_fo = det.upload_raw(ev.raw, ev.fed_offsets)
        o = det.alloc_outputs(1000, 4000)
        o.tensors["dev_status"].fill_(77)
        with pytest.raises(B.SSTError, match="SST_ERR_TOO_LARGE"):
            det.run_noalloc(d_raw, d_fo, cfg.thresholds[0], o)
        torch.cuda.synchronize()
        assert int(o.tensors["dev_status"][0]) == 77, "a refused call must enqueue nothing"
        det.run(d_raw, d_fo, cfg.thresholds[0], o)                  # the pooled path takes the same context
        torch.cuda.synchronize()
        assert int(o.tensors["n_clusters"][0]) > 0
    finally:
        det.close()
