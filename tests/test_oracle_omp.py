"""The OpenMP timing build of the oracle gives bit-identical results to the sequential oracle
for any N x M split (section 3 shape; oracle/sst_oracle_omp.c)."""
import numpy as np
import pytest

from paper_2101_11489_b200 import synth


@pytest.mark.parametrize("n_outer,n_inner", [(1, 1), (2, 3), (1, 8), (3, 1), (2, 24)])
def test_omp_matches_sequential(oracle, n_outer, n_inner):
    cfg, cal, evs = synth.make_config(3, n_feds=24, event_seeds=(1, 2, 3))
    seq = [oracle.run(e.raw, e.fed_offsets, 24, cal.gain, cal.noise, cal.bad, cal.chan_module, (2, 3, 5))
           for e in evs]
    ncl, nsd, hh = oracle.events_omp([e.raw for e in evs], [e.fed_offsets for e in evs], 24, cal.gain,
                                     cal.noise, cal.bad, cal.chan_module, (2, 3, 5), n_outer, n_inner)
    for k, r in enumerate(seq):
        assert ncl[k] == r.n_clusters and nsd[k] == r.seed_idx.size
        assert int(hh[k]) == oracle.result_hash(r)
