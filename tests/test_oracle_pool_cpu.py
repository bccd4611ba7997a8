"""The process-pool helpers the full-size GPU parity tests use must return exactly what the oracle returns."""
import numpy as np

import os, sys
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import oracle_pool
from oracle import nbs_oracle as O
from paper_1604_07983_b200 import synth


def test_pool_helpers_equal_plain_oracle_calls():
    L = 3
    S = {f: synth.propagator(51, i, 0, L, 0.1) for i, f in enumerate("uds")}
    chans = [("p", "L", "Sp", "n"), ("L", "L", "p", "Xm"), ("Xm", "X0", "Xm", "X0")]
    B = O.all_blocks(S, O.sink_names(chans))
    ref = O.correlator_fft(L, B, chans)
    got = oracle_pool.tierB_channels([(L, S, chans)], workers=2)[0]
    assert np.array_equal(got, ref)
    qs = np.array([1 + L * (2 + L * 0), 5, 26])
    Bq = oracle_pool.blocks_at_momenta(L, S, ["p", "L"], qs, chunk=10, workers=2)
    for name in ("p", "L"):
        full = O.fft_blocks(L, B[name])
        assert np.abs(Bq[name] - full[qs]).max() <= 1e-12 * np.abs(full).max()
