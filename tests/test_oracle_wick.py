"""Tier A (eq. 2.4 with baryon blocks) against tier W (brute-force Wick contraction of the
operators of eqs. 2.2-2.3, oracle/wick.c) on a 2^3 lattice -- BASELINE.json north_star."""
import numpy as np
import pytest

from oracle import nbs_oracle as O
from oracle import wick
from paper_1604_07983_b200 import synth


@pytest.fixture(scope="module")
def S2():
    return {f: synth.propagator(7, i, 0, 2, 0.1) for i, f in enumerate("uds")}


CASES = [
    # channel, spins, r values (None = all 8)
    (("p", "n", "p", "n"), [(0, 1, 0, 1), (2, 3, 3, 2)], None),
    (("p", "L", "p", "Xu"), [(1, 0, 0, 1)], [0, 3, 6]),          # the paper's worked example (eq. 2.7)
    (("Xm", "X0", "Xm", "X0"), [(0, 0, 1, 1), (3, 1, 1, 3)], [1, 7]),
    (("Sp", "n", "S0", "p"), [(0, 2, 2, 0)], [2, 5]),
    (("S0", "L", "Sp", "Sm"), [(1, 3, 3, 1)], [4]),
    (("L", "L", "L", "L"), [(0, 1, 1, 0)], [5]),                  # 81 elementary combinations
]


@pytest.mark.parametrize("ch,spins,rs", CASES, ids=["-".join(c[0]) for c in CASES])
def test_tierA_equals_bruteforce_wick(S2, ch, spins, rs):
    L = 2
    rs = list(range(8)) if rs is None else rs
    bl = O.all_blocks(S2, ch[:2])
    FA = O.correlator_direct(L, bl, ch, rs=rs)
    FW = wick.wick_fourpt(L, S2, ch, spins, rs)
    FAs = np.array([[FA[s][r] for s in spins] for r in rs])
    assert abs(FAs - FW).max() <= 1e-12 * abs(FW).max()
    assert abs(FW).max() > 0
