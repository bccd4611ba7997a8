"""Host-side checks of the C-ABI library that need no GPU: it builds, loads, exports every symbol
include/nbs.h declares, its table generator (row a0) reproduces the paper's printed counts, and the
product path fails loudly without a CUDA device (no CPU fallback)."""
import os
import re

import pytest

from conftest import ROOT, read_golden
from paper_1604_07983_b200 import nbs

GOLD = read_golden("paper_counts.txt")


def declared_functions():
    text = open(os.path.join(ROOT, "include", "nbs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(nbs_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = nbs.lib()
    names = declared_functions()
    assert {"nbs_create", "nbs_load_propagators", "nbs_correlator", "nbs_destroy"} <= set(names)
    for name in names:
        assert hasattr(lib, name), name
    assert sorted(nbs.EXPORTS) == names


def test_standard_channels_52():
    chans = nbs.nbs_std_channels()
    assert len(chans) == int(GOLD["n_channels"]) and len(set(chans)) == 52
    assert chans[0] == ("p", "n", "p", "n") and chans[-1] == ("Xm", "X0", "Xm", "X0")  # "from NN to Xi-Xi"


def test_paper_counts_pLpXu():
    """3456 literal terms, 370 = 1+9+144+144+36+36 effective terms."""
    st = nbs.nbs_diagram_stats(("p", "L", "p", "Xu"))
    assert st["literal_terms"] == int(GOLD["literal_terms_pLpXu"])
    assert sum(st["K"]) == int(GOLD["effective_terms_pLpXu"])
    assert sorted(st["K"]) == sorted(int(v) for v in GOLD["effective_sizes_pLpXu"].split())
    # enumeration order = lexicographic in P: the worked table of DESIGN.md (eq. 2.7 terms)
    assert st["K"] == [1, 9, 144, 144, 36, 36]
    assert st["sign"] == [+1, -1, -1, +1, +1, -1]


def test_derived_totals_over_52_channels():
    """655 diagrams, sum K = 43507, K histogram (derived)."""
    ks = []
    for ch in nbs.nbs_std_channels():
        ks += nbs.nbs_diagram_stats(ch)["K"]
    assert len(ks) == 655 and sum(ks) == 43507
    assert {k: ks.count(k) for k in set(ks)} == {1: 91, 9: 76, 36: 255, 144: 233}


def test_tables_agree_with_oracle_enumeration(oracle):
    """The CUDA path's host generator and the oracle are written independently; their diagram
    lists (K and sigma_P, in lexicographic order of P) must coincide channel by channel."""
    for ch in oracle.channels52():
        st = nbs.nbs_diagram_stats(ch)
        ds = oracle.diagrams(ch)
        assert st["diagrams"] == len(ds)
        assert st["K"] == [oracle.diagram_K(P) for _, _, P in ds]
        assert st["sign"] == [s for _, s, _ in ds]
    assert nbs.nbs_std_channels() == oracle.channels52()


def test_flavour_violating_channel_is_rejected():
    with pytest.raises(nbs.NbsError) as e:
        nbs.nbs_diagram_stats(("p", "n", "p", "p"))
    assert e.value.code == nbs.NBS_EINVAL


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(nbs.NbsError) as e:
        nbs.nbs_create(4, 1)
    assert e.value.code == nbs.NBS_ECUDA


def test_plan_tables_stay_in_bounds():
    """compute-sanitizer is closed on the target pool, so the indices the kernels take from tables are bounds-checked on
    the host: gather offsets inside the staged blocks, table extents including the pipeline's look-ahead, unit / diagram
    / chain / channel record ranges, expansion maps -- for the standard 52 channels and for user lists."""
    from paper_1604_07983_b200 import nbs
    assert nbs.nbs_plan_selfcheck() == 0
    assert nbs.nbs_plan_selfcheck([("p", "n", "p", "n")]) == 0
    assert nbs.nbs_plan_selfcheck([("L", "L", "L", "L"), ("S0", "S0", "Sp", "Sm"), ("p", "L", "p", "Xu"), ("Xu", "Xs", "Xd", "Xs")]) == 0
    assert nbs.nbs_plan_selfcheck([("p", "p", "p", "p"), ("n", "n", "n", "n"), ("p", "n", "p", "n")] * 40) == 0


def test_isospin_channel_relations_of_the_standard_list():
    """include/nbs.h nbs_iso_relations: the u <-> d images in the standard list are the nine relations the oracle pins
    (tests/test_oracle_pins.py::test_isospin_relations_u_equals_d), with their signs, found from the operator table;
    the reduced list passes the table self-check."""
    rel = nbs.nbs_iso_relations()
    derived = {i: r for i, r in enumerate(rel) if r[0] >= 0}
    assert derived == {12: (11, -1, 0), 21: (15, -1, 0), 22: (17, +1, 0), 23: (16, +1, 0), 24: (18, +1, 1),
                       25: (19, -1, 0), 26: (20, +1, 0), 35: (34, -1, 0), 39: (38, +1, 0)}
    for i, (src, _sign, _swap) in derived.items():
        assert src < i and rel[src][0] < 0
    reduced = [c for c, r in zip(nbs.nbs_std_channels(), rel) if r[0] < 0]
    assert len(reduced) == 43 and ("n", "X0") not in {(c[0], c[1]) for c in reduced}
    assert nbs.nbs_plan_selfcheck(reduced) == 0
    # no image in the list: nothing is derived; an image with exchanged source baryons carries the a3 <-> a4 flag
    assert all(r[0] < 0 for r in nbs.nbs_iso_relations([("p", "n", "p", "n"), ("Xm", "L", "Xm", "L")]))
    assert nbs.nbs_iso_relations([("p", "Xm", "Sp", "Sm"), ("n", "X0", "Sp", "Sm")]) == [(-1, 1, 0), (0, 1, 1)]
