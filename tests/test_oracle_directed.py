"""Directed boundary cases against the oracle: expected values are written by hand in tests/cases.py."""
import numpy as np
import pytest

import oracle
from cases import case_arrays, directed_cases
from paper_1411_3968_b200 import workload as W
from util import oracle_chain, single_tower_geo

CASES = directed_cases()


@pytest.mark.parametrize("c", CASES, ids=[c["name"] for c in CASES])
def test_directed_case(c, oracle_lib):
    h, seg = case_arrays(c)
    geo = single_tower_geo(c["table"])
    p = W.Params(**c["params"])
    r = oracle_chain(h, seg, geo, p)
    e = c["expect"]
    if "order" in e:
        assert r["perm"].tolist() == e["order"]
    if "flags" in e:
        assert r["flags"].tolist() == e["flags"]
    if "seeds" in e:
        assert r["seeds"].tolist() == e["seeds"]
    if "events" in e:
        got = [tuple(int(x) for x in ev) for ev in r["events"]]
        assert got == e["events"]


def test_bad_pmt_status(oracle_lib):
    """pmt_id >= n_pmt on an L1 hit: status bit 8, and the hit has no edges."""
    h = np.zeros(3, dtype=W.HIT_DTYPE)
    h["t_ps"] = [0, 10, 20]; h["pmt_id"] = [0, 9, 1]; h["charge"] = 400; h["floor"] = [0, 1, 2]
    geo = single_tower_geo(np.full((4, 4), 100_000, dtype=np.int32))
    r = oracle_chain(h, np.array([0, 3], dtype=np.uint32), geo, W.Params(l2_multiplicity=2))
    assert r["status"] & 8
    assert r["flags"].tolist() == [4 | 1 | 8 | 16 | 32, 4 | 1 | 32, 4 | 1 | 8 | 16 | 32]
