"""SURVEY 8(f) NEXT-4 on the GPU: the accuracy experiment of section IV (Eq.(36)) through the C ABI - data SFTs of the
fiducial signal made on the device (sft_ingest_timeseries), ([d,h]) from sft_inner_products - against the oracle's r on the
same inputs, and against the magnitudes the paper prints."""
import numpy as np
import pytest

from oracle import accuracy as oa
from paper_2502_11823_b200 import workloads as wl
from _util import to_oracle

pytestmark = pytest.mark.gpu


def _oracle_r(example, delta, dk, include_dc=0, f_start=None):
    from paper_2502_11823_b200 import accuracy_map as am
    w = wl.accuracy_case(example, am.t_sft_for(example, delta), dk // 2, f_start=f_start)
    w.desc = dict(w.desc, include_dc=include_dc)
    plan, store = to_oracle(w)
    return oa.accuracy_point(plan, store, w.params, w.series[0], 1.0 / w.desc["fs"])


@pytest.mark.parametrize("example,delta,dk,dc,f_start", [("bns", 3.0, 20, 0, 4.0), ("bns", 1.0, 4, 0, 4.0), ("bns", 0.5, 100, 0, 5.0),
                                                         ("mbhb", 1.0, 200, 1, 4e-4), ("mbhb", 0.05, 20, 0, 6e-4)])
def test_r_matches_the_oracle(example, delta, dk, dc, f_start):
    from paper_2502_11823_b200 import accuracy_map as am
    g = am.accuracy_point(example, delta, dk, dc, f_start)
    o = _oracle_r(example, delta, dk, dc, f_start)
    # same inputs, same algorithm: ([d,h]) within the parity bar; here d = h, so sqrt(<x,x><h,h>) ~ <h,h>
    assert abs(g["xh"] - o["xh"]) <= 5e-6 * o["exact"] and abs(g["hh"] - o["hh"]) <= 5e-6 * o["exact"]
    assert abs(g["exact"] - o["exact"]) <= 1e-12 * o["exact"]
    assert abs(g["r"] - o["r"]) <= 1e-5


def test_paper_magnitudes_full_size():
    """The two examples at full size: BNS delta = 3, Delta k = 20 -> r < 1 %; massive BBH delta = 1, Delta k = 200 with
    the k = 0 bin -> r ~ 3 %, an order of magnitude above the BNS value at the same (delta, Delta k)."""
    from paper_2502_11823_b200 import accuracy_map as am
    b = am.accuracy_point("bns", 3.0, 20, 0)
    assert abs(b["t_sft"] - 106.0) < 1.5 and 0.0 < b["r"] < 0.01
    b2 = am.accuracy_point("bns", 1.0, 200, 0)
    m = am.accuracy_point("mbhb", 1.0, 200, 1)
    assert 0.015 < m["r"] < 0.06 and m["r"] > 8.0 * b2["r"]
