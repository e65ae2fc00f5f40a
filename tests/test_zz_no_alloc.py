"""The allocation-free entry point ``sft_inner_products_static`` (include/sft.h) against the existing path
``sft_inner_products`` on the same plan and inputs, on two calls in a row.

Named ``test_zz_*`` so that pytest collects it last: the suite runs with ``pytest -x`` and a failure here must not hide
the other tests.  It passes alone in a fresh process and after the rest of the suite (it owns its plan and tensors; the only
thing it shares with anything else is the library's static scratch, which no other test touches).

Tolerance: the binding one of the parity tests (``test_gpu_parity.TOL`` = 1e-4, normalised by sqrt(<x,x>_band <h,h>)),
and beside it the far tighter bound that follows from what actually differs - the order of the fp64 chunk sums only.
"""
import numpy as np
import pytest

from oracle import inner as oin
from paper_2502_11823_b200 import workloads as wl
from _util import to_oracle

pytestmark = pytest.mark.gpu

TOL = 1e-4          # the parity tests' tolerance (test_gpu_parity.TOL)
ORDER = 1e-11       # fp64 summation order only


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _nan(n):
    import torch
    return torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")


def _compare(new, ref, xx):
    """new / ref: (xh, hh, xh_im) numpy triples of the static and of the existing path."""
    hh = np.maximum(ref[1], 1e-300)
    norm = np.sqrt(xx * hh)
    for name, a, b in zip(("xh", "hh", "xh_im"), new, ref):
        assert np.all(np.isfinite(a)), name
        e = np.abs(a - b) / norm
        assert e.max() <= TOL, (name, float(e.max()), int(e.argmax()))
        scale = np.maximum(np.abs(b), np.sqrt(hh))
        r = np.abs(a - b) / scale
        assert r.max() <= ORDER, (name, "summation-order bound", float(r.max()), int(r.argmax()))


@pytest.fixture(scope="module")
def et_static():
    """Config-2 recipe, 3200 SFT slots x 4096 templates (= SFT_STATIC_MAX_TEMPLATES): large enough that the static
    scratch caps the number of chunks (80 against the 100 the existing path uses), so both chunk rules are exercised."""
    return wl.et_bns(n_templates=4096, n_sft=3200, K=8, name="et-static")


def test_static_entry_point_matches_existing_path_twice(et_static):
    import torch
    from paper_2502_11823_b200 import api
    w = et_static
    oplan, ostore = to_oracle(w)
    xx = oin.xx_band(oplan, ostore)
    assert api.static_setup(0) == 8 * 1024 * 1024
    banks = [w.params, w.params[1000:1333][::-1]]          # two calls in a row: 4096 templates, then 333 other rows
    with api.plan_from_workload(w) as plan:
        P = [_dev(b) for b in banks]
        outs = [tuple(_nan(len(b)) for _ in range(3)) for b in banks]
        refs = [tuple(_nan(len(b)) for _ in range(3)) for b in banks]
        warm = tuple(_nan(1) for _ in range(3))
        plan.inner_products_static(P[0][:1].contiguous(), *warm)      # first launch of the kernels (module load)
        plan.sync()
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for p, o in zip(P, outs):                                     # back to back, no synchronisation in between
            plan.inner_products_static(p, *o)
        plan.sync()
        free1 = torch.cuda.mem_get_info()[0]
        # the existing path would have grown its 9.8 MB chunk-total buffer (and more) here; the static one takes nothing
        assert free1 == free0, ("device memory taken inside sft_inner_products_static", free0 - free1)
        for p, r in zip(P, refs):
            plan.inner_products(p, r[0], r[1], r[2], None)
        plan.sync()
        for o, r in zip(outs, refs):
            _compare([t.cpu().numpy() for t in o], [t.cpu().numpy() for t in r], xx)
        # a third call after the existing path ran on the same plan: still the same numbers (stale scratch is harmless)
        again = tuple(_nan(len(banks[1])) for _ in range(3))
        plan.inner_products_static(P[1], *again)
        plan.sync()
        for a, o in zip(again, outs[1]):
            assert torch.equal(a, o)
        # xh_im is optional
        xh, hh = _nan(len(banks[1])), _nan(len(banks[1]))
        plan.inner_products_static(P[1], xh, hh, None)
        plan.sync()
        assert torch.equal(xh, outs[1][0]) and torch.equal(hh, outs[1][1])


def test_static_entry_point_rejects_what_it_cannot_hold(et_static):
    from paper_2502_11823_b200 import api
    w = et_static
    n = api.STATIC_MAX_TEMPLATES + 1
    big = np.concatenate([w.params, w.params[:1]])
    with api.plan_from_workload(w) as plan:
        P, xh, hh = _dev(big), _nan(n), _nan(n)
        with pytest.raises(api.SftError) as ei:
            plan.inner_products_static(P, xh, hh, None)
        assert api.STATUS[ei.value.status] == "SFT_EUNSUPPORTED" and "SFT_STATIC_MAX_TEMPLATES" in str(ei.value)
        plan.sync()
        assert bool(xh.isnan().all()) and bool(hh.isnan().all())       # outputs untouched
        with pytest.raises(ValueError):                                # host arrays are refused by the binding
            plan.inner_products_static(big[:4], np.empty(4), np.empty(4))
        plan.inner_products_static(P[:0], xh[:0], hh[:0])              # n = 0: SFT_OK, no work
