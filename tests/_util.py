"""Test helpers: Workload -> oracle Plan/Store, and the oracle run over many templates on all host cores."""
import os
import numpy as np
from oracle import inner as oin


def to_oracle(w):
    d = dict(w.desc)
    plan = oin.Plan(**d)
    store = oin.Store(bins=w.bins.astype(np.complex128), psd_scale=w.psd_scale, psd_shape=w.psd_shape,
                      response=None if w.response is None else w.response.astype(np.complex128))
    return plan, store


# ---- the oracle (as it stands, one call per template) spread over the host cores with multiprocessing ----
_G = {}


def _init(desc, bins, psd_scale, psd_shape, response):
    _G["plan"] = oin.Plan(**desc)
    _G["store"] = oin.Store(bins=bins.astype(np.complex128), psd_scale=psd_scale, psd_shape=psd_shape,
                            response=None if response is None else response.astype(np.complex128))


def _totals(rows):
    o = oin.inner_products(_G["plan"], _G["store"], rows)
    return o["xh"], o["hh"], o["xh_im"]


def _cumulative_at(args):
    rows, idx = args
    o = oin.cumulative_snr(_G["plan"], _G["store"], rows)
    take = lambda a: np.take_along_axis(a, idx, axis=1)
    return take(o["cum_xh"]), take(o["cum_hh"]), take(o["snr"]), o["cum_xh"][:, -1], o["cum_hh"][:, -1]


def _pool(w):
    import multiprocessing as mp
    n = max(1, min(32, len(os.sched_getaffinity(0))))
    # "spawn": the parent may hold a CUDA context, which must not be forked
    return mp.get_context("spawn").Pool(n, initializer=_init,
                                        initargs=(dict(w.desc), w.bins, w.psd_scale, w.psd_shape, w.response)), n


def oracle_totals_parallel(w, params, block=8):
    """oracle.inner.inner_products for every row of ``params``: (xh, hh, xh_im)."""
    pool, _ = _pool(w)
    with pool:
        parts = pool.map(_totals, [params[i:i + block] for i in range(0, len(params), block)])
    return tuple(np.concatenate([p[j] for p in parts]) for j in range(3))


def oracle_cumulative_at_parallel(w, params, idx, block=8):
    """oracle.inner.cumulative_snr for every row of ``params``, kept at the SFT indices ``idx[row]`` only:
    (cum_xh, cum_hh, snr) [rows][n_idx] and the totals (xh, hh) [rows]."""
    pool, _ = _pool(w)
    with pool:
        parts = pool.map(_cumulative_at, [(params[i:i + block], idx[i:i + block]) for i in range(0, len(params), block)])
    return tuple(np.concatenate([p[j] for p in parts]) for j in range(5))
