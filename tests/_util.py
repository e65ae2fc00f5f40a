"""Test helpers: Workload -> oracle Plan/Store."""
import numpy as np
from oracle import inner as oin


def to_oracle(w):
    d = dict(w.desc)
    plan = oin.Plan(**d)
    store = oin.Store(bins=w.bins.astype(np.complex128), psd_scale=w.psd_scale, psd_shape=w.psd_shape,
                      response=None if w.response is None else w.response.astype(np.complex128))
    return plan, store
