"""Oracle side of the accuracy experiment of section IV.  Test infrastructure.

* ``relative_error`` - Eq.(36): ``r = 1 - sqrt(([d,h]) / <d,h>)``; where the ratio under the root is negative the
  ratio itself is returned in ``ratio`` and ``r`` is NaN (reading A15).
* ``exact_product``  - ``<d,h>`` "by direct integration": Eq.(1)/(14) P:20, P:149 for a flat PSD written in the time
  domain, ``(2 dt / S) sum_j d_j h_j`` (``oracle.sft.time_domain_product``; pinned by Parseval, P2).
* ``accuracy_point`` - one point of Fig. 3 / Fig. 4: the SFT product of the fiducial template with the data SFTs
  (``oracle.inner.inner_products``, the parity target) against the exact product.

The exact colour-map values of Fig. 3 / Fig. 4 are PARITY UNPINNED: they need IMRPhenomT and the authors' set-up.
What is pinned (tests/test_oracle_accuracy.py) are the magnitudes the paper prints - r < 1 % for delta <~ 3 and
Delta k >~ 20 in the BNS example - and what the mathematics fixes: r falls as the band widens and tends to the
truncation loss of the Dirichlet kernel (pin P8) for short SFTs; r = 0 for a signal that IS piecewise linear in frequency
with all its power inside the band.
"""
import numpy as np

from . import inner as oin
from . import sft as osft


def relative_error(xh_sft, xh_exact):
    """Eq.(36) P:274.  Returns (r, ratio)."""
    ratio = float(xh_sft) / float(xh_exact)
    return (1.0 - np.sqrt(ratio) if ratio >= 0.0 else float("nan")), ratio


def exact_product(d, h, dt, S_flat=1.0):
    """<d,h> by direct integration in the time domain (flat one-sided PSD)."""
    return osft.time_domain_product(d, h, dt, S_flat)


def accuracy_point(plan, store, params, series, dt):
    """r of Eq.(36) for the template ``params`` (one row) and the data whose time series is ``series`` (the noiseless
    fiducial signal, d = h): ([d,h]) from the SFT framework against <d,h> by direct integration."""
    o = oin.inner_products(plan, store, np.atleast_2d(params)[:1])
    exact = exact_product(series, series, dt)
    r, ratio = relative_error(o["xh"][0], exact)
    return dict(r=r, ratio=ratio, xh=float(o["xh"][0]), hh=float(o["hh"][0]), exact=exact)
